/*
 * splotch_oracle_mt.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * All-cores drivers around the UNCHANGED functions of splotch_oracle.c.  Nothing is computed here: every
 * function below only cuts the index range or the image into pieces and calls the single-threaded oracle on
 * each piece from an OpenMP loop.
 *
 *   orc_geometry_mt / orc_amplitude_mt   per-particle stages: contiguous particle ranges, one call per range.
 *                                        A particle's results depend on that particle only, so the outputs are
 *                                        bit-identical to one call over the whole range.
 *   orc_render_additive_mt / _ordered_mt the row-band scheme of SURVEY 8(d): the image rows are cut into
 *                                        contiguous bands, every band is rendered by one call that walks ALL
 *                                        particles in the same order (index order / far-to-near) and touches only
 *                                        its rows (the window arguments of the single-threaded functions), so
 *                                        every pixel receives the same contributions in the same order: the image
 *                                        is bit-identical to the single-threaded one in both modes.  It mirrors the
 *                                        paper's OpenMP scheme: image tiles taken by threads "first-come,
 *                                        first-serve".
 * tests/test_oracle_mt.py checks the bit-identity.
 *
 * Build (together with splotch_oracle.c): gcc -O2 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC
 */
#include <stdint.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* the single-threaded oracle (splotch_oracle.c) */
void orc_geometry(int64_t n, const float *x, const float *y, const float *z, const float *h,
                  const float cam[16], float chi, float r_small, float r_large, float z_near,
                  int W, int H, int T,
                  int8_t *cls, float *px, float *py, float *sp, float *rp, float *zc,
                  int32_t *pbox, int32_t *tbox, int32_t *ilabel);
void orc_amplitude(int64_t n, const float *I, const float *scalar, const float *h,
                   const int32_t *species_of, int n_species,
                   const double *brightness, const int32_t *use_colormap, const double *fixed_rgb,
                   const double *smin, const double *smax, const int32_t *use_log10,
                   const double *lut, const int32_t *lut_offset, const int32_t *lut_entries,
                   double *E, double *col);
void orc_render_additive(int64_t p_begin, int64_t p_end, const int8_t *cls,
                         const float *px, const float *py, const float *sp, const float *rp,
                         const int32_t *pbox, const double *E, const double *col, float chi,
                         int W, int H, int wx0, int wx1, int wy0, int wy1,
                         int apply_transfer, double *image);
void orc_render_ordered(int64_t m, const int64_t *order, const int8_t *cls,
                        const float *px, const float *py, const float *sp, const float *rp,
                        const int32_t *pbox, const double *E, const double *col, const double *kappa,
                        float chi, int W, int H, int wx0, int wx1, int wy0, int wy1, double *image);

int orc_mt_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

#define ORC_MT_RANGE (1 << 18)      /* particles per call of a per-particle stage */

void orc_geometry_mt(int threads, int64_t n, const float *x, const float *y, const float *z, const float *h,
                     const float cam[16], float chi, float r_small, float r_large, float z_near,
                     int W, int H, int T,
                     int8_t *cls, float *px, float *py, float *sp, float *rp, float *zc,
                     int32_t *pbox, int32_t *tbox, int32_t *ilabel)
{
    const int64_t nr = (n + ORC_MT_RANGE - 1) / ORC_MT_RANGE;
    int64_t r;
    (void)threads;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads)
    for (r = 0; r < nr; ++r) {
        const int64_t a = r * ORC_MT_RANGE, b = a + ORC_MT_RANGE < n ? a + ORC_MT_RANGE : n;
        orc_geometry(b - a, x + a, y + a, z + a, h + a, cam, chi, r_small, r_large, z_near, W, H, T,
                     cls + a, px + a, py + a, sp + a, rp + a, zc + a, pbox + 4 * a, tbox + 4 * a, ilabel + a);
    }
}

void orc_amplitude_mt(int threads, int64_t n, const float *I, const float *scalar, const float *h,
                      const int32_t *species_of, int n_species,
                      const double *brightness, const int32_t *use_colormap, const double *fixed_rgb,
                      const double *smin, const double *smax, const int32_t *use_log10,
                      const double *lut, const int32_t *lut_offset, const int32_t *lut_entries,
                      double *E, double *col)
{
    const int64_t nr = (n + ORC_MT_RANGE - 1) / ORC_MT_RANGE;
    int64_t r;
    (void)threads;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads)
    for (r = 0; r < nr; ++r) {
        const int64_t a = r * ORC_MT_RANGE, b = a + ORC_MT_RANGE < n ? a + ORC_MT_RANGE : n;
        orc_amplitude(b - a, I + a, scalar + a, h + a, species_of + a, n_species, brightness, use_colormap,
                      fixed_rgb, smin, smax, use_log10, lut, lut_offset, lut_entries, E + 3 * a, col + a);
    }
}

/* Row bands inside the window [wx0, wx1] x [wy0, wy1]; `bands` of them (at least one row each). */
void orc_render_additive_mt(int threads, int bands, int64_t p_begin, int64_t p_end, const int8_t *cls,
                            const float *px, const float *py, const float *sp, const float *rp,
                            const int32_t *pbox, const double *E, const double *col, float chi,
                            int W, int H, int wx0, int wx1, int wy0, int wy1,
                            int apply_transfer, double *image)
{
    const int rows = wy1 - wy0 + 1;
    int b;
    (void)threads;
    if (rows <= 0) return;
    if (bands > rows) bands = rows;
    if (bands < 1) bands = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads)
    for (b = 0; b < bands; ++b) {
        const int y0 = wy0 + (int)((int64_t)rows * b / bands), y1 = wy0 + (int)((int64_t)rows * (b + 1) / bands) - 1;
        if (y0 <= y1)
            orc_render_additive(p_begin, p_end, cls, px, py, sp, rp, pbox, E, col, chi, W, H, wx0, wx1, y0, y1,
                                apply_transfer, image);
    }
}

void orc_render_ordered_mt(int threads, int bands, int64_t m, const int64_t *order, const int8_t *cls,
                           const float *px, const float *py, const float *sp, const float *rp,
                           const int32_t *pbox, const double *E, const double *col, const double *kappa,
                           float chi, int W, int H, int wx0, int wx1, int wy0, int wy1, double *image)
{
    const int rows = wy1 - wy0 + 1;
    int b;
    (void)threads;
    if (rows <= 0) return;
    if (bands > rows) bands = rows;
    if (bands < 1) bands = 1;
#pragma omp parallel for schedule(dynamic, 1) num_threads(threads)
    for (b = 0; b < bands; ++b) {
        const int y0 = wy0 + (int)((int64_t)rows * b / bands), y1 = wy0 + (int)((int64_t)rows * (b + 1) / bands) - 1;
        if (y0 <= y1)
            orc_render_ordered(m, order, cls, px, py, sp, rp, pbox, E, col, kappa, chi, W, H, wx0, wx1, y0, y1, image);
    }
}
