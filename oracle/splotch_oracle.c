/*
 * splotch_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, single-threaded CPU statement of what the Splotch per-frame rendering path
 * computes, written from the paper (arxiv 1309.1114, PAPER.md) and the readings listed in
 * DESIGN.md ("Readings").  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call it.  It shares no code, header, table or
 * constant generator with the CUDA path under paper_1309_1114_b200/csrc/.
 *
 * Two parts:
 *   C1  canonical float32 screen geometry (roto-translation, perspective projection, projected
 *       radius, S/M/L classification, pixel / tile boxes, the paper's tile label i(p)).
 *       The paper computes in single precision and these values decide integers
 *       (class, boxes), so they are taken in float32 with one rounding per written operation;
 *       the CUDA path must reproduce them bit for bit.
 *   C2  everything that is accumulated (colour, column amplitude, Gaussian weights, the image)
 *       in double precision, particles in index order (additive) or far-to-near (ordered).
 *
 * Pins (tests/test_oracle_*.py): ODE integration of Eq. 1 through Eq. 2 along true perspective
 * rays, flux conservation, permutation invariance, reduction to a weighted 2-D histogram,
 * Fig. 2's five-particle scenario, resolution scaling, brute-force tile recount.
 * "Parity unpinned" by the paper itself (pinned only by DESIGN.md readings): the value of chi,
 * the SMALL-particle deposit rule (R6), the E/A/rho0 input mapping (R12), the depth-order rule
 * for E != A (R15), the normalisation of the vector colour mode (R24).
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC splotch_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { ORC_CULLED = 0, ORC_SMALL = 1, ORC_MEDIUM = 2, ORC_LARGE = 3 };

/* ---------------------------------------------------------------------------------------------
 * Camera constants ("roto-translated and projected according to camera settings").
 * Pin-hole camera: forward f = normalize(lookat - eye), right r = normalize(f x up), u = r x f;
 * pixel scale s = (W/2)/tan(fov/2) with fov the full horizontal angle; image centre (W/2, H/2).
 * Double arithmetic on the float inputs, one rounding to float32 at the end.
 * cam[0..2]=r  cam[3..5]=u  cam[6..8]=f  cam[9..11]=eye  cam[12]=s  cam[13]=c_x  cam[14]=c_y
 * Returns 0, or -1 for a degenerate camera.
 * ------------------------------------------------------------------------------------------- */
int orc_camera(const float eye[3], const float lookat[3], const float up[3], float fov_deg,
               int W, int H, float cam[16])
{
    double f[3], r[3], u[3], nf, nr;
    int k;
    for (k = 0; k < 3; ++k) f[k] = (double)lookat[k] - (double)eye[k];
    nf = sqrt(f[0] * f[0] + f[1] * f[1] + f[2] * f[2]);
    if (!(nf > 0.0) || !(fov_deg > 0.0f) || !(fov_deg < 180.0f) || W <= 0 || H <= 0) return -1;
    for (k = 0; k < 3; ++k) f[k] /= nf;
    r[0] = f[1] * (double)up[2] - f[2] * (double)up[1];
    r[1] = f[2] * (double)up[0] - f[0] * (double)up[2];
    r[2] = f[0] * (double)up[1] - f[1] * (double)up[0];
    nr = sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
    if (!(nr > 0.0)) return -1;
    for (k = 0; k < 3; ++k) r[k] /= nr;
    u[0] = r[1] * f[2] - r[2] * f[1];
    u[1] = r[2] * f[0] - r[0] * f[2];
    u[2] = r[0] * f[1] - r[1] * f[0];
    for (k = 0; k < 3; ++k) {
        cam[k] = (float)r[k];
        cam[3 + k] = (float)u[k];
        cam[6 + k] = (float)f[k];
        cam[9 + k] = eye[k];
    }
    cam[12] = (float)(0.5 * (double)W / tan(0.5 * ((double)fov_deg * (3.14159265358979323846 / 180.0))));
    cam[13] = (float)(0.5 * (double)W);
    cam[14] = (float)(0.5 * (double)H);
    cam[15] = 0.0f;
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * C1: per-particle geometry, classification and labels.
 *   camera space  (x_c, y_c, z_c) = (r.d, u.d, f.d),  d = x_p - eye      (roto-translation, :76)
 *   k = s / z_c ;  p_x = c_x + x_c k ;  p_y = c_y - y_c k                 (perspective, row 0 = top)
 *   sigma in pixels  sp = h k ;  r(p) = chi sp                            (Eq. 7)
 *   Small r(p) <= r_sml, Medium r_sml < r(p) <= r_0, Large r(p) > r_0     (r = r_0 -> M)
 *   inactive = "completely outside the scene" (:76): behind the near plane, or no pixel centre of the
 *   screen inside its bounding box; an off-screen centre with an on-screen box stays active (Fig. 2, :187)
 *   i(p): -2 inactive, N_tiles small, -1 large, else tile of the (clamped) centre pixel
 * Every float operation below is a single IEEE binary32 operation (fmaf = one rounding).
 * ------------------------------------------------------------------------------------------- */
static float orc_dot3(const float *a, float dx, float dy, float dz)
{
    return fmaf(a[2], dz, fmaf(a[1], dy, a[0] * dx));
}

void orc_geometry(int64_t n, const float *x, const float *y, const float *z, const float *h,
                  const float cam[16], float chi, float r_small, float r_large, float z_near,
                  int W, int H, int T,
                  int8_t *cls, float *px, float *py, float *sp, float *rp, float *zc,
                  int32_t *pbox /* 4n: x0 x1 y0 y1 */, int32_t *tbox /* 4n: tx0 tx1 ty0 ty1 */,
                  int32_t *ilabel)
{
    const int ntx = (W + T - 1) / T, nty = (H + T - 1) / T;
    const float fW = (float)W, fH = (float)H;
    int64_t p;
    for (p = 0; p < n; ++p) {
        float dx = x[p] - cam[9], dy = y[p] - cam[10], dz = z[p] - cam[11];
        float xc = orc_dot3(cam + 0, dx, dy, dz);
        float yc = orc_dot3(cam + 3, dx, dy, dz);
        float z_c = orc_dot3(cam + 6, dx, dy, dz);
        int c = ORC_CULLED;
        int32_t b[4] = {0, -1, 0, -1}, t[4] = {0, -1, 0, -1};
        float ppx = 0.0f, ppy = 0.0f, ssp = 0.0f, rr = 0.0f;
        if (z_c > z_near) {
            float k = cam[12] / z_c;
            ppx = fmaf(xc, k, cam[13]);
            ppy = fmaf(-yc, k, cam[14]);
            ssp = h[p] * k;
            rr = chi * ssp;
            if (rr >= 0.0f && rr <= 3.0e38f) {
                if (rr <= r_small) {
                    if (ppx >= 0.0f && ppx < fW && ppy >= 0.0f && ppy < fH) {
                        c = ORC_SMALL;
                        b[0] = b[1] = (int32_t)floorf(ppx);
                        b[2] = b[3] = (int32_t)floorf(ppy);
                    }
                } else {
                    float fx0 = fmaxf(ceilf((ppx - rr) - 0.5f), 0.0f);
                    float fx1 = fmaxf(fminf(floorf((ppx + rr) - 0.5f), fW - 1.0f), -1.0f);
                    float fy0 = fmaxf(ceilf((ppy - rr) - 0.5f), 0.0f);
                    float fy1 = fmaxf(fminf(floorf((ppy + rr) - 0.5f), fH - 1.0f), -1.0f);
                    if (fx0 <= fx1 && fy0 <= fy1) {
                        c = (rr <= r_large) ? ORC_MEDIUM : ORC_LARGE;
                        b[0] = (int32_t)fx0; b[1] = (int32_t)fx1;
                        b[2] = (int32_t)fy0; b[3] = (int32_t)fy1;
                    }
                }
            }
        }
        if (c != ORC_CULLED) {
            t[0] = b[0] / T; t[1] = b[1] / T; t[2] = b[2] / T; t[3] = b[3] / T;
        }
        cls[p] = (int8_t)c;
        px[p] = ppx; py[p] = ppy; sp[p] = ssp; rp[p] = rr; zc[p] = z_c;
        memcpy(pbox + 4 * p, b, sizeof b);
        memcpy(tbox + 4 * p, t, sizeof t);
        if (c == ORC_CULLED) ilabel[p] = -2;
        else if (c == ORC_LARGE) ilabel[p] = -1;
        else if (c == ORC_SMALL) ilabel[p] = ntx * nty;
        else {
            float cxp = fminf(fmaxf(floorf(ppx), 0.0f), fW - 1.0f);
            float cyp = fminf(fmaxf(floorf(ppy), 0.0f), fH - 1.0f);
            ilabel[p] = ((int32_t)cyp / T) * ntx + (int32_t)cxp / T;
        }
    }
}

/* Number of particles whose tile box contains each tile (the coverage binning the renderer uses). */
void orc_tile_counts(int64_t n, const int8_t *cls, const int32_t *tbox, int ntx, int nty,
                     int count_large, uint32_t *counts /* nty*ntx, zeroed here */)
{
    int64_t p;
    int tx, ty;
    memset(counts, 0, sizeof(uint32_t) * (size_t)ntx * (size_t)nty);
    for (p = 0; p < n; ++p) {
        if (cls[p] == ORC_CULLED) continue;
        if (cls[p] == ORC_LARGE && !count_large) continue;
        for (ty = tbox[4 * p + 2]; ty <= tbox[4 * p + 3]; ++ty)
            for (tx = tbox[4 * p + 0]; tx <= tbox[4 * p + 1]; ++tx)
                counts[ty * ntx + tx] += 1u;
    }
}

/* ---------------------------------------------------------------------------------------------
 * C2: colour and column amplitude (double).
 *   "Active particles ... are assigned with RGB color components" (:76); "a scalar quantity ... can be
 *   mapped to RGB components via look-up tables (or palettes)" (:85); normalisation and logarithms
 *   with user-given min/max (:76, :166 fn. 1).
 *   v = scalar (or log10 scalar); t = clamp((v - min)/(max - min), 0, 1); piecewise-linear LUT.
 *   E[c] = brightness * colour[c];  column constant col = sqrt(pi) * h * I, the line integral of
 *   Eq. 2 through the particle centre with rho_0 = I and sigma = h (world units).
 * species_of[p] gives the species; lut holds all species' tables back to back.
 * ------------------------------------------------------------------------------------------- */
void orc_amplitude(int64_t n, const float *I, const float *scalar, const float *h,
                   const int32_t *species_of, int n_species,
                   const double *brightness, const int32_t *use_colormap, const double *fixed_rgb,
                   const double *smin, const double *smax, const int32_t *use_log10,
                   const double *lut, const int32_t *lut_offset, const int32_t *lut_entries,
                   double *E /* 3n */, double *col /* n */)
{
    const double sqrt_pi = sqrt(3.14159265358979323846);
    int64_t p;
    int c;
    (void)n_species;
    for (p = 0; p < n; ++p) {
        int s = species_of[p];
        double rgb[3];
        if (use_colormap[s]) {
            int K = lut_entries[s];
            const double *L = lut + 3 * (size_t)lut_offset[s];
            double v = (double)scalar[p], t, uu;
            int i0;
            if (use_log10[s]) v = log10(v);
            t = (v - smin[s]) / (smax[s] - smin[s]);
            if (!(t > 0.0)) t = 0.0;               /* NaN (log of a negative) clamps to 0 */
            if (t > 1.0) t = 1.0;
            uu = t * (double)(K - 1);
            i0 = (int)floor(uu);
            if (i0 > K - 2) i0 = K - 2;
            for (c = 0; c < 3; ++c)
                rgb[c] = L[3 * i0 + c] + (uu - (double)i0) * (L[3 * (i0 + 1) + c] - L[3 * i0 + c]);
        } else {
            for (c = 0; c < 3; ++c) rgb[c] = fixed_rgb[3 * s + c];
        }
        for (c = 0; c < 3; ++c) E[3 * p + c] = brightness[s] * rgb[c];
        col[p] = sqrt_pi * (double)h[p] * (double)I[p];
    }
}

/* ---------------------------------------------------------------------------------------------
 * Weight of particle p at pixel (i, j):  exp(-d^2 / sp^2) inside the clip disc d <= chi sp
 * (Eq. 2 integrated along the ray, clipped at chi sigma on the screen).
 * The inside test is the float32 predicate of C1 so that both sides splat the same pixel set;
 * the value is double, from the float32 centre and sigma promoted to double.
 * ------------------------------------------------------------------------------------------- */
static int orc_inside(int i, int j, float ppx, float ppy, float rr)
{
    float dxf = ((float)i + 0.5f) - ppx;
    float dyf = ((float)j + 0.5f) - ppy;
    float d2 = fmaf(dxf, dxf, dyf * dyf);
    return d2 <= rr * rr;
}

static double orc_weight(int i, int j, float ppx, float ppy, float ssp)
{
    double dx = ((double)i + 0.5) - (double)ppx;
    double dy = ((double)j + 0.5) - (double)ppy;
    double s = (double)ssp;
    return exp(-(dx * dx + dy * dy) / (s * s));
}

/* A SMALL particle "falls inside a single pixel" (:162) and "only its location has to be calculated"
 * (:179): it deposits the whole flux of its clipped 2-D Gaussian, pi sp^2 (1 - exp(-chi^2)), there. */
static double orc_small_weight(float ssp, float chi)
{
    double s = (double)ssp, x = (double)chi;
    return 3.14159265358979323846 * s * s * (1.0 - exp(-x * x));
}

/* ---------------------------------------------------------------------------------------------
 * Additive mode, E_p = A_p: the solution of Eq. 1 over all particles is
 * I = 1 - exp(-S),  S = sum_p E_p tau_p,  tau_p = col_p w_p, independent of the order.
 * image[j][i][c] (double, H x W x 3) receives S, or 1 - exp(-S) when apply_transfer != 0.
 * Only pixels inside the window [wx0, wx1] x [wy0, wy1] are evaluated (whole image: 0, W-1, 0, H-1).
 * Particles are visited in index order; [p_begin, p_end) selects a sub-range.
 * ------------------------------------------------------------------------------------------- */
void orc_render_additive(int64_t p_begin, int64_t p_end, const int8_t *cls,
                         const float *px, const float *py, const float *sp, const float *rp,
                         const int32_t *pbox, const double *E, const double *col, float chi,
                         int W, int H, int wx0, int wx1, int wy0, int wy1,
                         int apply_transfer, double *image)
{
    int64_t p;
    int i, j, c;
    (void)H;
    for (p = p_begin; p < p_end; ++p) {
        int x0 = pbox[4 * p], x1 = pbox[4 * p + 1], y0 = pbox[4 * p + 2], y1 = pbox[4 * p + 3];
        if (cls[p] == ORC_CULLED) continue;
        if (x0 < wx0) x0 = wx0;
        if (x1 > wx1) x1 = wx1;
        if (y0 < wy0) y0 = wy0;
        if (y1 > wy1) y1 = wy1;
        if (cls[p] == ORC_SMALL) {
            if (x0 <= x1 && y0 <= y1) {
                double w = orc_small_weight(sp[p], chi) * col[p];
                double *px_out = image + 3 * ((size_t)y0 * (size_t)W + (size_t)x0);
                for (c = 0; c < 3; ++c) px_out[c] += E[3 * p + c] * w;
            }
            continue;
        }
        for (j = y0; j <= y1; ++j)
            for (i = x0; i <= x1; ++i)
                if (orc_inside(i, j, px[p], py[p], rp[p])) {
                    double w = orc_weight(i, j, px[p], py[p], sp[p]) * col[p];
                    double *px_out = image + 3 * ((size_t)j * (size_t)W + (size_t)i);
                    for (c = 0; c < 3; ++c) px_out[c] += E[3 * p + c] * w;
                }
    }
    if (apply_transfer) {
        for (j = wy0; j <= wy1; ++j)
            for (i = wx0; i <= wx1; ++i) {
                double *q = image + 3 * ((size_t)j * (size_t)W + (size_t)i);
                for (c = 0; c < 3; ++c) q[c] = -expm1(-q[c]);
            }
    }
}

/* ---------------------------------------------------------------------------------------------
 * Ordered mode, E_p != A_p: Eq. 1 for one particle is linear in I, so crossing particle p changes
 * the intensity to  I_out = E/A + (I_in - E/A) exp(-A tau),  tau = col_p w_p.  Particles are
 * crossed one after the other from the farthest to the nearest (r in Eq. 1 runs toward the
 * observer), ordered by the float32 camera depth z_c, ties by lower index first; I starts at 0.
 * A[c] = kappa_p (grey absorption of the particle's species); A == 0 gives I += E tau.
 * order[] is the visiting order (built by orc_depth_order).
 * ------------------------------------------------------------------------------------------- */
typedef struct { float z; int64_t idx; } orc_key;

static int orc_key_cmp(const void *a, const void *b)
{
    const orc_key *ka = (const orc_key *)a, *kb = (const orc_key *)b;
    if (ka->z > kb->z) return -1;
    if (ka->z < kb->z) return 1;
    return (ka->idx > kb->idx) - (ka->idx < kb->idx);
}

int64_t orc_depth_order(int64_t n, const int8_t *cls, const float *zc, int64_t *order)
{
    int64_t p, m = 0;
    orc_key *keys = (orc_key *)malloc(sizeof(orc_key) * (size_t)(n > 0 ? n : 1));
    if (!keys) return -1;
    for (p = 0; p < n; ++p)
        if (cls[p] != ORC_CULLED) { keys[m].z = zc[p]; keys[m].idx = p; ++m; }
    qsort(keys, (size_t)m, sizeof(orc_key), orc_key_cmp);
    for (p = 0; p < m; ++p) order[p] = keys[p].idx;
    free(keys);
    return m;
}

void orc_render_ordered(int64_t m, const int64_t *order, const int8_t *cls,
                        const float *px, const float *py, const float *sp, const float *rp,
                        const int32_t *pbox, const double *E, const double *col, const double *kappa,
                        float chi, int W, int H, int wx0, int wx1, int wy0, int wy1, double *image)
{
    int64_t q;
    int i, j, c;
    (void)H;
    for (q = 0; q < m; ++q) {
        int64_t p = order[q];
        int x0 = pbox[4 * p], x1 = pbox[4 * p + 1], y0 = pbox[4 * p + 2], y1 = pbox[4 * p + 3];
        double A = kappa[p];
        if (x0 < wx0) x0 = wx0;
        if (x1 > wx1) x1 = wx1;
        if (y0 < wy0) y0 = wy0;
        if (y1 > wy1) y1 = wy1;
        for (j = y0; j <= y1; ++j)
            for (i = x0; i <= x1; ++i) {
                double tau;
                double *I = image + 3 * ((size_t)j * (size_t)W + (size_t)i);
                if (cls[p] == ORC_SMALL) tau = orc_small_weight(sp[p], chi) * col[p];
                else if (orc_inside(i, j, px[p], py[p], rp[p]))
                    tau = orc_weight(i, j, px[p], py[p], sp[p]) * col[p];
                else continue;
                for (c = 0; c < 3; ++c) {
                    if (A > 0.0) I[c] += (E[3 * p + c] / A - I[c]) * (-expm1(-A * tau));
                    else I[c] += E[3 * p + c] * tau;
                }
            }
    }
}

/* ---------------------------------------------------------------------------------------------
 * Pre-processing.
 *
 * Normalisation range of a species' colour quantity when the user gives none: "normalization together
 * with other necessary calculations (e.g. for logarithms of processed quantities)";
 * the extrema are "user-specified ... otherwise they are precomputed" (:166 fn. 1).  Plain loop over
 * ALL particles of the species (active or not): v = scalar, or log10(scalar) when use_log10; values
 * that are not finite (NaN, +-Inf, log10 of a non-positive number) are skipped.  The extrema are the
 * float32 values themselves (log10 is taken in double and rounded once to float32, the precision the
 * range is handed on in).  A species without a finite value gets min = 0, max = 1.
 * ------------------------------------------------------------------------------------------- */
void orc_scalar_range(int64_t n, const float *scalar, const int32_t *species_of, int n_species,
                      const int32_t *use_log10, float *vmin /* n_species */, float *vmax /* n_species */)
{
    int64_t p;
    int s;
    for (s = 0; s < n_species; ++s) { vmin[s] = INFINITY; vmax[s] = -INFINITY; }
    for (p = 0; p < n; ++p) {
        float v = scalar[p];
        s = species_of[p];
        if (use_log10[s]) v = (float)log10((double)v);
        if (!(v >= -3.0e38f && v <= 3.0e38f)) continue;      /* NaN and +-Inf are skipped */
        if (v < vmin[s]) vmin[s] = v;
        if (v > vmax[s]) vmax[s] = v;
    }
    for (s = 0; s < n_species; ++s)
        if (!(vmin[s] <= vmax[s])) { vmin[s] = 0.0f; vmax[s] = 1.0f; }
}

/* Vector colour mode: "for velocity v = (v_x, v_y, v_z) we assign rho^R = v_x, rho^G = v_y and
 * rho^B = v_z".  Reading R24 of DESIGN.md: each component is normalised with the
 * species' range like the scalar of the look-up-table mode (:76), t_c = clamp((v_c - min) /
 * (max - min), 0, 1), NaN -> 0, and E[c] = brightness * t_c; the column constant is the one of
 * orc_amplitude.  Overwrites E for the particles of species with vector_mode != 0 only. */
void orc_amplitude_vector(int64_t n, const float *vr, const float *vg, const float *vb,
                          const int32_t *species_of, const int32_t *vector_mode,
                          const double *brightness, const double *smin, const double *smax,
                          double *E /* 3n */)
{
    int64_t p;
    int c;
    for (p = 0; p < n; ++p) {
        int s = species_of[p];
        double v[3];
        if (!vector_mode[s]) continue;
        v[0] = (double)vr[p]; v[1] = (double)vg[p]; v[2] = (double)vb[p];
        for (c = 0; c < 3; ++c) {
            double t = (v[c] - smin[s]) / (smax[s] - smin[s]);
            if (!(t > 0.0)) t = 0.0;
            if (t > 1.0) t = 1.0;
            E[3 * p + c] = brightness[s] * t;
        }
    }
}
