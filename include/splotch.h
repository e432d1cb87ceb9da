/*
 * splotch.h -- C ABI of the B200-native Splotch per-frame particle rendering path.
 *
 * Method: "GPU Accelerated Particle Visualization with Splotch", arxiv 1309.1114.
 * One frame = roto-translation + perspective projection of every particle (Eq. 7 :138),
 * colourisation through a scalar -> RGB look-up table with intensity scaling (:76, :85), classification
 * into inactive / small / medium / large by projected radius r(p) (:156-173), binning of active particles
 * to screen tiles (:164-175) and accumulation of each particle's Gaussian contribution, the solution of the
 * radiative-transfer equation Eq. 1 with the profile of Eq. 2 clipped at chi*sigma (:79-85), into an RGB image.
 * The readings taken where the paper is silent are listed in DESIGN.md ("Readings R1..R23").
 *
 * Conventions
 *   - plain C, no C++/torch types.  Every pointer argument says HOST or DEVICE.
 *   - all functions return 0 (SPLOTCH_OK) or a negative error code; nothing throws or aborts.
 *     splotch_last_error() gives a human-readable message for the last failing call on that context.
 *   - a context is bound to one CUDA device (sm_100 required) and is thread-compatible, not thread-safe.
 *   - the caller owns particle arrays, the image and the workspace (e.g. torch tensors); the library owns
 *     only the context (camera constants, colour tables in device memory, CUDA events).
 *   - there is no CPU fallback: without a CUDA device every compute entry point fails with SPLOTCH_ECUDA.
 */
#ifndef SPLOTCH_H
#define SPLOTCH_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SPLOTCH_OK            0
#define SPLOTCH_EINVAL       -1   /* bad argument (null pointer, n > max_particles, bad fov, bad tile, ...)  */
#define SPLOTCH_ENOMEM       -2   /* workspace too small for the fixed part or for this frame's pairs         */
#define SPLOTCH_ECUDA        -3   /* CUDA runtime error (sticky; message in splotch_last_error)              */
#define SPLOTCH_EDEVICE      -4   /* device is not compute capability 10.x                                   */
#define SPLOTCH_ESTATE       -5   /* camera or a needed colour map not set, or no frame rendered yet         */

#define SPLOTCH_MAX_SPECIES      8
#define SPLOTCH_MAX_LUT_ENTRIES  1024

/* particle classes */
#define SPLOTCH_CULLED  0   /* inactive: "completely outside the scene" (:76), i(p) = -2  */
#define SPLOTCH_SMALL   1   /* r(p) <= r_small, i(p) = N_tiles                            */
#define SPLOTCH_MEDIUM  2   /* r_small < r(p) <= r_large, i(p) = tile of the centre       */
#define SPLOTCH_LARGE   3   /* r(p) > r_large, i(p) = -1                                  */

typedef struct splotch_ctx splotch_ctx;   /* opaque */

/* Particle set, structure of arrays, float32, length n.  "At least three scalars are required representing
 * particle coordinates" plus smoothing length and the quantities that drive intensity and colour
 * (PAPER.md:75, :81-85, :246).  For splotch_render the six arrays are DEVICE pointers, for
 * splotch_render_host they are HOST pointers (pinned memory makes the copies asynchronous).
 * All arrays are read-only for the library and stay owned by the caller.  16-byte aligned arrays take the
 * vectorised load path; any alignment is accepted. */
typedef struct {
    const float *x, *y, *z;          /* world coordinates                                                   */
    const float *h;                  /* smoothing length sigma_p of Eq. 2, world units                      */
    const float *I;                  /* rho_0,p of Eq. 2: the intensity-like quantity                       */
    const float *scalar;             /* quantity mapped through the colour look-up table                    */
    const uint64_t *species_offsets; /* HOST, n_species + 1 ascending entries, [0] = 0, [n_species] = n:
                                        species s owns the index range [off[s], off[s+1]) (Gadget-style
                                        type blocks).  NULL means one species.                */
    int n_species;                   /* 1 .. SPLOTCH_MAX_SPECIES (ignored when species_offsets is NULL)     */
    const float *cr, *cg, *cb;       /* vector quantity (e.g. velocity) for species in vector colour mode:
                                        rho^R = v_x, rho^G = v_y, rho^B = v_z.  Same placement and
                                        length as the other fields; may be NULL when no species uses them.   */
} splotch_particles;

typedef struct {
    float brightness;                /* b_s : E_p = b_s * colour                                            */
    float absorb;                    /* kappa_s : grey absorption A_p, used only when additive == 0         */
    int   use_colormap;              /* 1: colour = LUT_s(scalar)   0: colour = fixed_rgb                   */
    float fixed_rgb[3];
    float scalar_min, scalar_max;    /* user-specified normalisation range (PAPER.md:166 fn. 1)             */
    int   scalar_log10;              /* take log10(scalar) before normalising                 */
    int   auto_range;                /* 1: ignore scalar_min / scalar_max and take the extrema of the species' finite
                                        values, found on the device (PAPER.md:166 fn. 1 "otherwise they are
                                        precomputed"): of the scalar (after log10 if set), or of the three vector
                                        components together in vector colour mode                             */
    int   vector_colour;             /* 1: colour[c] = clamp((v_c - min) / (max - min), 0, 1) from cr, cg, cb
                                        (reading R24); use_colormap is then ignored    */
} splotch_species_params;

typedef struct {
    float chi;                       /* clip factor of Eq. 2; 3.0 is the documented default   */
    float r_small;                   /* r_sml, 0.5 in the paper (:162)                                      */
    float r_large;                   /* r_0 (:160); px                                                      */
    float z_near;                    /* particles with camera depth z_c <= z_near are inactive              */
    int   tile;                      /* tile side t_x = t_y in px (Eq. 8, :164): 8, 16, 32 or 64 (ordered: <= 32) */
    int   additive;                  /* 1: E_p = A_p mode (:85), order independent.  0: ordered E != A mode */
    int   apply_transfer;            /* additive only: 0 -> image = S = sum_p E_p tau_p, 1 -> 1 - exp(-S)   */
    const splotch_species_params *species;  /* HOST, n_species entries                                      */
    int   renderer;                  /* 0: coverage-binned tile renderer (default).  1: the paper's own medium-particle
                                        scheme, for comparison: particles binned to the tile of their
                                        centre, Btile = body + boundary of r_0 in shared memory, blocks of (2 r_0 + 1)^2
                                        threads, three boundary images + composition; additive mode, tile 8 or 16,
                                        r_large = r_0 <= tile (:224)                                           */
    int   btile_np;                  /* renderer 1: particles staged per read, n_p (Table 1, :254-266); 0 = 16 */
} splotch_params;

typedef struct {
    uint64_t n;                      /* particles of the last frame                                         */
    uint64_t count[4];               /* per class, indexed by SPLOTCH_CULLED .. SPLOTCH_LARGE               */
    uint64_t pairs;                  /* (particle, tile) pairs of SMALL + MEDIUM particles (ordered mode:
                                        of all active particles, LARGE ones are binned to tiles as well)    */
    uint64_t large_pairs;            /* (particle, super-tile) pairs of LARGE particles                     */
    uint64_t chunks;                 /* work items of the tile renderer                                     */
    uint64_t pair_capacity;          /* records the workspace could hold                                    */
    int32_t  overflow;               /* 1: pairs + large_pairs > pair_capacity, the image is all zero       */
    int32_t  n_stages;               /* number of valid entries in stage_ms (0 unless profiling is on)      */
    float    stage_ms[8];            /* additive: count, scan, scatter, splat, large, compose; ordered: count, scan,
                                        pairs, sort, bounds, render, combine (see splotch_stage_name)        */
    int32_t  sort_key_bits;          /* ordered mode: bits of the (tile, depth) sort key this frame used;
                                        ceil(bits / 8) radix passes ran.  0 in additive mode                 */
    int32_t  reserved;
} splotch_stats;

/* Create a context for images of width x height on CUDA device `device`; at most max_particles per frame.
 * *out is set on success and must be released with splotch_destroy.  Errors: EINVAL, EDEVICE, ECUDA. */
int splotch_create(splotch_ctx **out, int device, int width, int height, uint64_t max_particles);
int splotch_destroy(splotch_ctx *ctx);

/* Pin-hole camera ("roto-translated and projected according to camera settings").
 * eye, lookat, up: HOST float[3], world units; fov_deg: full horizontal field of view in (0, 180).
 * Errors: EINVAL for eye == lookat, up parallel to the view direction or a bad fov. */
int splotch_set_camera(splotch_ctx *ctx, const float eye[3], const float lookat[3], const float up[3],
                       float fov_deg);

/* The 16 float32 constants the kernels use: right[3], up'[3], forward[3], eye[3], s, c_x, c_y, 0. HOST out. */
int splotch_get_camera_constants(const splotch_ctx *ctx, float out[16]);

/* Colour look-up table of one species: rgb is HOST, n_entries x 3 float32, copied.
 * 2 <= n_entries <= SPLOTCH_MAX_LUT_ENTRIES.  Entries are interpolated linearly, clamped at both ends. */
int splotch_set_colormap(splotch_ctx *ctx, int species, const float *rgb, int n_entries);

/* Record per-stage CUDA-event timings on the render stream during splotch_render.  splotch_get_stats then
 * returns, per stage, the mean over the frames rendered since this call (at most the last 256).  A profiling
 * session covers one mode and one stream: a frame of the other mode, or on another stream, starts it afresh. */
int splotch_set_profiling(splotch_ctx *ctx, int enabled);

/* Bytes of DEVICE scratch splotch_render needs for n particles, a tile side `tile` and room for
 * pair_capacity (particle, tile) records; pair_capacity == 0 picks the default 2 n + 2^20.
 * with_host_staging != 0 adds the staging buffers splotch_render_host needs.  Returns 0 on bad arguments. */
size_t splotch_workspace_bytes(const splotch_ctx *ctx, uint64_t n, int tile, uint64_t pair_capacity,
                               int with_host_staging);

/* Render one frame.  All stages run as CUDA kernels enqueued on `cuda_stream` (a cudaStream_t, NULL = the
 * default stream); the call does not synchronise with the host.
 *   particles  : DEVICE arrays (see splotch_particles), n <= max_particles; n == 0 gives a zero image
 *   image_out  : DEVICE, height x width x 3 float32, row 0 = top, RGB interleaved; overwritten
 *   workspace  : DEVICE scratch of workspace_bytes bytes, 256-byte aligned, caller-owned; its contents
 *                must stay untouched until splotch_get_stats / splotch_debug_tile_counts were called
 * Errors: EINVAL, ESTATE, ENOMEM (workspace below the fixed minimum), ECUDA.  A frame whose pairs exceed the
 * record capacity is reported through splotch_stats.overflow (the image is then all zero).  * All work is enqueued on `cuda_stream` (kernels and memsets only, no synchronisation, no allocation): the call may be
 * captured into a CUDA graph and replayed while the pointers and parameters stay the same. */
int splotch_render(splotch_ctx *ctx, const splotch_particles *particles, uint64_t n,
                   const splotch_params *params, float *image_out,
                   void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Same frame from HOST particle arrays into a HOST image, synchronising the stream before returning.
 * workspace must have been sized with with_host_staging = 1.
 * Additive mode: the paper's per-chunk offload loop (Fig. 3; Eq. 3-4 :111-120) with copy / compute
 * overlap (:354): the set streams through two staging buffers in chunks (splotch_set_host_chunk), the copy of chunk
 * k + 1 runs on a second stream while chunk k is binned and splatted, the chunks' partial images add up exactly in the
 * tiles' fixed-point sums.  Only one chunk's records live in the workspace at a time, so a set whose pairs exceed the
 * workspace's record capacity still renders as long as every chunk's pairs fit (out-of-core rendering).
 * splotch_get_stats then reports the totals of the frame; splotch_debug_tile_counts the last chunk only; per-stage
 * timings are not recorded for chunked frames.
 * Ordered mode: the depth order needs the whole set: one copy in, one frame, one copy out, nothing overlaps. */
int splotch_render_host(splotch_ctx *ctx, const splotch_particles *host_particles, uint64_t n,
                        const splotch_params *params, float *host_image_out,
                        void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Particles per chunk of splotch_render_host (additive mode).  0 (the default) picks about four chunks of 2^20 ..
 * 2^27 particles.  The staging buffers of the workspace are sized for this value: set it before asking
 * splotch_workspace_bytes. */
int splotch_set_host_chunk(splotch_ctx *ctx, uint64_t particles_per_chunk);

/* Statistics of the last frame.  Synchronises the stream of that frame.  HOST out. */
int splotch_get_stats(splotch_ctx *ctx, splotch_stats *out);
const char *splotch_stage_name(int additive, int stage);   /* stage names of an additive / ordered frame */

/* image <- 1 - exp(-image) in place (DEVICE, height x width x 3 float32): the exact E = A transfer for a
 * frame whose partial images S were rendered with apply_transfer = 0 and summed elsewhere, e.g. by the image all-reduce of
 * a particle-sharded multi-GPU frame.  Asynchronous on `cuda_stream`. */
int splotch_apply_transfer(splotch_ctx *ctx, float *image, void *cuda_stream);

/* The two ALU rates the splat stages' roofline fractions are quoted against, measured on this context's device by
 * a register-only microbenchmark: out[0] = FP32 FMA lane-operations per second (one FMA = one
 * operation), out[1] = ex2.approx results per second, whole GPU.  HOST out; synchronises `cuda_stream`. */
int splotch_measure_peaks(splotch_ctx *ctx, double out[2], void *cuda_stream);

/* Test hooks: the per-particle results of the classification stage, written to DEVICE arrays of length n
 * (any may be NULL): cls int8; px, py (screen centre), sp (sigma in px), rp (r(p)), zc (camera depth)
 * float32; pbox int32[4] = x0 x1 y0 y1 (pixel box, inclusive); tbox int32[4] = tile box; ilabel = the
 * paper's tile index i(p). */
int splotch_debug_geometry(splotch_ctx *ctx, const splotch_particles *particles, uint64_t n,
                           const splotch_params *params, int8_t *cls, float *px, float *py, float *sp,
                           float *rp, float *zc, int32_t *pbox, int32_t *tbox, int32_t *ilabel,
                           void *cuda_stream);
/* Per-tile pair counts of the last frame: DEVICE out, nty x ntx uint32 (SMALL + MEDIUM; ordered mode: all). */
int splotch_debug_tile_counts(splotch_ctx *ctx, uint32_t *out, void *cuda_stream);

/* The image of a particle-sharded frame ("chunks of particles among different processors, each ... producing a
 * partial rendering, the root processor composing final renderings") from the shards' workspaces, in ONE kernel: every shard
 * was rendered with splotch_render (additive mode, same image size and tile) into its own workspace, which then holds the tiles'
 * exact 64-bit fixed-point sums; this call adds them per pixel (in double precision: the result does not depend on the order of
 * the shards) and writes tiles [tile_begin, tile_end) of the image (tile_end < 0: all tiles), with the transfer 1 - exp(-S)
 * when apply_transfer != 0.  It replaces the float32 partial images and their all-reduce.
 *   workspaces : HOST array of n_shards (<= 16) DEVICE pointers, the workspaces the shards were rendered into, untouched since.
 *                They may be peer-mapped memory of other GPUs (peer access enabled by the caller): the loads then cross
 *                NVLink and a rank can compose its own share of the tiles.
 *   image_out  : DEVICE, height x width x 3 float32 of this context's image size; only the tiles of the range are written.
 * A shard whose frame overflowed its pair capacity makes the composed tiles zero.  Asynchronous on `cuda_stream`. */
int splotch_compose_shards(splotch_ctx *ctx, const void *const *workspaces, int n_shards, int tile, int tile_begin,
                           int tile_end, int apply_transfer, float *image_out, void *cuda_stream);

/* Classes and per-tile pair counts of a particle set (steps A1, A3, A4a: PAPER.md:76, :138, :156-173 and the counting half
 * of :175) for callers that cannot allocate: the call makes NO allocation (no cudaMalloc / cudaFree, no allocating library
 * routine) and takes no workspace.  Its scratch, the count matrix, is a file-scope device array of 16 MiB inside the library
 * (held on every GPU that loads the library until the process exits); splotch_create looks its address up once per device.
 *   particles        : DEVICE arrays as for splotch_render (x, y, z, h are read), n <= max_particles
 *   params           : additive != 0, renderer == 0; tile, chi, r_small, r_large, z_near as for splotch_render
 *   tile_counts_out  : DEVICE, nty x ntx uint32: (particle, tile) pairs per tile, SMALL + MEDIUM (what
 *                      splotch_debug_tile_counts reports after an additive frame); overwritten
 *   class_counts_out : DEVICE, uint64[4] = {culled, small, medium, large} (splotch_stats.count); overwritten
 * Limit: 4 x (bins + 4) x SMs bytes must fit in the 16 MiB, bins = 2 x tiles + super-tiles (+ tiles with 32-px tiles): at
 * most about 28,000 bins on a 148-SM GPU (1920 x 1080 at 16 px fits, 4096 x 4096 needs 64-px tiles).  Larger requests return
 * SPLOTCH_EINVAL and splotch_last_error says so.
 * All calls share the array and it keeps the last call's contents; every call clears the part it uses first.  Calls that
 * overlap on the GPU (other streams, other contexts of the same device) race: serialise them.  Enqueues on `cuda_stream`
 * without synchronising, like splotch_render. */
int splotch_count_static(splotch_ctx *ctx, const splotch_particles *particles, uint64_t n,
                         const splotch_params *params, uint32_t *tile_counts_out, uint64_t *class_counts_out,
                         void *cuda_stream);

const char *splotch_last_error(const splotch_ctx *ctx);
const char *splotch_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPLOTCH_H */
