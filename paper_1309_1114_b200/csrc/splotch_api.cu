// splotch_api.cu -- host side of the C ABI declared in include/splotch.h.
// Argument checking, camera constants, workspace layout and the per-frame kernel sequence.  No compute happens on
// the host: every stage of the path is one of the kernels in splotch_kernels.cuh.
#include "splotch_kernels.cuh"
#include "splotch_splat.cuh"
#include "splotch_large.cuh"
#include "splotch_ordered.cuh"
#include "splotch_peaks.cuh"
#include "splotch_btile.cuh"
#include "../../include/splotch.h"

#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>
#include <new>

using namespace splotch;

// ---- splotch_count_static: the one entry point that allocates nothing ------------------------------------------------
// Its scratch (the count matrix of the classify-and-count stage) lives in this file-scope device array instead of a
// caller-owned workspace: 16 MiB on every GPU that loads the library, until the process exits.  In HOST code the name
// g_static_scratch is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, once per device with that device current (static_scratch_address, called by splotch_create).
// Every call shares the array and it keeps the last call's contents: the call clears the part it uses, and calls that
// overlap on the GPU (two streams, two contexts of one device) race.
constexpr size_t kStaticScratchBytes = 16u << 20;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

// per-tile pair counts (the tile's SMALL, MEDIUM and, with 32-px tiles, wide-MEDIUM bins summed over the rows of the count
// matrix) and the class totals {particles, SMALL, MEDIUM, LARGE}; k_static_count_finish turns the first into CULLED
__global__ void __launch_bounds__(256)
k_static_count_reduce(const unsigned int *__restrict__ counts, const unsigned int *__restrict__ cls_counts, int nrows,
                      int nbins, int n_tiles, int n_super, int n_big, unsigned int *__restrict__ tile_out,
                      unsigned long long *__restrict__ class_out)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned int small = 0u;
    if (t < n_tiles) {
        unsigned int med = 0u, wide = 0u;
        for (int r = 0; r < nrows; ++r) {
            const unsigned int *row = counts + (size_t)r * nbins;
            med += row[2 * t]; small += row[2 * t + 1];
            if (n_big) wide += row[2 * n_tiles + n_super + t];
        }
        tile_out[t] = med + small + wide;
    }
    small = __reduce_add_sync(0xffffffffu, small);
    if ((threadIdx.x & 31) == 0 && small) atomicAdd(class_out + 1, (unsigned long long)small);
    if (blockIdx.x == 0) {
        unsigned long long tot = 0ull, med = 0ull, large = 0ull;
        for (int r = threadIdx.x; r < nrows; r += blockDim.x) { tot += cls_counts[4 * r]; med += cls_counts[4 * r + 2]; large += cls_counts[4 * r + 3]; }
        if (tot) atomicAdd(class_out + 0, tot);
        if (med) atomicAdd(class_out + 2, med);
        if (large) atomicAdd(class_out + 3, large);
    }
}

__global__ void k_static_count_finish(unsigned long long *class_out)
{
    class_out[0] -= class_out[1] + class_out[2] + class_out[3];       // particles -> CULLED
}

namespace {

constexpr int kStages = 7;                  // most stages a frame has (ordered mode); additive frames have 5
constexpr int kStagesAdditive = 6, kStagesOrdered = 7;
constexpr int kProfRing = 256;              // frames of per-stage events kept while profiling
const char *kStageNamesAdditive[kStagesAdditive] = {"count", "scan", "scatter", "splat", "large", "compose"};
const char *kStageNamesOrdered[kStagesOrdered] = {"count", "scan", "pairs", "sort", "bounds", "render", "combine"};

struct Layout {
    size_t ranges, planes, planes_bytes, counts, counts_bytes, cursors, cls_counts, bin_count, vstart, large_off, run, stats, accum, accum_bytes, records, staging, total;
    bool ghist;
    unsigned long long capacity;
    int nrows;
    // ordered mode
    size_t blk_pairs, tile_start, rec, keys[2], vals[2], hist, sums, seg;
    int nblk_o, nblk_rs, n_sums;
    unsigned int m_hist;
};

}  // namespace

struct splotch_ctx {
    int device = 0, width = 0, height = 0;
    unsigned long long max_particles = 0;
    int n_sm = 0, smem_optin = 0;
    bool camera_set = false;
    float cam[16] = {0};
    float4 *lut = nullptr;                   // device, [kMaxSpecies][kMaxLut]
    unsigned char *static_scratch = nullptr; // device address of g_static_scratch on this context's device
    int lut_n[kMaxSpecies] = {0};
    bool profiling = false;
    cudaEvent_t (*ev_ring)[kStages + 1] = nullptr;   // [kProfRing][kStages + 1], created when profiling is first enabled
    cudaEvent_t *ev = nullptr;                       // slot of the frame being recorded
    unsigned long long prof_frames = 0;              // frames recorded since profiling was (re)enabled
    // last frame
    bool have_frame = false;
    char *ws = nullptr;
    Layout lay{};
    FrameParams fp{};
    unsigned long long last_n = 0;
    bool last_additive = true;
    int prof_stages = kStagesAdditive;              // stages of the frames recorded since profiling was enabled
    cudaStream_t last_stream = nullptr;
    unsigned long long host_chunk = 0;       // particles per chunk of splotch_render_host (0: automatic)
    cudaStream_t copy_stream = nullptr;      // host-to-device copies of splotch_render_host run here, beside the kernels
    cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_consumed[2] = {nullptr, nullptr}, ev_start = nullptr;
    int splat_blocks_per_sm[4] = {0, 0, 0, 0};  // T = 8, 16, 32, 64
    int orender_blocks_per_sm[3] = {0, 0, 0};
    int large_blocks_per_sm = 0;
    char err[512] = {0};
};

namespace {

char g_create_err[512] = "";               // last splotch_create failure (there is no context to hold it)

int fail(splotch_ctx *c, int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(c ? c->err : g_create_err, sizeof g_create_err, fmt, ap);
    va_end(ap);
    return code;
}

#define CU_TRY(ctx, expr)                                                                               \
    do {                                                                                                \
        cudaError_t e_ = (expr);                                                                        \
        if (e_ != cudaSuccess)                                                                          \
            return fail(ctx, SPLOTCH_ECUDA, "%s failed: %s", #expr, cudaGetErrorString(e_));           \
    } while (0)

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

int tile_shift(int T) { return T == 8 ? 3 : T == 16 ? 4 : T == 32 ? 5 : T == 64 ? 6 : -1; }

// Device address of g_static_scratch on `device` (which must be current): looked up once per device and kept.
int static_scratch_address(splotch_ctx *c, int device, unsigned char **out)
{
    static unsigned char *ptr_of_device[64] = {nullptr};
    if (device < 0 || device >= 64) return fail(c, SPLOTCH_EINVAL, "device index %d out of range", device);
    if (!ptr_of_device[device]) {
        unsigned char *ptr = nullptr;
        CU_TRY(c, cudaGetSymbolAddress((void **)&ptr, g_static_scratch));
        ptr_of_device[device] = ptr;
    }
    *out = ptr_of_device[device];
    return SPLOTCH_OK;
}

// LARGE particles are binned to super-tiles of 8 x 8 tiles, at most 128 px a side (record boxes are 8 bits per bound)
int super_shift(int T) { const int s = tile_shift(T) + kSuperShift; return s < kSuperMaxShift ? s : kSuperMaxShift; }

size_t hist_bytes(int W, int H, int T)
{
    const int ntx = (W + T - 1) / T, nty = (H + T - 1) / T;
    const int S = 1 << super_shift(T);
    const int nsx = (W + S - 1) / S, nsy = (H + S - 1) / S;
    // two bins per tile (MEDIUM, SMALL) + one per super-tile + with 32-px tiles one more per tile (wide MEDIUM discs, k_large's)
    return sizeof(unsigned int) * (2 * (size_t)ntx * nty + (size_t)nsx * nsy + (T == 32 ? (size_t)ntx * nty : 0));
}

// dynamic shared memory of k_count / k_scatter: the block's histogram / cursors plus room for the colour tables
size_t bin_smem_bytes(int W, int H, int T) { return hist_bytes(W, H, T) + 16 + sizeof(float4) * kLutSmemMax; }

// images with more bins than fit in shared memory (4096^2 at 16 px: 131,072 + 1,024 bins) keep the histogram / cursors
// in the block's row of the count matrix instead (global atomics, L2 resident)
bool use_global_hist(const splotch_ctx *c, int T);

bool use_global_hist(const splotch_ctx *c, int T) { return bin_smem_bytes(c->width, c->height, T) + 1024 > (size_t)c->smem_optin; }

int bin_rows(const splotch_ctx *c, int T)
{
    (void)T;
    return c->n_sm;                         // one 1024-thread CTA per SM, each with a private histogram over all bins
}

constexpr int kHostFields = 9;

// Particles per chunk of a chunked host frame: about four chunks, between 2^20 and 2^27 particles, a multiple of 4
unsigned long long host_chunk_particles(const splotch_ctx *c, unsigned long long n)
{
    unsigned long long ch = c->host_chunk;
    if (ch == 0) {
        ch = (n + 3) / 4;
        if (ch < (1ull << 20)) ch = 1ull << 20;
        if (ch > (1ull << 27)) ch = 1ull << 27;
    }
    ch = (ch + 3) / 4 * 4;
    return ch < n ? ch : (n + 3) / 4 * 4;
}

// staging of splotch_render_host: two buffers of six fields for one chunk each (additive) or one buffer for the whole
// set (ordered), then the device image
size_t staging_bytes(const splotch_ctx *c, unsigned long long n, bool additive)
{
    const unsigned long long per = additive ? host_chunk_particles(c, n) : n;
    const size_t fields = kHostFields * align_up(sizeof(float) * per, 256) * (additive ? 2 : 1);     // six fields + the vector components
    return align_up(fields, 256) + align_up(sizeof(float) * 3 * (size_t)c->width * c->height, 256);
}

// Workspace layout.  Either `capacity` is given (sizing query) or derived from `bytes` (render).
bool make_layout(const splotch_ctx *c, unsigned long long n, int T, unsigned long long capacity, size_t bytes,
                 bool staging, Layout *L)
{
    const int ntx = (c->width + T - 1) / T, nty = (c->height + T - 1) / T;
    const size_t n_tiles = (size_t)ntx * nty;
    const size_t nbins = hist_bytes(c->width, c->height, T) / sizeof(unsigned int);
    L->nrows = bin_rows(c, T);
    L->ghist = use_global_hist(c, T);
    size_t off = 0;
    L->ranges = off;      off = align_up(off + (sizeof(RangeRaw) + sizeof(float2)) * kMaxSpecies, 256);
    // partial images of the paper's Btile renderer (tiles of 8 or 16 px only)
    L->planes = off;      L->planes_bytes = T <= 16 ? sizeof(float) * 3 * kBtilePlanes * (size_t)c->width * c->height : 0; off = align_up(off + L->planes_bytes, 256);
    L->counts = off;      L->counts_bytes = sizeof(unsigned int) * nbins * L->nrows; off = align_up(off + L->counts_bytes, 256);
    L->cursors = off;     if (L->ghist) off = align_up(off + L->counts_bytes, 256);      // k_scatter's cursors when they do not fit in shared memory
    L->cls_counts = off;  off = align_up(off + sizeof(unsigned int) * 4 * L->nrows, 256);
    L->bin_count = off;   off = align_up(off + sizeof(unsigned int) * nbins, 256);
    L->vstart = off;      off = align_up(off + sizeof(unsigned int) * (nbins + 1), 256);
    L->large_off = off;   off = align_up(off + sizeof(unsigned int) * (nbins - 2 * n_tiles + 1), 256);
    L->run = off;         off = align_up(off + sizeof(uint2) * kMaxSlabs * nbins, 256);
    // DeviceStats and the tiles' 64-bit sums sit together: one memset clears both before every frame
    L->stats = off;       off = align_up(off + sizeof(DeviceStats), 256);
    L->accum = off;
    L->accum_bytes = sizeof(unsigned long long) * 3 * (size_t)T * T * n_tiles;
    off = align_up(off + L->accum_bytes, 256);
    L->staging = off;
    if (staging) off = align_up(off + staging_bytes(c, n, true), 256);
    // every run of SMALL records may be padded by one 16-byte unit (k_layout): an allowance beside the capacity
    const size_t pad = align_up(16 * (size_t)kMaxSlabs * n_tiles + 16 * nbins, 256);
    const size_t fixed = off + pad;
    if (capacity == 0) {
        // derive from bytes: capacity * 32 <= bytes - fixed - reserve
        const size_t need0 = fixed + 8192;
        if (bytes < need0) return false;
        capacity = (unsigned long long)((bytes - need0) / 32);
        if (capacity > 0x7ff00000ull) capacity = 0x7ff00000ull;            // 16-byte unit offsets are 32 bits
    }
    L->capacity = capacity;
    L->records = off;  off = align_up(off + 32ull * capacity + pad, 256);
    L->total = off;
    return bytes == 0 || off <= bytes;
}

// Workspace layout of the ordered mode for a given pair capacity.
void make_layout_ordered(const splotch_ctx *c, unsigned long long n, int T, unsigned long long capacity, bool staging, Layout *L)
{
    const int ntx = (c->width + T - 1) / T, nty = (c->height + T - 1) / T;
    const size_t n_tiles = (size_t)ntx * nty;
    L->capacity = capacity;
    L->nblk_o = (int)((n + kOBlockParticles - 1) / kOBlockParticles);
    L->nblk_rs = (int)((capacity + kRsTile - 1) / kRsTile);
    if (L->nblk_rs < 1) L->nblk_rs = 1;
    L->m_hist = 256u * (unsigned int)L->nblk_rs;
    L->n_sums = (int)((L->m_hist + kScTile - 1) / kScTile);
    size_t off = 0;
    L->ranges = off;      off = align_up(off + (sizeof(RangeRaw) + sizeof(float2)) * kMaxSpecies, 256);
    L->stats = off;       off = align_up(off + sizeof(DeviceStats), 256);
    L->blk_pairs = off;   off = align_up(off + sizeof(unsigned int) * (size_t)(L->nblk_o + 1), 256);
    L->tile_start = off;  off = align_up(off + sizeof(unsigned int) * (n_tiles + 1), 256);
    L->hist = off;        off = align_up(off + sizeof(unsigned int) * (size_t)L->m_hist, 256);
    L->sums = off;        off = align_up(off + sizeof(unsigned int) * (size_t)L->n_sums, 256);
    L->rec = off;         off = align_up(off + 32ull * n, 256);
    L->staging = off;
    if (staging) off = align_up(off + staging_bytes(c, n, false), 256);
    for (int k = 0; k < 2; ++k) { L->keys[k] = off; off = align_up(off + 8ull * capacity, 256); }
    for (int k = 0; k < 2; ++k) { L->vals[k] = off; off = align_up(off + 4ull * capacity, 256); }
    // one (t, c_R, c_G, c_B) per pixel and segment; segment slot = chunk + tile; k_oscan cuts the pairs into at most
    // 128 chunks per SM, or capacity / kOChunkMax when that is more
    L->seg = off;
    {
        const size_t by_sm = (size_t)c->n_sm * 128, by_cap = (size_t)(capacity / kOChunkMax) + 1;
        const size_t by_min = (size_t)(capacity / kOChunkMin) + 1;             // no chunk is shorter than kOChunkMin
        size_t chunks = by_sm > by_cap ? by_sm : by_cap;
        if (chunks > by_min) chunks = by_min;
        off = align_up(off + sizeof(float4) * (size_t)T * T * (chunks + n_tiles + 2), 256);
    }
    L->total = off;
}

// Largest capacity whose ordered layout fits in `bytes` (0 if not even an empty frame fits).
bool fit_layout_ordered(const splotch_ctx *c, unsigned long long n, int T, size_t bytes, bool staging, Layout *L)
{
    make_layout_ordered(c, n, T, 0, staging, L);
    if (L->total + 8192 > bytes) return false;
    unsigned long long lo = 0, hi = 0xfffffff0ull;
    while (lo < hi) {
        const unsigned long long mid = lo + (hi - lo + 1) / 2;
        make_layout_ordered(c, n, T, mid, staging, L);
        if (L->total + 8192 <= bytes) lo = mid; else hi = mid - 1;
    }
    make_layout_ordered(c, n, T, lo, staging, L);
    return true;
}

template <int T>
int query_splat_occupancy(splotch_ctx *c, int *out)
{
    CU_TRY(c, cudaFuncSetAttribute(k_splat<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Splat2Cfg<T>::kSmemBytes));
    CU_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(out, k_splat<T>, Splat2Cfg<T>::kThreads, Splat2Cfg<T>::kSmemBytes));
    if (*out < 1) *out = 1;
    return SPLOTCH_OK;
}

int check_params(splotch_ctx *c, const splotch_particles *p, unsigned long long n, const splotch_params *q,
                 FrameParams *fp)
{
    if (!p || !q) return fail(c, SPLOTCH_EINVAL, "null particles or params");
    if (n > c->max_particles) return fail(c, SPLOTCH_EINVAL, "n = %llu exceeds max_particles = %llu", n, c->max_particles);
    if (n > 0 && (!p->x || !p->y || !p->z || !p->h || !p->I || !p->scalar))
        return fail(c, SPLOTCH_EINVAL, "null particle field");
    if (!c->camera_set) return fail(c, SPLOTCH_ESTATE, "camera not set");
    const int ts = tile_shift(q->tile);
    if (ts < 0) return fail(c, SPLOTCH_EINVAL, "tile must be 8, 16, 32 or 64 (got %d)", q->tile);
    if (!q->additive && q->tile == 64) return fail(c, SPLOTCH_EINVAL, "the ordered mode takes tiles of 8, 16 or 32 px");
    if (!(q->chi > 0.0f) || !(q->r_small >= 0.0f) || !(q->r_small < q->r_large))
        return fail(c, SPLOTCH_EINVAL, "need chi > 0 and 0 <= r_small < r_large");
    if (!q->additive)
        for (int s = 0; s < (p->species_offsets ? p->n_species : 1) && s < kMaxSpecies && q->species; ++s)
            if (!(q->species[s].absorb >= 0.0f)) return fail(c, SPLOTCH_EINVAL, "species %d: absorb must be >= 0", s);
    const int ns = p->species_offsets ? p->n_species : 1;
    if (ns < 1 || ns > kMaxSpecies) return fail(c, SPLOTCH_EINVAL, "n_species must be 1..%d", kMaxSpecies);
    if (!q->species) return fail(c, SPLOTCH_EINVAL, "null species parameters");
    memset(fp, 0, sizeof *fp);
    memcpy(fp->cam, c->cam, sizeof fp->cam);
    fp->chi = q->chi; fp->r_small = q->r_small; fp->r_large = q->r_large; fp->z_near = q->z_near;
    fp->W = c->width; fp->H = c->height; fp->fW = (float)c->width; fp->fH = (float)c->height;
    fp->fWm1 = (float)(c->width - 1); fp->fHm1 = (float)(c->height - 1);
    fp->csmall = (float)(3.14159265358979323846 * (1.0 - exp(-(double)q->chi * (double)q->chi)));
    fp->T = q->tile; fp->tshift = ts;
    fp->ntx = (c->width + q->tile - 1) / q->tile; fp->nty = (c->height + q->tile - 1) / q->tile;
    fp->n_tiles = fp->ntx * fp->nty;
    fp->sshift = super_shift(q->tile);
    const int S = 1 << fp->sshift;
    fp->nsx = (c->width + S - 1) / S; fp->nsy = (c->height + S - 1) / S;
    fp->n_super = fp->nsx * fp->nsy;
    fp->n_big = (q->tile == 32 && q->renderer == 0) ? fp->n_tiles : 0;
    fp->r_route = kRouteRadius;
    fp->nbins = 2 * fp->n_tiles + fp->n_super + (q->tile == 32 ? fp->n_tiles : 0);       // the bins exist with 32-px tiles (workspace layout), used when n_big > 0
    if (q->renderer != 0 && q->renderer != 1) return fail(c, SPLOTCH_EINVAL, "renderer must be 0 (default) or 1 (the paper's Btile scheme)");
    if (q->renderer == 1) {
        // the paper's constraints: additive mode (:85), r_0 <= min(t_x, t_y) (:224); the Btile must fit the 6-bit box fields
        const int r0 = (int)ceilf(q->r_large);
        if (!q->additive || q->tile > 16 || r0 > q->tile || r0 < 1)
            return fail(c, SPLOTCH_EINVAL, "the Btile renderer needs additive mode, tile 8 or 16 and 1 <= r_large <= tile");
        fp->btile = 1; fp->btile_r0 = r0; fp->btile_np = q->btile_np > 0 ? (q->btile_np < 256 ? q->btile_np : 256) : 16;
    }
    fp->additive = q->additive ? 1 : 0;
    fp->apply_transfer = q->apply_transfer ? 1 : 0;
    fp->n_species = ns;
    fp->lut = c->lut;
    for (int s = 0; s <= ns; ++s) {
        const unsigned long long o = p->species_offsets ? p->species_offsets[s] : (s == 0 ? 0ull : n);
        if ((s == 0 && o != 0) || (s == ns && o != n) || (s > 0 && o < fp->sp_begin[s - 1]))
            return fail(c, SPLOTCH_EINVAL, "species_offsets must ascend from 0 to n");
        fp->sp_begin[s] = (unsigned int)o;
    }
    int lut_total = 0;
    for (int s = 0; s < ns; ++s) {
        const splotch_species_params &sp = q->species[s];
        SpeciesDev &d = fp->sp[s];
        d.brightness = sp.brightness; d.absorb = sp.absorb;
        d.fixed_r = sp.fixed_rgb[0]; d.fixed_g = sp.fixed_rgb[1]; d.fixed_b = sp.fixed_rgb[2];
        d.vector = sp.vector_colour ? 1 : 0; d.auto_range = sp.auto_range ? 1 : 0;
        d.use_colormap = (sp.use_colormap && !d.vector) ? 1 : 0; d.use_log10 = sp.scalar_log10 ? 1 : 0;
        if (d.vector) { fp->any_vector = 1; d.use_log10 = 0; }
        if (d.auto_range) fp->any_auto = 1;
        d.smin = sp.scalar_min;
        d.inv_range = (float)(1.0 / ((double)sp.scalar_max - (double)sp.scalar_min));
        d.lut_n = c->lut_n[s];
        d.lut_nm1 = (float)(d.lut_n - 1); d.lut_nm2 = (float)(d.lut_n - 2);
        d.lut_off = lut_total;
        if (d.use_colormap) lut_total += d.lut_n;
        if (d.use_colormap) {
            if (d.lut_n < 2) return fail(c, SPLOTCH_ESTATE, "species %d uses a colour map but none was set", s);
            if (!d.auto_range && !(sp.scalar_max != sp.scalar_min)) return fail(c, SPLOTCH_EINVAL, "species %d: scalar_min == scalar_max", s);
        }
        if (d.vector && !d.auto_range && !(sp.scalar_max != sp.scalar_min)) return fail(c, SPLOTCH_EINVAL, "species %d: scalar_min == scalar_max", s);
    }
    fp->lut_total = lut_total <= kLutSmemMax ? lut_total : 0;      // larger tables are read from global memory
    if (fp->any_vector && n > 0 && (!p->cr || !p->cg || !p->cb)) return fail(c, SPLOTCH_EINVAL, "a species is in vector colour mode but cr / cg / cb are null");
    fp->vec[0] = p->cr; fp->vec[1] = p->cg; fp->vec[2] = p->cb;
    return SPLOTCH_OK;
}

bool aligned16(const splotch_particles *p)
{
    const uintptr_t m = (uintptr_t)p->x | (uintptr_t)p->y | (uintptr_t)p->z | (uintptr_t)p->h | (uintptr_t)p->I |
                        (uintptr_t)p->scalar;
    return (m & 15u) == 0;
}

template <int T>
int launch_render_tail(splotch_ctx *c, const Layout &L, char *ws, const FrameParams &fp, float *image, cudaStream_t st, bool prof, bool compose)
{
    const int ti = T == 8 ? 0 : T == 16 ? 1 : T == 32 ? 2 : 3;
    const int grid = c->n_sm * c->splat_blocks_per_sm[ti];
    if (fp.btile) {
        const int side = T + 2 * fp.btile_r0, B = 2 * fp.btile_r0 + 1;
        const int threads = ((B * B + 31) / 32 * 32) < 1024 ? (B * B + 31) / 32 * 32 : 1024;
        const size_t smem = sizeof(float) * ((3 * side * side + 3) & ~3) + 32 * (size_t)fp.btile_np;
        k_btile<<<fp.n_tiles, threads, smem, st>>>((const float4 *)(ws + L.records), (const uint2 *)(ws + L.run), (const DeviceStats *)(ws + L.stats),
                                                  (float *)(ws + L.planes), fp);
    } else {
        k_splat<T><<<grid, Splat2Cfg<T>::kThreads, Splat2Cfg<T>::kSmemBytes, st>>>(
            (const float4 *)(ws + L.records), (const unsigned int *)(ws + L.vstart), (const uint2 *)(ws + L.run), (DeviceStats *)(ws + L.stats),
            (unsigned long long *)(ws + L.accum), fp);
    }
    if (prof) cudaEventRecord(c->ev[4], st);
    k_large<<<c->n_sm * c->large_blocks_per_sm, kLargeThreads, sizeof(LargeSmem), st>>>(
        (const float4 *)(ws + L.records), (const unsigned int *)(ws + L.bin_count), (const uint2 *)(ws + L.run), (const unsigned int *)(ws + L.large_off),
        (DeviceStats *)(ws + L.stats), (unsigned long long *)(ws + L.accum), fp);
    if (prof) cudaEventRecord(c->ev[5], st);
    if (compose && fp.btile) {
        FrameParams fl = fp;
        fl.apply_transfer = 0;                    // the transfer comes after the partial images are added
        k_compose<T><<<fp.n_tiles, 256, 0, st>>>((const unsigned long long *)(ws + L.accum), (const DeviceStats *)(ws + L.stats), fl, image);
        k_btile_compose<<<4 * c->n_sm, 256, 0, st>>>((const float *)(ws + L.planes), 3 * (size_t)fp.W * fp.H, fp.apply_transfer, image);
    } else if (compose) {
        k_compose<T><<<fp.n_tiles, 256, 0, st>>>((const unsigned long long *)(ws + L.accum), (const DeviceStats *)(ws + L.stats), fp, image);
    }
    if (prof) cudaEventRecord(c->ev[6], st);
    return SPLOTCH_OK;
}

template <bool AL, bool GH, bool BT>
void launch_bin_kernels_count(const Layout &L, size_t hbytes, const splotch_particles *p, unsigned long long n, unsigned long long per,
                              const FrameParams &fp, unsigned int *counts, unsigned int *cls_counts, cudaStream_t st)
{
    k_count<AL, GH, BT><<<L.nrows, kBinThreads, GH ? 0 : hbytes, st>>>(p->x, p->y, p->z, p->h, n, per, fp, counts, cls_counts);
}

template <bool AL, bool GH, bool BT>
void launch_bin_kernels_scatter(const Layout &L, size_t hbytes, const splotch_particles *p, unsigned long long n, unsigned long long per,
                                const FrameParams &fp, unsigned int *counts, unsigned int *cursors, const uint2 *run, DeviceStats *stats,
                                float4 *records, cudaStream_t st)
{
    k_scatter<AL, GH, BT><<<L.nrows, kBinThreads, GH ? sizeof(float4) * kLutSmemMax : hbytes, st>>>(p->x, p->y, p->z, p->h, p->I, p->scalar, n, per, fp,
                                                                                               counts, cursors, run, stats, records);
}

// the eight variants: 16-byte aligned fields or not, histogram in shared memory or in the count matrix, default or Btile binning
#define SPLOTCH_DISPATCH3(fn, al, gh, bt, ...)                                                                          \
    do {                                                                                                                \
        if (al) { if (gh) { if (bt) fn<true, true, true>(__VA_ARGS__); else fn<true, true, false>(__VA_ARGS__); }       \
                  else    { if (bt) fn<true, false, true>(__VA_ARGS__); else fn<true, false, false>(__VA_ARGS__); } }   \
        else    { if (gh) { if (bt) fn<false, true, true>(__VA_ARGS__); else fn<false, true, false>(__VA_ARGS__); }     \
                  else    { if (bt) fn<false, false, true>(__VA_ARGS__); else fn<false, false, false>(__VA_ARGS__); } } \
    } while (0)

// Normalisation ranges found on the device (PAPER.md:166 fn. 1) for the species with auto_range: particles [lo, lo + len) of
// the set the pointers of `p` address; species ranges sp_begin are relative to that set.  init / finish bracket the passes.
void range_pass(splotch_ctx *c, const splotch_particles *p, unsigned long long len, const FrameParams &fp, char *ws, const Layout &L,
                cudaStream_t st, bool init, bool finish)
{
    RangeRaw *raw = (RangeRaw *)(ws + L.ranges);
    float2 *rng = (float2 *)(raw + kMaxSpecies);
    if (init) k_range_init<<<1, 32, 0, st>>>(raw);
    for (int s = 0; s < fp.n_species && len > 0; ++s) {
        if (!fp.sp[s].auto_range) continue;
        const unsigned long long b = fp.sp_begin[s], e = fp.sp_begin[s + 1] < len ? fp.sp_begin[s + 1] : len;
        if (b >= e) continue;
        const unsigned long long cnt = e - b;
        const int grid = (int)((cnt + 511) / 512 < (unsigned long long)(8 * c->n_sm) ? (cnt + 511) / 512 : 8 * c->n_sm);
        if (fp.sp[s].vector) {
            const float *v[3] = {p->cr, p->cg, p->cb};
            for (int k = 0; k < 3; ++k) k_minmax<<<grid, 512, 0, st>>>(v[k] + b, cnt, 0, raw, s);
        } else {
            k_minmax<<<grid, 512, 0, st>>>(p->scalar + b, cnt, fp.sp[s].use_log10, raw, s);
        }
    }
    if (finish) k_range_finish<<<1, 32, 0, st>>>(raw, rng);
}

struct ChunkCtl { bool first, last, chunked; };     // one-shot frame: {true, true, false}

int render_device(splotch_ctx *c, const splotch_particles *p, unsigned long long n, const FrameParams &fp,
                  const Layout &L, float *image, char *ws, cudaStream_t st, ChunkCtl ctl = {true, true, false})
{
    const bool al = aligned16(p);
    const bool prof = c->profiling && !ctl.chunked;          // per-stage events describe one-shot frames
    const size_t hbytes = bin_smem_bytes(fp.W, fp.H, fp.T);
    unsigned long long per = (n + L.nrows - 1) / L.nrows;
    per = (per + 3) / 4 * 4;
    if (per == 0) per = 4;
    unsigned int *counts = (unsigned int *)(ws + L.counts);
    unsigned int *cls_counts = (unsigned int *)(ws + L.cls_counts);
    unsigned int *bin_count = (unsigned int *)(ws + L.bin_count);
    unsigned int *vstart = (unsigned int *)(ws + L.vstart);
    uint2 *run = (uint2 *)(ws + L.run);
    DeviceStats *stats = (DeviceStats *)(ws + L.stats);
    if (prof) {
        if (c->prof_stages != kStagesAdditive || c->last_stream != st) c->prof_frames = 0;   // a session covers one mode and one stream
        c->ev = c->ev_ring[c->prof_frames % kProfRing];
        cudaEventRecord(c->ev[0], st);
    }
    if (ctl.first) cudaMemsetAsync(ws + L.stats, 0, (L.accum - L.stats) + L.accum_bytes, st);      // DeviceStats + the tiles' sums
    if (ctl.first && fp.btile) cudaMemsetAsync(ws + L.planes, 0, L.planes_bytes, st);
    else cudaMemsetAsync(ws + L.stats, 0, offsetof(DeviceStats, f_count), st);                     // the chunk part of DeviceStats
    if (L.ghist) cudaMemsetAsync(counts, 0, L.counts_bytes, st);                    // the blocks count straight into their rows
    SPLOTCH_DISPATCH3(launch_bin_kernels_count, al, L.ghist, fp.btile != 0, L, hbytes, p, n, per, fp, counts, cls_counts, st);
    if (prof) cudaEventRecord(c->ev[1], st);
    const int bps = 1 << (fp.sshift - 5);               // 32-px blocks per super-tile side (k_large's work items)
    k_scan<<<(fp.nbins + 31) / 32, kScanThreads, 0, st>>>(counts, L.nrows, fp.nbins, fp.n_tiles, bin_count, vstart, cls_counts, 2ull * L.capacity,
                                                          c->n_sm, (unsigned int *)(ws + L.large_off), (unsigned int)kLargeChunk,
                                                          (unsigned int)(bps * bps), fp.n_super, stats);
    k_layout<<<kMaxSlabs, kLayoutThreads, 0, st>>>(counts, bin_count, L.nrows, fp.nbins, fp.n_tiles, run, stats);
    if (prof) cudaEventRecord(c->ev[2], st);
    float4 *records = (float4 *)(ws + L.records);
    unsigned int *cursors = (unsigned int *)(ws + L.cursors);
    SPLOTCH_DISPATCH3(launch_bin_kernels_scatter, al, L.ghist, fp.btile != 0, L, hbytes, p, n, per, fp, counts, cursors, run, stats, records, st);
    if (prof) cudaEventRecord(c->ev[3], st);
    if (ctl.chunked) {        // the tiles' sums follow the fixed-point unit of the largest amplitude so far
        k_rescale<<<4 * c->n_sm, 256, 0, st>>>((long long *)(ws + L.accum), L.accum_bytes / sizeof(long long), stats);
        k_rescale_done<<<1, 1, 0, st>>>(stats);
    }
    int rc;
    if (fp.T == 8) rc = launch_render_tail<8>(c, L, ws, fp, image, st, prof, ctl.last);
    else if (fp.T == 16) rc = launch_render_tail<16>(c, L, ws, fp, image, st, prof, ctl.last);
    else if (fp.T == 32) rc = launch_render_tail<32>(c, L, ws, fp, image, st, prof, ctl.last);
    else rc = launch_render_tail<64>(c, L, ws, fp, image, st, prof, ctl.last);
    if (rc != SPLOTCH_OK) return rc;
    CU_TRY(c, cudaGetLastError());
    c->have_frame = true; c->ws = ws; c->lay = L; c->fp = fp; c->last_n = n; c->last_stream = st; c->last_additive = true;
    if (prof) { ++c->prof_frames; c->prof_stages = kStagesAdditive; }
    return SPLOTCH_OK;
}

template <int T>
void launch_ordered_tail(splotch_ctx *c, const Layout &L, char *ws, const FrameParams &fp, const unsigned int *vals0,
                         const unsigned int *vals1, float *image, cudaStream_t st)
{
    const int ti = T == 8 ? 0 : T == 16 ? 1 : 2;
    DeviceStats *stats = (DeviceStats *)(ws + L.stats);
    const unsigned int *tile_start = (const unsigned int *)(ws + L.tile_start);
    k_orender<T><<<c->n_sm * c->orender_blocks_per_sm[ti], kORThreads, sizeof(ORenderSmem<T>), st>>>(
        (const float4 *)(ws + L.rec), vals0, vals1, tile_start, stats, (float4 *)(ws + L.seg), fp);
    if (c->profiling) cudaEventRecord(c->ev[6], st);
    k_ocombine<T><<<fp.n_tiles * (T * T / kCombinePix), kCombinePix * kCombineSlices, 0, st>>>((const float4 *)(ws + L.seg), tile_start, stats, fp, image);
    if (c->profiling) cudaEventRecord(c->ev[7], st);
}

// Ordered (E != A) frame: count -> scan -> pairs -> radix sort -> bounds -> render -> combine, all on `st`.
int render_ordered(splotch_ctx *c, const splotch_particles *p, unsigned long long n, const FrameParams &fp,
                   const Layout &L, float *image, char *ws, cudaStream_t st)
{
    const bool al = aligned16(p);
    DeviceStats *stats = (DeviceStats *)(ws + L.stats);
    unsigned int *blk = (unsigned int *)(ws + L.blk_pairs);
    unsigned int *hist = (unsigned int *)(ws + L.hist), *sums = (unsigned int *)(ws + L.sums);
    unsigned long long *keys[2] = {(unsigned long long *)(ws + L.keys[0]), (unsigned long long *)(ws + L.keys[1])};
    unsigned int *vals[2] = {(unsigned int *)(ws + L.vals[0]), (unsigned int *)(ws + L.vals[1])};
    if (c->profiling) {
        if (c->prof_stages != kStagesOrdered || c->last_stream != st) c->prof_frames = 0;    // a session covers one mode and one stream
        c->ev = c->ev_ring[c->prof_frames % kProfRing];
        cudaEventRecord(c->ev[0], st);
    }
    cudaMemsetAsync(stats, 0, sizeof(DeviceStats), st);
    if (L.nblk_o > 0) {
        if (al) k_ocount<true><<<L.nblk_o, kOThreads, 0, st>>>(p->x, p->y, p->z, p->h, n, fp, blk, stats);
        else    k_ocount<false><<<L.nblk_o, kOThreads, 0, st>>>(p->x, p->y, p->z, p->h, n, fp, blk, stats);
    }
    if (c->profiling) cudaEventRecord(c->ev[1], st);
    k_oscan<<<1, kOScanThreads, 0, st>>>(blk, L.nblk_o, n, L.capacity, c->n_sm, fp.n_tiles, stats);
    if (c->profiling) cudaEventRecord(c->ev[2], st);
    if (L.nblk_o > 0) {
        const size_t lsm = sizeof(float4) * kLutSmemMax;
        if (al) k_opairs<true><<<L.nblk_o, kOThreads, lsm, st>>>(p->x, p->y, p->z, p->h, p->I, p->scalar, n, fp, blk, stats,
                                                                 (float4 *)(ws + L.rec), keys[0], vals[0]);
        else    k_opairs<false><<<L.nblk_o, kOThreads, lsm, st>>>(p->x, p->y, p->z, p->h, p->I, p->scalar, n, fp, blk, stats,
                                                                  (float4 *)(ws + L.rec), keys[0], vals[0]);
    }
    if (c->profiling) cudaEventRecord(c->ev[3], st);
    // radix passes: as many as the widest possible key needs (32 depth bits + the tile bits); the passes beyond the
    // bits this frame's keys really use return at once (the key layout is decided on the device, by k_oscan)
    int tile_bytes = 1;
    while (tile_bytes < 4 && (fp.n_tiles - 1) >> (8 * tile_bytes)) ++tile_bytes;
    int cur = 0;
    for (int pass = 0; pass < 4 + tile_bytes; ++pass) {
        const int shift = 8 * pass;
        k_rs_count<<<L.nblk_rs, kRsThreads, 0, st>>>(keys[cur], stats, shift, L.nblk_rs, hist);
        k_sc_reduce<<<L.n_sums, kScThreads, 0, st>>>(hist, L.m_hist, sums, stats, shift);
        k_sc_top<<<1, 1024, 0, st>>>(sums, L.n_sums, stats, shift);
        k_sc_apply<<<L.n_sums, kScThreads, 0, st>>>(hist, L.m_hist, sums, stats, shift);
        k_rs_scatter<<<L.nblk_rs, kRsThreads, sizeof(RsSmem), st>>>(keys[cur], vals[cur], keys[cur ^ 1], vals[cur ^ 1], stats, shift,
                                                                     L.nblk_rs, hist);
        cur ^= 1;
    }
    if (c->profiling) cudaEventRecord(c->ev[4], st);
    {
        const unsigned long long work = L.capacity > (unsigned long long)fp.n_tiles + 1 ? L.capacity : (unsigned long long)fp.n_tiles + 1;
        k_obounds<<<(unsigned int)(((work + 3) / 4 + 255) / 256), 256, 0, st>>>(keys[0], keys[1], stats, fp.n_tiles, (unsigned int *)(ws + L.tile_start));
    }
    if (c->profiling) cudaEventRecord(c->ev[5], st);
    if (fp.T == 8) launch_ordered_tail<8>(c, L, ws, fp, vals[0], vals[1], image, st);
    else if (fp.T == 16) launch_ordered_tail<16>(c, L, ws, fp, vals[0], vals[1], image, st);
    else launch_ordered_tail<32>(c, L, ws, fp, vals[0], vals[1], image, st);
    CU_TRY(c, cudaGetLastError());
    c->have_frame = true; c->ws = ws; c->lay = L; c->fp = fp; c->last_n = n; c->last_stream = st; c->last_additive = false;
    if (c->profiling) { ++c->prof_frames; c->prof_stages = kStagesOrdered; }
    return SPLOTCH_OK;
}

// Layout of a frame from the caller's workspace; ENOMEM message on failure.
int frame_layout(splotch_ctx *c, unsigned long long n, const splotch_params *q, size_t bytes, bool staging, Layout *L)
{
    const bool ok = q->additive ? make_layout(c, n, q->tile, 0, bytes, staging, L)
                                : fit_layout_ordered(c, n, q->tile, bytes, staging, L);
    if (!ok) return fail(c, SPLOTCH_ENOMEM, "workspace of %zu bytes is below the fixed minimum%s; ask splotch_workspace_bytes",
                         bytes, staging ? " (with host staging)" : "");
    return SPLOTCH_OK;
}

}  // namespace

extern "C" {

const char *splotch_version(void) { return "splotch-b200 0.1 (sm_100a)"; }

const char *splotch_stage_name(int additive, int s)
{
    if (additive) return (s >= 0 && s < kStagesAdditive) ? kStageNamesAdditive[s] : "";
    return (s >= 0 && s < kStagesOrdered) ? kStageNamesOrdered[s] : "";
}

const char *splotch_last_error(const splotch_ctx *c) { return c ? c->err : g_create_err; }

int splotch_create(splotch_ctx **out, int device, int width, int height, uint64_t max_particles)
{
    if (!out) return SPLOTCH_EINVAL;
    *out = nullptr;
    if (width <= 0 || height <= 0 || width > 32768 || height > 32768 || max_particles > 0xfffffff0ull)
        return fail(nullptr, SPLOTCH_EINVAL, "bad image size or max_particles");
    int ndev = 0;
    CU_TRY(nullptr, cudaGetDeviceCount(&ndev));
    if (device < 0 || device >= ndev) return fail(nullptr, SPLOTCH_ECUDA, "no CUDA device %d (%d visible)", device, ndev);
    cudaDeviceProp prop;
    CU_TRY(nullptr, cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10) return fail(nullptr, SPLOTCH_EDEVICE, "device %d is sm_%d%d, need sm_100", device, prop.major, prop.minor);
    CU_TRY(nullptr, cudaSetDevice(device));
    splotch_ctx *c = new (std::nothrow) splotch_ctx();
    if (!c) return fail(nullptr, SPLOTCH_ENOMEM, "host allocation failed");
    c->device = device; c->width = width; c->height = height; c->max_particles = max_particles;
    c->n_sm = prop.multiProcessorCount;
    c->smem_optin = (int)prop.sharedMemPerBlockOptin;
    const int hb = c->smem_optin - 1024;      // dynamic shared memory the binning kernels may ask for
    int rc = [&]() -> int {
        CU_TRY(c, cudaMalloc(&c->lut, sizeof(float4) * kMaxSpecies * kMaxLut));
        CU_TRY(c, cudaMemset(c->lut, 0, sizeof(float4) * kMaxSpecies * kMaxLut));
        { const int rs = static_scratch_address(c, device, &c->static_scratch); if (rs != SPLOTCH_OK) return rs; }   // `device` is current
        CU_TRY(c, (cudaFuncSetAttribute(k_count<true, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, hb)));
        CU_TRY(c, (cudaFuncSetAttribute(k_count<false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, hb)));
        CU_TRY(c, (cudaFuncSetAttribute(k_scatter<true, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, hb)));
        CU_TRY(c, (cudaFuncSetAttribute(k_scatter<false, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, hb)));
        CU_TRY(c, (cudaFuncSetAttribute(k_count<true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, hb)));
        CU_TRY(c, (cudaFuncSetAttribute(k_count<false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, hb)));
        CU_TRY(c, (cudaFuncSetAttribute(k_scatter<true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, hb)));
        CU_TRY(c, (cudaFuncSetAttribute(k_scatter<false, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, hb)));
        int r = query_splat_occupancy<8>(c, &c->splat_blocks_per_sm[0]);
        if (r == SPLOTCH_OK) r = query_splat_occupancy<16>(c, &c->splat_blocks_per_sm[1]);
        if (r == SPLOTCH_OK) r = query_splat_occupancy<32>(c, &c->splat_blocks_per_sm[2]);
        if (r == SPLOTCH_OK) r = query_splat_occupancy<64>(c, &c->splat_blocks_per_sm[3]);
        if (r != SPLOTCH_OK) return r;
        CU_TRY(c, cudaFuncSetAttribute(k_rs_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(RsSmem)));
        CU_TRY(c, cudaFuncSetAttribute(k_orender<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ORenderSmem<8>)));
        CU_TRY(c, cudaFuncSetAttribute(k_orender<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ORenderSmem<16>)));
        CU_TRY(c, cudaFuncSetAttribute(k_orender<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ORenderSmem<32>)));
        CU_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->orender_blocks_per_sm[0], k_orender<8>, kORThreads, sizeof(ORenderSmem<8>)));
        CU_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->orender_blocks_per_sm[1], k_orender<16>, kORThreads, sizeof(ORenderSmem<16>)));
        CU_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c->orender_blocks_per_sm[2], k_orender<32>, kORThreads, sizeof(ORenderSmem<32>)));
        for (int k = 0; k < 3; ++k) if (c->orender_blocks_per_sm[k] < 1) c->orender_blocks_per_sm[k] = 1;
        {   // k_large allocates tensor memory, which the occupancy calculator answers with one block per SM: count registers,
            // shared memory and tensor-memory columns here
            cudaFuncAttributes fa;
            cudaDeviceProp prop;
            CU_TRY(c, cudaFuncSetAttribute(k_large, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(LargeSmem)));
            CU_TRY(c, cudaFuncGetAttributes(&fa, k_large));
            CU_TRY(c, cudaGetDeviceProperties(&prop, c->device));
            const int regs_per_block = ((fa.numRegs + 7) / 8 * 8) * kLargeThreads;
            const int by_regs = prop.regsPerMultiprocessor / (regs_per_block > 0 ? regs_per_block : 1);
            const int by_smem = (int)(prop.sharedMemPerMultiprocessor / (fa.sharedSizeBytes + sizeof(LargeSmem) + 1024));
            const int by_tmem = 512 / (int)kLargeTmemCols;
            int b = by_regs < by_smem ? by_regs : by_smem;
            if (by_tmem < b) b = by_tmem;
            c->large_blocks_per_sm = b < 1 ? 1 : b;
        }
        return r;
    }();
    if (rc != SPLOTCH_OK) {
        snprintf(g_create_err, sizeof g_create_err, "%s", c->err);
        splotch_destroy(c);
        return rc;
    }
    *out = c;
    return SPLOTCH_OK;
}

int splotch_destroy(splotch_ctx *c)
{
    if (!c) return SPLOTCH_EINVAL;
    cudaSetDevice(c->device);
    if (c->lut) cudaFree(c->lut);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    for (int k = 0; k < 2; ++k) { if (c->ev_copied[k]) cudaEventDestroy(c->ev_copied[k]); if (c->ev_consumed[k]) cudaEventDestroy(c->ev_consumed[k]); }
    if (c->ev_start) cudaEventDestroy(c->ev_start);
    if (c->ev_ring) {
        for (int f = 0; f < kProfRing; ++f)
            for (int i = 0; i <= kStages; ++i)
                if (c->ev_ring[f][i]) cudaEventDestroy(c->ev_ring[f][i]);
        delete[] c->ev_ring;
    }
    delete c;
    return SPLOTCH_OK;
}

// Camera constants: double arithmetic on the float inputs, one rounding to float32 (C1 "host constants").
int splotch_set_camera(splotch_ctx *c, const float eye[3], const float lookat[3], const float up[3], float fov_deg)
{
    if (!c) return SPLOTCH_EINVAL;
    if (!eye || !lookat || !up) return fail(c, SPLOTCH_EINVAL, "null camera vector");
    if (!(fov_deg > 0.0f) || !(fov_deg < 180.0f)) return fail(c, SPLOTCH_EINVAL, "fov must be in (0, 180) degrees");
    double fwd[3], rgt[3], upp[3];
    for (int k = 0; k < 3; ++k) fwd[k] = (double)lookat[k] - (double)eye[k];
    const double nf = sqrt(fwd[0] * fwd[0] + fwd[1] * fwd[1] + fwd[2] * fwd[2]);
    if (!(nf > 0.0)) return fail(c, SPLOTCH_EINVAL, "eye == lookat");
    for (int k = 0; k < 3; ++k) fwd[k] /= nf;
    rgt[0] = fwd[1] * (double)up[2] - fwd[2] * (double)up[1];
    rgt[1] = fwd[2] * (double)up[0] - fwd[0] * (double)up[2];
    rgt[2] = fwd[0] * (double)up[1] - fwd[1] * (double)up[0];
    const double nr = sqrt(rgt[0] * rgt[0] + rgt[1] * rgt[1] + rgt[2] * rgt[2]);
    if (!(nr > 0.0)) return fail(c, SPLOTCH_EINVAL, "up is parallel to the view direction");
    for (int k = 0; k < 3; ++k) rgt[k] /= nr;
    upp[0] = rgt[1] * fwd[2] - rgt[2] * fwd[1];
    upp[1] = rgt[2] * fwd[0] - rgt[0] * fwd[2];
    upp[2] = rgt[0] * fwd[1] - rgt[1] * fwd[0];
    for (int k = 0; k < 3; ++k) {
        c->cam[k] = (float)rgt[k]; c->cam[3 + k] = (float)upp[k]; c->cam[6 + k] = (float)fwd[k]; c->cam[9 + k] = eye[k];
    }
    const double half = 0.5 * ((double)fov_deg * (3.14159265358979323846 / 180.0));
    c->cam[12] = (float)(0.5 * (double)c->width / tan(half));
    c->cam[13] = (float)(0.5 * (double)c->width);
    c->cam[14] = (float)(0.5 * (double)c->height);
    c->cam[15] = 0.0f;
    c->camera_set = true;
    return SPLOTCH_OK;
}

int splotch_get_camera_constants(const splotch_ctx *c, float out[16])
{
    if (!c || !out) return SPLOTCH_EINVAL;
    if (!c->camera_set) return SPLOTCH_ESTATE;
    memcpy(out, c->cam, sizeof c->cam);
    return SPLOTCH_OK;
}

int splotch_set_colormap(splotch_ctx *c, int species, const float *rgb, int n_entries)
{
    if (!c) return SPLOTCH_EINVAL;
    if (species < 0 || species >= kMaxSpecies || !rgb || n_entries < 2 || n_entries > kMaxLut)
        return fail(c, SPLOTCH_EINVAL, "bad colour map (species 0..%d, 2..%d entries)", kMaxSpecies - 1, kMaxLut);
    float4 *tmp = new (std::nothrow) float4[n_entries];
    if (!tmp) return fail(c, SPLOTCH_ENOMEM, "host allocation failed");
    for (int i = 0; i < n_entries; ++i) tmp[i] = make_float4(rgb[3 * i], rgb[3 * i + 1], rgb[3 * i + 2], 0.0f);
    cudaSetDevice(c->device);
    const cudaError_t e = cudaMemcpy(c->lut + species * kMaxLut, tmp, sizeof(float4) * n_entries, cudaMemcpyHostToDevice);
    delete[] tmp;
    if (e != cudaSuccess) return fail(c, SPLOTCH_ECUDA, "colour map upload failed: %s", cudaGetErrorString(e));
    c->lut_n[species] = n_entries;
    return SPLOTCH_OK;
}

int splotch_set_profiling(splotch_ctx *c, int enabled)
{
    if (!c) return SPLOTCH_EINVAL;
    if (enabled && !c->ev_ring) {
        CU_TRY(c, cudaSetDevice(c->device));
        c->ev_ring = new (std::nothrow) cudaEvent_t[kProfRing][kStages + 1]();
        if (!c->ev_ring) return fail(c, SPLOTCH_ENOMEM, "host allocation failed");
        for (int f = 0; f < kProfRing; ++f)
            for (int i = 0; i <= kStages; ++i) CU_TRY(c, cudaEventCreate(&c->ev_ring[f][i]));
    }
    c->profiling = enabled != 0;
    c->prof_frames = 0;
    return SPLOTCH_OK;
}

size_t splotch_workspace_bytes(const splotch_ctx *c, uint64_t n, int tile, uint64_t pair_capacity, int with_host_staging)
{
    if (!c || tile_shift(tile) < 0 || n > c->max_particles) return 0;
    if (pair_capacity == 0) pair_capacity = 2ull * n + (1ull << 20);
    if (pair_capacity > 0x7ff00000ull) return 0;
    Layout L, Lo;
    make_layout(c, n, tile, pair_capacity, 0, with_host_staging != 0, &L);
    make_layout_ordered(c, n, tile, pair_capacity, with_host_staging != 0, &Lo);       // either mode must fit
    // the same 8192-byte reserve on both sides: splotch_render derives its capacity as (bytes - fixed - 8192) / 32
    return (L.total > Lo.total ? L.total : Lo.total) + 8192 + 4096;
}

int splotch_render(splotch_ctx *c, const splotch_particles *p, uint64_t n, const splotch_params *q, float *image_out,
                   void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!c) return SPLOTCH_EINVAL;
    FrameParams fp;
    int rc = check_params(c, p, n, q, &fp);
    if (rc != SPLOTCH_OK) return rc;
    if (!image_out || !workspace) return fail(c, SPLOTCH_EINVAL, "null image or workspace");
    if (((uintptr_t)workspace & 255u) != 0) return fail(c, SPLOTCH_EINVAL, "workspace must be 256-byte aligned");
    Layout L;
    rc = frame_layout(c, n, q, workspace_bytes, false, &L);
    if (rc != SPLOTCH_OK) return rc;
    CU_TRY(c, cudaSetDevice(c->device));
    fp.dev_range = (const float2 *)((RangeRaw *)((char *)workspace + L.ranges) + kMaxSpecies);
    fp.btile_planes = (float *)((char *)workspace + L.planes);
    if (fp.any_auto) range_pass(c, p, n, fp, (char *)workspace, L, (cudaStream_t)cuda_stream, true, true);
    if (!q->additive) return render_ordered(c, p, n, fp, L, image_out, (char *)workspace, (cudaStream_t)cuda_stream);
    return render_device(c, p, n, fp, L, image_out, (char *)workspace, (cudaStream_t)cuda_stream);
}

int splotch_set_host_chunk(splotch_ctx *c, uint64_t particles_per_chunk)
{
    if (!c) return SPLOTCH_EINVAL;
    c->host_chunk = particles_per_chunk;
    return SPLOTCH_OK;
}

// The paper's per-chunk offload loop (Fig. 3; Eq. 3-4 :111-120) with the copy / compute overlap it names
// as future work (:354): the particle set streams through two staging buffers, the host-to-device copy of chunk k + 1 runs
// on the context's copy stream while chunk k is counted, binned and splatted on the caller's stream; the chunks' partial
// images accumulate in the tiles' fixed-point sums (exact, order independent), one k_compose and one copy back at the end.
// The ordered mode needs the whole set for its depth sort: one copy in, one frame, one copy out.
int splotch_render_host(splotch_ctx *c, const splotch_particles *hp, uint64_t n, const splotch_params *q,
                        float *host_image_out, void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!c) return SPLOTCH_EINVAL;
    FrameParams fp;
    int rc = check_params(c, hp, n, q, &fp);
    if (rc != SPLOTCH_OK) return rc;
    if (!host_image_out || !workspace) return fail(c, SPLOTCH_EINVAL, "null image or workspace");
    if (((uintptr_t)workspace & 255u) != 0) return fail(c, SPLOTCH_EINVAL, "workspace must be 256-byte aligned");
    Layout L;
    rc = frame_layout(c, n, q, workspace_bytes, true, &L);
    if (rc != SPLOTCH_OK) return rc;
    CU_TRY(c, cudaSetDevice(c->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char *ws = (char *)workspace;
    const int nf = fp.any_vector ? kHostFields : 6;
    const float *src[kHostFields] = {hp->x, hp->y, hp->z, hp->h, hp->I, hp->scalar, hp->cr, hp->cg, hp->cb};
    const size_t image_bytes = sizeof(float) * 3 * (size_t)c->width * c->height;
    fp.dev_range = (const float2 *)((RangeRaw *)(ws + L.ranges) + kMaxSpecies);
    fp.btile_planes = (float *)(ws + L.planes);
    auto device_view = [&](float *const *dst) {
        splotch_particles dp = *hp;
        dp.x = dst[0]; dp.y = dst[1]; dp.z = dst[2]; dp.h = dst[3]; dp.I = dst[4]; dp.scalar = dst[5];
        dp.cr = dst[6]; dp.cg = dst[7]; dp.cb = dst[8];
        return dp;
    };
    if (!q->additive) {
        const size_t fstride = align_up(sizeof(float) * n, 256);
        float *dst[kHostFields];
        for (int k = 0; k < kHostFields; ++k) {
            dst[k] = (float *)(ws + L.staging + k * fstride);
            if (n && k < nf) CU_TRY(c, cudaMemcpyAsync(dst[k], src[k], sizeof(float) * n, cudaMemcpyHostToDevice, st));
        }
        float *dimg = (float *)(ws + L.staging + align_up(kHostFields * fstride, 256));
        const splotch_particles dp = device_view(dst);
        fp.vec[0] = dp.cr; fp.vec[1] = dp.cg; fp.vec[2] = dp.cb;
        if (fp.any_auto) range_pass(c, &dp, n, fp, ws, L, st, true, true);
        rc = render_ordered(c, &dp, n, fp, L, dimg, ws, st);
        if (rc != SPLOTCH_OK) return rc;
        CU_TRY(c, cudaMemcpyAsync(host_image_out, dimg, image_bytes, cudaMemcpyDeviceToHost, st));
        CU_TRY(c, cudaStreamSynchronize(st));
        return SPLOTCH_OK;
    }
    // ---- additive: chunks on two streams
    if (!c->copy_stream) {
        CU_TRY(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        for (int k = 0; k < 2; ++k) {
            CU_TRY(c, cudaEventCreateWithFlags(&c->ev_copied[k], cudaEventDisableTiming));
            CU_TRY(c, cudaEventCreateWithFlags(&c->ev_consumed[k], cudaEventDisableTiming));
        }
        CU_TRY(c, cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming));
    }
    const unsigned long long ch = host_chunk_particles(c, n);
    const size_t fstride = align_up(sizeof(float) * ch, 256);
    float *dimg = (float *)(ws + L.staging + align_up(2 * kHostFields * fstride, 256));
    const unsigned long long nchunks = n ? (n + ch - 1) / ch : 1;
    const int ns = fp.n_species;
    unsigned long long sp_begin[kMaxSpecies + 1];
    for (int s = 0; s <= ns; ++s) sp_begin[s] = hp->species_offsets ? hp->species_offsets[s] : (s == 0 ? 0ull : n);
    auto chunk_params = [&](unsigned long long lo, unsigned long long len, float *const *dst) {
        FrameParams fc = fp;                                      // the chunk's own species ranges and field pointers
        for (int s = 0; s <= ns; ++s) {
            const unsigned long long o = sp_begin[s] < lo ? 0ull : (sp_begin[s] - lo < len ? sp_begin[s] - lo : len);
            fc.sp_begin[s] = (unsigned int)o;
        }
        fc.vec[0] = dst[6]; fc.vec[1] = dst[7]; fc.vec[2] = dst[8];
        return fc;
    };
    if (fp.any_auto) {
        // the ranges need the whole set before the first chunk is coloured: one more pass over the colour quantities
        // (scalar, or the vector components), through staging buffer 0 on the caller's stream
        for (unsigned long long k = 0; k < nchunks; ++k) {
            const unsigned long long lo = k * ch, len = n ? (lo + ch < n ? ch : n - lo) : 0;
            float *dst[kHostFields];
            for (int f = 0; f < kHostFields; ++f) {
                dst[f] = (float *)(ws + L.staging + (size_t)f * fstride);
                if (len && f >= 5 && f < nf) CU_TRY(c, cudaMemcpyAsync(dst[f], src[f] + lo, sizeof(float) * len, cudaMemcpyHostToDevice, st));
            }
            const splotch_particles dp = device_view(dst);
            const FrameParams fc = chunk_params(lo, len, dst);
            range_pass(c, &dp, len, fc, ws, L, st, k == 0, k + 1 == nchunks);
        }
    }
    CU_TRY(c, cudaEventRecord(c->ev_start, st));                 // the staging buffers are free once earlier work on `st` is done
    CU_TRY(c, cudaStreamWaitEvent(c->copy_stream, c->ev_start, 0));
    // The chunks ramp up (an eighth, a quarter, half a chunk, then whole chunks): the kernels cannot start before the first chunk has
    // arrived, and a chunk's kernels take longer than the next chunk's copy as long as that one is not more than about 1.5 times larger
    unsigned long long lo_next = 0, k = 0;
    for (; k == 0 || lo_next < n; ++k) {
        unsigned long long want = ch;
        if (n > ch && k < 3) { want = (ch >> (3 - k)); want = want < (1ull << 20) ? (1ull << 20) : want; want = (want + 3) / 4 * 4; if (want > ch) want = ch; }
        const unsigned long long lo = lo_next, len = n ? (lo + want < n ? want : n - lo) : 0;
        lo_next = lo + len;
        const bool last = lo_next >= n;
        const int b = (int)(k & 1);
        float *dst[kHostFields];
        if (k >= 2) CU_TRY(c, cudaStreamWaitEvent(c->copy_stream, c->ev_consumed[b], 0));
        for (int f = 0; f < kHostFields; ++f) {
            dst[f] = (float *)(ws + L.staging + (size_t)(kHostFields * b + f) * fstride);
            if (len && f < nf) CU_TRY(c, cudaMemcpyAsync(dst[f], src[f] + lo, sizeof(float) * len, cudaMemcpyHostToDevice, c->copy_stream));
        }
        CU_TRY(c, cudaEventRecord(c->ev_copied[b], c->copy_stream));
        CU_TRY(c, cudaStreamWaitEvent(st, c->ev_copied[b], 0));
        const splotch_particles dp = device_view(dst);
        const FrameParams fc = chunk_params(lo, len, dst);
        rc = render_device(c, &dp, len, fc, L, dimg, ws, st, ChunkCtl{k == 0, last, nchunks > 1});
        if (rc != SPLOTCH_OK) return rc;
        CU_TRY(c, cudaEventRecord(c->ev_consumed[b], st));
    }
    c->last_n = n;
    CU_TRY(c, cudaMemcpyAsync(host_image_out, dimg, image_bytes, cudaMemcpyDeviceToHost, st));
    CU_TRY(c, cudaStreamSynchronize(st));
    return SPLOTCH_OK;
}

int splotch_get_stats(splotch_ctx *c, splotch_stats *out)
{
    if (!c || !out) return SPLOTCH_EINVAL;
    if (!c->have_frame) return fail(c, SPLOTCH_ESTATE, "no frame rendered yet");
    CU_TRY(c, cudaSetDevice(c->device));
    CU_TRY(c, cudaStreamSynchronize(c->last_stream));
    DeviceStats ds;
    CU_TRY(c, cudaMemcpy(&ds, c->ws + c->lay.stats, sizeof ds, cudaMemcpyDeviceToHost));
    memset(out, 0, sizeof *out);
    out->n = c->last_n;
    if (c->last_additive) {       // totals of the frame (a chunked host frame sums its chunks)
        for (int k = 0; k < 4; ++k) out->count[k] = ds.f_count[k];
        out->pairs = ds.f_pairs; out->large_pairs = ds.f_large_pairs; out->chunks = ds.f_chunks;
        out->overflow = (int32_t)ds.f_overflow;
    } else {
        for (int k = 0; k < 4; ++k) out->count[k] = ds.count[k];
        out->pairs = ds.pairs; out->large_pairs = ds.large_pairs; out->chunks = ds.chunks;
        out->overflow = (int32_t)ds.overflow;
    }
    out->pair_capacity = ds.capacity;
    out->sort_key_bits = c->last_additive ? 0 : (int32_t)ds.key_bits;
    if (c->profiling && c->prof_frames > 0) {
        // mean per frame over the frames recorded since profiling was enabled (at most the last kProfRing)
        const unsigned long long nf = c->prof_frames < kProfRing ? c->prof_frames : kProfRing;
        out->n_stages = c->prof_stages;
        for (int s = 0; s < c->prof_stages; ++s) {
            double sum = 0.0;
            for (unsigned long long f = 0; f < nf; ++f) {
                float ms = 0.0f;
                CU_TRY(c, cudaEventElapsedTime(&ms, c->ev_ring[f][s], c->ev_ring[f][s + 1]));
                sum += ms;
            }
            out->stage_ms[s] = (float)(sum / (double)nf);
        }
    }
    return SPLOTCH_OK;
}

int splotch_apply_transfer(splotch_ctx *c, float *image, void *cuda_stream)
{
    if (!c || !image) return SPLOTCH_EINVAL;
    CU_TRY(c, cudaSetDevice(c->device));
    k_apply_transfer<<<4 * c->n_sm, 256, 0, (cudaStream_t)cuda_stream>>>(image, 3 * (size_t)c->width * c->height);
    CU_TRY(c, cudaGetLastError());
    return SPLOTCH_OK;
}

int splotch_compose_shards(splotch_ctx *c, const void *const *workspaces, int n_shards, int tile, int tile_begin, int tile_end,
                           int apply_transfer, float *image_out, void *cuda_stream)
{
    if (!c || !workspaces || !image_out) return SPLOTCH_EINVAL;
    if (n_shards < 1 || n_shards > kMaxShards) return fail(c, SPLOTCH_EINVAL, "n_shards must be 1..%d", kMaxShards);
    const int ts = tile_shift(tile);
    if (ts < 0) return fail(c, SPLOTCH_EINVAL, "tile must be 8, 16, 32 or 64 (got %d)", tile);
    // the offsets of the sums and of the statistics inside a workspace depend on the image size, the tile side and the SM count only
    Layout L;
    if (!make_layout(c, 0, tile, 1, 0, false, &L)) return fail(c, SPLOTCH_EINVAL, "no layout for this image and tile");
    FrameParams fp;
    memset(&fp, 0, sizeof fp);
    fp.W = c->width; fp.H = c->height; fp.T = tile; fp.tshift = ts;
    fp.ntx = (c->width + tile - 1) / tile; fp.nty = (c->height + tile - 1) / tile; fp.n_tiles = fp.ntx * fp.nty;
    if (tile_end < 0) tile_end = fp.n_tiles;
    if (tile_begin < 0 || tile_begin > tile_end || tile_end > fp.n_tiles) return fail(c, SPLOTCH_EINVAL, "bad tile range [%d, %d) of %d", tile_begin, tile_end, fp.n_tiles);
    ShardPtrs sh;
    memset(&sh, 0, sizeof sh);
    sh.n = n_shards;
    for (int k = 0; k < n_shards; ++k) {
        if (!workspaces[k] || ((uintptr_t)workspaces[k] & 255u)) return fail(c, SPLOTCH_EINVAL, "workspace %d is null or not 256-byte aligned", k);
        sh.accum[k] = (const unsigned long long *)((const char *)workspaces[k] + L.accum);
        sh.stats[k] = (const DeviceStats *)((const char *)workspaces[k] + L.stats);
    }
    if (tile_end == tile_begin) return SPLOTCH_OK;
    CU_TRY(c, cudaSetDevice(c->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int grid = tile_end - tile_begin;
    if (tile == 8) k_compose_shards<8><<<grid, 256, 0, st>>>(sh, fp, tile_begin, apply_transfer, image_out);
    else if (tile == 16) k_compose_shards<16><<<grid, 256, 0, st>>>(sh, fp, tile_begin, apply_transfer, image_out);
    else if (tile == 32) k_compose_shards<32><<<grid, 256, 0, st>>>(sh, fp, tile_begin, apply_transfer, image_out);
    else k_compose_shards<64><<<grid, 256, 0, st>>>(sh, fp, tile_begin, apply_transfer, image_out);
    CU_TRY(c, cudaGetLastError());
    return SPLOTCH_OK;
}

int splotch_measure_peaks(splotch_ctx *c, double out[2], void *cuda_stream)
{
    if (!c || !out) return SPLOTCH_EINVAL;
    CU_TRY(c, cudaSetDevice(c->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int grid = 2 * c->n_sm;
    float *buf = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    CU_TRY(c, cudaMalloc(&buf, sizeof(float) * (size_t)grid * kPeakThreads));
    int rc = [&]() -> int {
        CU_TRY(c, cudaEventCreate(&e0));
        CU_TRY(c, cudaEventCreate(&e1));
        const double ops = (double)grid * kPeakThreads * kPeakIters * kPeakChains;
        for (int op = 0; op < 2; ++op) {
            float best = 0.0f;
            for (int rep = 0; rep < 4; ++rep) {           // the first launch warms up; keep the best of the rest
                CU_TRY(c, cudaEventRecord(e0, st));
                if (op == 0) k_peak<0><<<grid, kPeakThreads, 0, st>>>(buf, 0.3f);
                else         k_peak<1><<<grid, kPeakThreads, 0, st>>>(buf, 0.3f);
                CU_TRY(c, cudaEventRecord(e1, st));
                CU_TRY(c, cudaEventSynchronize(e1));
                float ms = 0.0f;
                CU_TRY(c, cudaEventElapsedTime(&ms, e0, e1));
                if (rep > 0 && (best == 0.0f || ms < best)) best = ms;
            }
            out[op] = ops / ((double)best * 1e-3);
        }
        return SPLOTCH_OK;
    }();
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf);
    return rc;
}

int splotch_debug_geometry(splotch_ctx *c, const splotch_particles *p, uint64_t n, const splotch_params *q, int8_t *cls,
                           float *px, float *py, float *sp, float *rp, float *zc, int32_t *pbox, int32_t *tbox,
                           int32_t *ilabel, void *cuda_stream)
{
    if (!c) return SPLOTCH_EINVAL;
    FrameParams fp;
    const int rc = check_params(c, p, n, q, &fp);
    if (rc != SPLOTCH_OK) return rc;
    if (n == 0) return SPLOTCH_OK;
    CU_TRY(c, cudaSetDevice(c->device));
    k_debug_geometry<<<(unsigned int)((n + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(
        p->x, p->y, p->z, p->h, n, fp, cls, px, py, sp, rp, zc, (int4 *)pbox, (int4 *)tbox, ilabel);
    CU_TRY(c, cudaGetLastError());
    return SPLOTCH_OK;
}

int splotch_debug_tile_counts(splotch_ctx *c, uint32_t *out, void *cuda_stream)
{
    if (!c || !out) return SPLOTCH_EINVAL;
    if (!c->have_frame) return fail(c, SPLOTCH_ESTATE, "no frame rendered yet");
    CU_TRY(c, cudaSetDevice(c->device));
    if (c->last_additive) {
        k_tile_counts<<<(c->fp.n_tiles + 255) / 256, 256, 0, (cudaStream_t)cuda_stream>>>((const unsigned int *)(c->ws + c->lay.bin_count),
                                                                                            c->fp.n_tiles, c->fp.n_super, c->fp.n_big, out);
        CU_TRY(c, cudaGetLastError());
    } else {
        k_odiff<<<(c->fp.n_tiles + 255) / 256, 256, 0, (cudaStream_t)cuda_stream>>>((const unsigned int *)(c->ws + c->lay.tile_start),
                                                                                     c->fp.n_tiles, out);
        CU_TRY(c, cudaGetLastError());
    }
    return SPLOTCH_OK;
}

// Classes and per-tile pair counts of a particle set (steps A1, A3, A4a) without any allocation and without a workspace.
int splotch_count_static(splotch_ctx *c, const splotch_particles *p, uint64_t n, const splotch_params *q,
                         uint32_t *tile_counts_out, uint64_t *class_counts_out, void *cuda_stream)
{
    if (!c) return SPLOTCH_EINVAL;
    if (!tile_counts_out || !class_counts_out) return fail(c, SPLOTCH_EINVAL, "null output");
    FrameParams fp;
    const int rc = check_params(c, p, n, q, &fp);
    if (rc != SPLOTCH_OK) return rc;
    if (!q->additive || q->renderer != 0) return fail(c, SPLOTCH_EINVAL, "splotch_count_static takes the additive mode and the default renderer");
    if (!c->static_scratch) return fail(c, SPLOTCH_ESTATE, "static scratch was not set up");
    const int nrows = c->n_sm;
    const size_t counts_bytes = sizeof(unsigned int) * (size_t)nrows * fp.nbins;
    const size_t need = align_up(counts_bytes, 256) + sizeof(unsigned int) * 4 * (size_t)nrows;
    if (need > kStaticScratchBytes)
        return fail(c, SPLOTCH_EINVAL, "splotch_count_static: %d bins x %d rows need %zu bytes of scratch, the static array holds %zu "
                                        "(at most %zu bins: use a larger tile or splotch_render with a workspace)",
                    fp.nbins, nrows, need, kStaticScratchBytes, (kStaticScratchBytes - 16 * (size_t)nrows - 256) / (sizeof(unsigned int) * nrows));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU_TRY(c, cudaSetDevice(c->device));
    unsigned int *counts = (unsigned int *)c->static_scratch;
    unsigned int *cls_counts = (unsigned int *)(c->static_scratch + align_up(counts_bytes, 256));
    // the array keeps the last call's contents: the blocks count into their rows with atomics, so the rows start at zero
    CU_TRY(c, cudaMemsetAsync(c->static_scratch, 0, need, st));
    CU_TRY(c, cudaMemsetAsync(class_counts_out, 0, 4 * sizeof(unsigned long long), st));
    unsigned long long per = (n + nrows - 1) / nrows;
    per = (per + 3) / 4 * 4;
    if (per == 0) per = 4;
    if (aligned16(p)) k_count<true, true, false><<<nrows, kBinThreads, 0, st>>>(p->x, p->y, p->z, p->h, n, per, fp, counts, cls_counts);
    else              k_count<false, true, false><<<nrows, kBinThreads, 0, st>>>(p->x, p->y, p->z, p->h, n, per, fp, counts, cls_counts);
    k_static_count_reduce<<<(fp.n_tiles + 255) / 256, 256, 0, st>>>(counts, cls_counts, nrows, fp.nbins, fp.n_tiles, fp.n_super, fp.n_big,
                                                                    tile_counts_out, (unsigned long long *)class_counts_out);
    k_static_count_finish<<<1, 1, 0, st>>>((unsigned long long *)class_counts_out);
    CU_TRY(c, cudaGetLastError());
    return SPLOTCH_OK;
}

}  // extern "C"
