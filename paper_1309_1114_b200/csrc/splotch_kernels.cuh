// splotch_kernels.cuh -- device code of the B200-native Splotch rendering path (sm_100a).
//
// Stage map (paper passages in PAPER.md):
//   k_count    A1+A3+A4a  roto-translate, project, classify (:76, :138, :156-173) and count (particle, bin) pairs
//   k_scan     A4b        per-bin exclusive scan down the rows of the count matrix (replaces thrust::reduce_by_key,
//                         :203); the last block to finish builds the frame statistics, the virtual bin order, the chunk size
//                         and k_large's item table (replaces inclusive_scan, :205)
//   k_layout   A4b        the runs of every bin inside the slabs of the record array
//   k_scatter  A1-A3+A2+A4c  recompute geometry, colourise (:76, :85), write render records in bin order
//                            (replaces copy_if + sort_by_key, :196-202)
//   k_splat    A5         (splotch_splat.cuh) SMALL + MEDIUM records of the tile bins: a producer warp streams the records into
//                         shared memory with bulk copies, consumer warps add SMALL records and tiny boxes straight into the
//                         tile's fixed-point planes and evaluate the others as owners of 8 x 8-pixel strips (the paper's
//                         medium-particle kernel, :183, :224-228, without its halo copies)
//   k_large    A6         (splotch_large.cuh) LARGE particles, which the paper renders on the CPU (:232-238), and with 32-px tiles
//                         the MEDIUM discs wider than 32 px: items of (chunk of a region's records) x (32 x 32-px block); bands
//                         inside their disc are summed on the tensor cores (tcgen05), the others per pixel
//   k_compose  A8         per tile: fixed-point sums -> float32, optional 1-exp(-S), write the image once
//
// Canonical float32 geometry: every operation that decides an integer (class, pixel box, tile box, the inside
// test) is written with round-to-nearest intrinsics (__fmul_rn, __fmaf_rn, __fdiv_rn ...) which nvcc never
// contracts or reorders, so the values equal those of any IEEE-754 binary32 implementation of the same sequence.
// floor / ceil / float->int of the (clamped) box bounds are taken with the 1.5 * 2^23 addition trick: exact for
// arguments in [-1, 32768], and on the FMA / ALU pipes instead of the quarter-rate conversion pipe (FRND, F2I),
// which bounded the first version of every kernel here (profiles/r1_step1_*).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace splotch {

constexpr int kMaxSpecies   = 8;
constexpr int kMaxLut       = 1024;
constexpr int kChunkMax     = 32768;  // 16-byte units per work item of k_splat (upper bound; the frame picks its own)
constexpr int kChunkMin     = 256;
constexpr int kBinThreads   = 1024;   // k_count / k_scatter block size: one CTA per SM (fewer histogram rows and write streams than 2 x 512)
constexpr int kSuperShift   = 3;      // super-tile = 8 x 8 tiles, at most 128 px (LARGE particles are binned to super-tiles)
constexpr int kSuperMaxShift = 7;      // 128 px: k_large tests every record of a super-tile against each of its 32-px blocks (16 instead of 64 at
                                       // 256 px: cfg3 k_large 282 -> 245 ms for 1 ms more in k_count and 1.7 ms more in k_scatter; 64 px: frame 341.5 -> 335.6 ms
                                       // but 410 M LARGE records, several GB more in the workspace: not taken)
constexpr float kRouteRadius = 32.0f;  // 32-px tiles: MEDIUM discs with r(p) above this go to k_large's block renderer instead of k_splat's strips
constexpr int kLutSmemMax   = 1024;   // colour-table entries (all species together) staged in shared memory by k_scatter
constexpr int kFixedBits    = 30;     // the largest record amplitude maps to [2^29, 2^30) fixed-point units

enum { CULLED = 0, SMALL = 1, MEDIUM = 2, LARGE = 3 };

struct SpeciesDev {
    float brightness, absorb;
    float fixed_r, fixed_g, fixed_b;
    float smin, inv_range;                           // t = (v - smin) * inv_range
    float lut_nm1, lut_nm2;                          // (float)(lut_n - 1), (float)(lut_n - 2)
    int   use_colormap, use_log10, lut_n, lut_off;   // lut_off: first entry in the packed shared-memory table
    int   vector, auto_range;                        // colour from the vector fields; range found on the device (:166 fn. 1)
};

struct FrameParams {
    float cam[16];               // r[3] u[3] f[3] eye[3] s cx cy 0
    float chi, r_small, r_large, z_near;
    float fW, fH, fWm1, fHm1;
    float csmall;                // pi (1 - exp(-chi^2)): flux of the clipped unit Gaussian per sigma_px^2
    int   W, H, T, tshift;
    int   ntx, nty, n_tiles;
    int   sshift, nsx, nsy, n_super, nbins;
    int   n_big;                 // n_tiles when MEDIUM discs wider than r_route are filed in a third bin per tile (rendered by k_large), else 0
    float r_route;
    int   additive, apply_transfer;
    int   n_species, lut_total;  // lut_total: packed entries of all colour-mapped species, 0 = read tables from global
    int   any_vector, any_auto;
    int   btile, btile_r0, btile_np;   // the paper's Btile renderer (splotch_btile.cuh): MEDIUM particles binned by home tile
    float *btile_planes;         // [5][H][W][3] partial images of that renderer
    const float *vec[3];         // cr, cg, cb: per-particle vector components for species in vector colour mode
    const float2 *dev_range;     // [kMaxSpecies] {min, 1 / (max - min)} of the species with auto_range (k_range_finish)
    unsigned int sp_begin[kMaxSpecies + 1];
    SpeciesDev sp[kMaxSpecies];
    const float4 *lut;           // [kMaxSpecies][kMaxLut] rgb0
};

struct DeviceStats {             // cleared before every frame; written by k_scan / k_scatter, read back by splotch_get_stats
    unsigned long long count[4];
    unsigned long long pairs, large_pairs, chunks, capacity;
    unsigned long long sort_n;   // ordered mode: pairs the sort and the renderer work on (0 on overflow)
    // ordered mode, sort key = tile << zbits | (~bits(z_c) - zkey_min): only the bits that differ in this frame are sorted
    unsigned int zkey_max, nzkey_max, zkey_min, zbits, key_bits, pad2;     // nzkey_max = max of ~zkey (its complement is the min)
    unsigned int overflow, work_counter, chunk_size, pad3, scan_done, large_counter;   // large_counter: work items of k_large
    // additive layout (k_scan, k_layout): all offsets in 16-byte units
    unsigned int slabs, rows_per_slab, tile_units, total_units, layout_done, small_pairs;
    unsigned int slab_base[32];
    // ---- frame part: cleared once per frame.  A frame rendered in chunks (splotch_render_host streams the particle set
    //      through the device) clears only what is above between chunks and sums its totals here
    unsigned long long f_count[4], f_pairs, f_large_pairs, f_chunks;
    unsigned int f_overflow;
    unsigned int amax_bits;      // largest record amplitude so far (float bits): fixes the fixed-point unit of the tiles' sums
    int accum_exp;               // exponent the tiles' sums are held in (chunked frames: k_rescale follows amax_bits)
    unsigned int accum_exp_set;
};

struct Geo {
    int   cls;
    float px, py, sp, rp, zc;
    int   x0, x1, y0, y1;        // pixel box, inclusive
};

__device__ __forceinline__ float dot3(const float *a, float dx, float dy, float dz)
{
    return __fmaf_rn(a[2], dz, __fmaf_rn(a[1], dy, __fmul_rn(a[0], dx)));
}

constexpr float kMagic     = 12582912.0f;     // 1.5 * 2^23: v + kMagic has ulp 1 for |v| < 2^22
constexpr int   kMagicBits = 0x4B400000;

// floor / ceil of v in [-1, 2^22] as an int: v + 1.5 * 2^23 is rounded toward -inf / +inf to a multiple of one ulp = 1
// (FADD.RM / FADD.RP on the FMA pipe; the integer is the mantissa).  One add and one integer subtract per bound,
// instead of the quarter-rate conversion pipe (FRND, F2I) or a round-to-nearest add with a compare-and-fix-up.
__device__ __forceinline__ int floor_magic(float v) { return __float_as_int(__fadd_rd(v, kMagic)) - kMagicBits; }
__device__ __forceinline__ int ceil_magic(float v)  { return __float_as_int(__fadd_ru(v, kMagic)) - kMagicBits; }

// round-to-nearest-even integer of v in [-1, 32768] and the float it came from: r = rint(v), i = (int)r
__device__ __forceinline__ int rint_small(float v, float &r)
{
    const float t = __fadd_rn(v, kMagic);
    r = __fsub_rn(t, kMagic);
    return __float_as_int(t) - kMagicBits;
}

// C1 of DESIGN.md: the canonical float32 sequence (PAPER.md:76 projection, Eq. 7 :138 radius, :156-160 classes).
// Written without branches (every lane evaluates both the SMALL and the box formulas and selects): the warps of
// the streaming kernels stay converged whatever the mix of classes.  The box bounds are clamped to the screen
// BEFORE rounding, which gives the same integers as C1's "round, then clamp" (floor and ceil are monotonic, the
// clamp limits are integers, fminf / fmaxf drop a NaN operand on both sides) and keeps the rounding argument in
// the range where the addition trick is exact; a lower bound beyond the screen becomes W (H): the box is empty
// either way.
__device__ __forceinline__ Geo geometry(float x, float y, float z, float h, const FrameParams &fp)
{
    Geo g;
    const float dx = __fsub_rn(x, fp.cam[9]), dy = __fsub_rn(y, fp.cam[10]), dz = __fsub_rn(z, fp.cam[11]);
    const float xc = dot3(fp.cam + 0, dx, dy, dz);
    const float yc = dot3(fp.cam + 3, dx, dy, dz);
    g.zc = dot3(fp.cam + 6, dx, dy, dz);
    bool ok = g.zc > fp.z_near;
    const float k = __fdiv_rn(fp.cam[12], g.zc);
    g.px = __fmaf_rn(xc, k, fp.cam[13]);
    g.py = __fmaf_rn(-yc, k, fp.cam[14]);
    g.sp = __fmul_rn(h, k);
    g.rp = __fmul_rn(fp.chi, g.sp);
    ok = ok && g.rp >= 0.0f && g.rp <= 3.0e38f;
    const bool small = g.rp <= fp.r_small;
    const bool s_ok = g.px >= 0.0f && g.px < fp.fW && g.py >= 0.0f && g.py < fp.fH;
    // MEDIUM / LARGE: x0 = ceil((p - rp) - 0.5) clamped to [0, W], x1 = floor((p + rp) - 0.5) clamped to [-1, W - 1]
    const int x0m = ceil_magic(fminf(fmaxf(__fsub_rn(__fsub_rn(g.px, g.rp), 0.5f), 0.0f), fp.fW));
    const int y0m = ceil_magic(fminf(fmaxf(__fsub_rn(__fsub_rn(g.py, g.rp), 0.5f), 0.0f), fp.fH));
    const int x1m = floor_magic(fmaxf(fminf(__fsub_rn(__fadd_rn(g.px, g.rp), 0.5f), fp.fWm1), -1.0f));
    const int y1m = floor_magic(fmaxf(fminf(__fsub_rn(__fadd_rn(g.py, g.rp), 0.5f), fp.fHm1), -1.0f));
    // SMALL: the pixel that holds the centre (used only when s_ok: 0 <= p < W <= 32768)
    const int x0s = floor_magic(g.px), y0s = floor_magic(g.py);
    const bool b_ok = x0m <= x1m && y0m <= y1m;
    const int big = (g.rp <= fp.r_large) ? MEDIUM : LARGE;
    g.cls = ok ? (small ? (s_ok ? SMALL : CULLED) : (b_ok ? big : CULLED)) : CULLED;
    const bool act = g.cls != CULLED;
    g.x0 = act ? (small ? x0s : x0m) : 0;
    g.x1 = act ? (small ? x0s : x1m) : -1;
    g.y0 = act ? (small ? y0s : y0m) : 0;
    g.y1 = act ? (small ? y0s : y1m) : -1;
    return g;
}

// The paper's tile index i(p).
__device__ __forceinline__ int paper_label(const Geo &g, const FrameParams &fp)
{
    if (g.cls == CULLED) return -2;
    if (g.cls == LARGE) return -1;
    if (g.cls == SMALL) return fp.n_tiles;
    const float cx = fminf(fmaxf(floorf(g.px), 0.0f), __fsub_rn(fp.fW, 1.0f));
    const float cy = fminf(fmaxf(floorf(g.py), 0.0f), __fsub_rn(fp.fH, 1.0f));
    return ((int)cy >> fp.tshift) * fp.ntx + ((int)cx >> fp.tshift);
}

// tile of the (clamped) centre pixel: the paper's i(p) of a MEDIUM particle
__device__ __forceinline__ int2 home_tile(const Geo &g, const FrameParams &fp)
{
    const float cx = fminf(fmaxf(floorf(g.px), 0.0f), __fsub_rn(fp.fW, 1.0f));
    const float cy = fminf(fmaxf(floorf(g.py), 0.0f), __fsub_rn(fp.fH, 1.0f));
    return make_int2((int)cx >> fp.tshift, (int)cy >> fp.tshift);
}

// ---- bins ----------------------------------------------------------------------------------------------------------
// Bin b < 2 n_tiles: tile b >> 1; even bins hold the tile's MEDIUM records (32 bytes = 2 units of 16 bytes), odd bins
// its SMALL records (16 bytes = 1 unit: "only their location ... has to be calculated").  Bins
// 2 n_tiles + s hold the LARGE records of super-tile s (2 units).  A tile's two bins are neighbours, so the tile
// renderer meets them back to back.  With 32-px tiles there is a third bin per tile, 2 n_tiles + n_super + t: the MEDIUM records of
// tile t whose disc is wider than kRouteRadius.  They are tile assignments like the others (the per-tile pair counts include them) but
// k_large renders them, the tile as its 32 x 32 block: k_splat's 64-pixel strips spent 20 warp instructions per record and strip on
// them (cfg3: 80 ms), k_large's bands 61 per 256 pixels or the tensor cores.  cfg3 frame by kRouteRadius: none 341.5 ms, 12 px 333.0,
// 24 px 330.5, 40 px 329.9 (k_splat 80 -> 24 ms, k_large 245 -> 289 ms).
__device__ __forceinline__ unsigned int bin_unit_size(int b, int n_tiles) { return (b < 2 * n_tiles && (b & 1)) ? 1u : 2u; }

// ---- streaming loads / stores ----------------------------------------------------------------------------------
__device__ __forceinline__ float4 ldg_stream4(const float *p)
{
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// one 32-byte render record at 16-byte unit `unit` (even), one request (256-bit global access, sm_100)
__device__ __forceinline__ void st_record(float4 *rec, unsigned int unit, const float4 &a, const float4 &b)
{
    asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 :: "l"(rec + unit), "f"(a.x), "f"(a.y), "f"(a.z), "f"(a.w), "f"(b.x), "f"(b.y), "f"(b.z), "f"(b.w)
                 : "memory");
}

__device__ __forceinline__ void ld_record(const float4 *rec, unsigned int slot, float4 &a, float4 &b)
{
    asm volatile("ld.global.nc.L1::no_allocate.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w)
                 : "l"(rec + 2ull * slot));
}

template <bool ALIGNED>
__device__ __forceinline__ void load4(const float *__restrict__ a, unsigned int i, unsigned int len, float (&v)[4])
{
    if (ALIGNED && i + 4 <= len) {
        const float4 q = ldg_stream4(a + i);
        v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) v[j] = (i + j < len) ? __ldg(a + i + j) : 0.0f;
    }
}

// histogram / cursor update without a return value: shared memory (the common case) or, when the bins of a large
// image do not fit in shared memory, the block's own row of the count matrix in global memory (L2 resident)
template <bool GHIST>
__device__ __forceinline__ void hist_inc(unsigned int *p)
{
    if (GHIST) asm volatile("red.global.add.u32 [%0], 1;" :: "l"(p) : "memory");
    else asm volatile("red.shared.add.u32 [%0], 1;" :: "r"((unsigned int)__cvta_generic_to_shared(p)) : "memory");
}

__device__ __forceinline__ unsigned int warp_sum(unsigned int v)
{
    return __reduce_add_sync(0xffffffffu, v);
}

// ---- A1 + A3 + A4a: classify and count ------------------------------------------------------------------------
// Block b owns the particle range [b*per, (b+1)*per) and a private histogram over all bins; row b of `counts`
// receives it, so the count stage needs no atomics between blocks and is deterministic.
// Bins of an active particle: the tiles of its pixel box (SMALL: its pixel's tile, odd bin; MEDIUM: even bins) or the
// super-tiles of the box (LARGE).  k_count and k_scatter walk them with ONE warp-uniform loop (lanes whose box is
// exhausted idle): a single call site keeps the kernels small (divergent per-lane loops with several inlined record
// writers ran at 5 active lanes per instruction and stalled on instruction fetch on cfg3, profiles/r2_step3_*).
struct BinWalk {
    int bx0, bx1, by0, by1, sh, pitch, base, mult, odd, n;      // bin = base + mult * (by * pitch + bx) + odd
    int route;                                                  // 0 tile bins, 1 super-tile bins (LARGE), 2 the tile's bin for wide MEDIUM discs
};

template <bool BTILE>
__device__ __forceinline__ BinWalk bin_walk(const Geo &g, int cls, const FrameParams &fp)
{
    BinWalk w;
    const bool large = cls == LARGE;
    const bool wide = !BTILE && cls == MEDIUM && fp.n_big > 0 && g.rp > fp.r_route;
    w.route = large ? 1 : (wide ? 2 : 0);
    w.sh = large ? fp.sshift : fp.tshift;
    w.pitch = large ? fp.nsx : fp.ntx;
    w.base = large ? 2 * fp.n_tiles : (wide ? 2 * fp.n_tiles + fp.n_super : 0);
    w.mult = (large || wide) ? 1 : 2;
    w.odd = cls == SMALL ? 1 : 0;
    w.bx0 = g.x0 >> w.sh; w.bx1 = g.x1 >> w.sh; w.by0 = g.y0 >> w.sh; w.by1 = g.y1 >> w.sh;
    if (BTILE && cls == MEDIUM) { const int2 ht = home_tile(g, fp); w.bx0 = w.bx1 = ht.x; w.by0 = w.by1 = ht.y; }   // i(p): the tile of the centre
    w.n = cls == CULLED ? 0 : (w.bx1 - w.bx0 + 1) * (w.by1 - w.by0 + 1);
    return w;
}

// The bins of the lanes whose box covers more than a few bins, walked by the whole warp: the lanes' bin counts are prefix-summed and the
// warp takes 32 (lane, bin) pairs per step, whichever lanes they come from.  (One warp-uniform loop in which every lane walked its own
// box ran as long as the largest box of the warp: 20 steps for two or three busy lanes on cfg3, where discs of 64 px cover 5 x 5 tiles
// and LARGE discs several super-tiles; profiles/r2_step1_*: 15.7 warp instructions per particle in k_count against 5.3 on cfg2.)
// emit(ok, source lane, bx, by, route of the source) is called by all lanes together.
__device__ __forceinline__ int routed_bin(int route, int bx, int by, const FrameParams &fp)
{
    return route == 1 ? 2 * fp.n_tiles + by * fp.nsx + bx : (route == 2 ? 2 * fp.n_tiles + fp.n_super + by * fp.ntx + bx : 2 * (by * fp.ntx + bx));
}

template <typename Emit>
__device__ __forceinline__ void coop_bin_walk(bool big, const BinWalk &w, int lane, Emit emit)
{
    const unsigned int cnt = big ? (unsigned int)w.n : 0u;
    unsigned int inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    const unsigned int total = __shfl_sync(0xffffffffu, inc, 31), excl = inc - cnt;
    const int width = w.bx1 - w.bx0 + 1;
#pragma unroll 1
    for (unsigned int f0 = 0u; f0 < total; f0 += 32u) {
        const unsigned int f = f0 + (unsigned int)lane;
        int sl = 0;                                  // the last lane whose exclusive prefix is <= f (prefixes ascend; lanes without bins share their successor's)
#pragma unroll
        for (int st = 16; st >= 1; st >>= 1) {
            const unsigned int e = __shfl_sync(0xffffffffu, excl, sl + st);
            if (e <= f) sl += st;
        }
        const unsigned int se = __shfl_sync(0xffffffffu, excl, sl);
        const int sbx0 = __shfl_sync(0xffffffffu, w.bx0, sl), sby0 = __shfl_sync(0xffffffffu, w.by0, sl);
        const int sw = __shfl_sync(0xffffffffu, width, sl), sroute = __shfl_sync(0xffffffffu, w.route, sl);
        const unsigned int k = f - se;
        const int ky = __float2int_rz(__fdividef((float)k + 0.5f, (float)sw)), kx = (int)k - ky * sw;     // k / width, k % width (k < 2^20)
        emit(f < total, sl, sbx0 + kx, sby0 + ky, sroute);
    }
}

template <bool ALIGNED, bool GHIST, bool BTILE>
__global__ void __launch_bounds__(kBinThreads, 1)
k_count(const float *__restrict__ x, const float *__restrict__ y, const float *__restrict__ z,
        const float *__restrict__ h, unsigned long long n, unsigned long long per, const __grid_constant__ FrameParams fp,
        unsigned int *__restrict__ counts, unsigned int *__restrict__ cls_counts)
{
    extern __shared__ unsigned int hist_s[];
    __shared__ unsigned int s_cls[4];
    unsigned int *row = counts + (size_t)blockIdx.x * fp.nbins;
    unsigned int *hist = GHIST ? row : hist_s;          // GHIST: the row was cleared with the frame's memset
    if (!GHIST) for (int i = threadIdx.x; i < fp.nbins; i += kBinThreads) hist_s[i] = 0u;
    if (threadIdx.x < 4) s_cls[threadIdx.x] = 0u;
    __syncthreads();
    const unsigned long long lo = (unsigned long long)blockIdx.x * per;
    const unsigned int len = lo < n ? (unsigned int)min(n - lo, per) : 0u;
    x += lo; y += lo; z += lo; h += lo;
    unsigned int c2 = 0, c3 = 0;                  // MEDIUM / LARGE particles of this thread (SMALL ones are the sum of the odd bins)
    // the loop bound is the same for the 32 lanes of a warp (lanes past the end idle), so warps stay converged
    const unsigned int lane4 = 4u * (threadIdx.x & 31u);
    for (unsigned int iw = 4u * (threadIdx.x & ~31u); iw < len; iw += 4u * kBinThreads) {
        const unsigned int i = iw + lane4;
        float xs[4], ys[4], zs[4], hs[4];
        load4<ALIGNED>(x, i, len, xs);
        load4<ALIGNED>(y, i, len, ys);
        load4<ALIGNED>(z, i, len, zs);
        load4<ALIGNED>(h, i, len, hs);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const Geo g = geometry(xs[j], ys[j], zs[j], hs[j], fp);
            const int cls = (i + j < len) ? g.cls : CULLED;
            c2 += cls == MEDIUM; c3 += cls == LARGE;
            const BinWalk w = bin_walk<BTILE>(g, cls, fp);
            // a box covers at most 2 x 2 bins unless it is wider than a bin: four predicated increments; the others go to the warp's
            // common walk
            unsigned int *h00 = hist + (w.base + w.mult * (w.by0 * w.pitch + w.bx0) + w.odd);
            const bool any = w.n > 0, w2 = w.bx1 > w.bx0, h2 = w.by1 > w.by0;
            const bool big = any && (w.bx1 - w.bx0 > 1 || w.by1 - w.by0 > 1);
            const bool few = any && !big;
            if (few) hist_inc<GHIST>(h00);
            if (few && w2) hist_inc<GHIST>(h00 + w.mult);
            if (few && h2) hist_inc<GHIST>(h00 + w.mult * w.pitch);
            if (few && w2 && h2) hist_inc<GHIST>(h00 + w.mult * w.pitch + w.mult);
            if (__any_sync(0xffffffffu, big))
                coop_bin_walk(big, w, (int)(threadIdx.x & 31u), [&](bool ok, int, int bx, int by, int route) {
                    if (ok) hist_inc<GHIST>(hist + routed_bin(route, bx, by, fp));
                });
        }
    }
    c2 = warp_sum(c2); c3 = warp_sum(c3);
    if ((threadIdx.x & 31) == 0) { atomicAdd(&s_cls[2], c2); atomicAdd(&s_cls[3], c3); }
    __syncthreads();
    if (!GHIST) for (int i = threadIdx.x; i < fp.nbins; i += kBinThreads) row[i] = hist_s[i];
    if (threadIdx.x == 0) s_cls[0] = len;           // particles of this block: k_scan turns it into the CULLED count
    __syncthreads();
    if (threadIdx.x < 4) cls_counts[blockIdx.x * 4 + threadIdx.x] = s_cls[threadIdx.x];
}

// ---- A4b + A4c: scans ----------------------------------------------------------------------------------------------
constexpr int kScanThreads = 256;
constexpr int kMaxSlabs = 32;                 // the record array is cut into at most 32 slabs (one lane of a warp each)
constexpr unsigned int kSlabBytes = 96u << 20;   // target size of a slab (see k_scan)

__device__ __forceinline__ unsigned long long block_excl_scan_256(unsigned long long v, unsigned long long *s_warp,
                                                                  unsigned long long *total)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned long long inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_warp[w] = inc;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long run = 0;
        for (int k = 0; k < kScanThreads / 32; ++k) { const unsigned long long c = s_warp[k]; s_warp[k] = run; run += c; }
        *total = run;
    }
    __syncthreads();
    const unsigned long long r = s_warp[w] + inc - v;
    __syncthreads();
    return r;
}

// Phase 1, every block: 32 bins x 8 row groups.  Thread (bin, g) sums its rows of the count matrix (independent
// loads, bins of neighbouring lanes are neighbours in memory), the groups are combined through shared memory, and
// the rows are rewritten as exclusive prefixes: counts[b][bin] becomes the number of the bin's records that blocks
// before b produce.
// Phase 2, the last block to finish (a counter in DeviceStats, cleared with it before every frame): the frame's
// statistics and its layout parameters:
//   * vstart[bin], the bin's first 16-byte unit in the VIRTUAL order the renderers consume (bin after bin; a bin's
//     units are padded to an even number so that 32-byte records never straddle a chunk boundary); the tile part,
//     [0, tile_units), is cut into chunks of chunk_size units, the work items of k_splat;
//   * the number of slabs: in MEMORY the records are slab-major.  The count / scatter blocks are divided into groups of
//     rows_per_slab consecutive blocks; a group writes its records, bin after bin, into its own contiguous slab of about
//     96 MB.  A block's stores then stay inside a window the TLB covers (256 MB) instead of wandering over the whole
//     array (measured: 32-byte stores spread over 4 GB reach 1.2 TB/s, inside 128 MB windows 2.3 - 5.8 TB/s depending on
//     the number of bins); the renderers read a bin as `slabs` runs (k_layout builds the run table);
//   * the item table of k_large.
__global__ void __launch_bounds__(kScanThreads)
k_scan(unsigned int *__restrict__ counts, int nrows, int nbins, int n_tiles, unsigned int *__restrict__ bin_count,
       unsigned int *__restrict__ vstart, const unsigned int *__restrict__ cls_counts, unsigned long long capacity_units, int n_sm,
       unsigned int *__restrict__ large_off, unsigned int large_chunk, unsigned int large_blocks, int n_super, DeviceStats *__restrict__ stats)
{
    __shared__ unsigned int s_part[8][32];
    __shared__ unsigned long long s_warp[kScanThreads / 32];
    __shared__ unsigned long long s_tot_tiles, s_tot_all, s_tot_items, s_tot_small;
    __shared__ unsigned int s_ticket, s_cls[4];
    {
        const int bin = blockIdx.x * 32 + (threadIdx.x & 31), g = threadIdx.x >> 5;
        const int rpg = (nrows + 7) / 8;
        const int rb = min(nrows, g * rpg), re = min(nrows, rb + rpg);
        unsigned int sum = 0;
        if (bin < nbins) {
            int r = rb;
            for (; r + 8 <= re; r += 8) {
                unsigned int c[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) c[k] = counts[(size_t)(r + k) * nbins + bin];
#pragma unroll
                for (int k = 0; k < 8; ++k) sum += c[k];
            }
            for (; r < re; ++r) sum += counts[(size_t)r * nbins + bin];
        }
        s_part[g][threadIdx.x & 31] = sum;
        __syncthreads();
        unsigned int run = 0;
        for (int k = 0; k < g; ++k) run += s_part[k][threadIdx.x & 31];
        if (bin < nbins) {
            if (g == 7) bin_count[bin] = run + sum;
            int r = rb;
            for (; r + 8 <= re; r += 8) {
                unsigned int c[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) c[k] = counts[(size_t)(r + k) * nbins + bin];
#pragma unroll
                for (int k = 0; k < 8; ++k) { counts[(size_t)(r + k) * nbins + bin] = run; run += c[k]; }
            }
            for (; r < re; ++r) {
                const unsigned int c = counts[(size_t)r * nbins + bin];
                counts[(size_t)r * nbins + bin] = run;
                run += c;
            }
        }
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_ticket = atomicAdd(&stats->scan_done, 1u);
    __syncthreads();
    if (s_ticket != gridDim.x - 1) return;
    __threadfence();
    // ---- phase 2: one block.  Units of a bin: records x unit size, padded to even
    const int per = (nbins + kScanThreads - 1) / kScanThreads;
    const int b0 = min(nbins, (int)threadIdx.x * per), b1 = min(nbins, b0 + per);
    unsigned long long u_all = 0, u_tiles = 0, n_small = 0, n_tilerec = 0, n_largerec = 0;
    for (int bb = b0; bb < b1; bb += 8) {
        unsigned int c8[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) c8[k] = (bb + k < b1) ? __ldcg(bin_count + bb + k) : 0u;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int b = bb + k;
            const unsigned int u = (c8[k] * bin_unit_size(b, n_tiles) + 1u) & ~1u;
            u_all += u;
            if (b < 2 * n_tiles) { u_tiles += u; n_tilerec += c8[k]; if (b & 1) n_small += c8[k]; }
            else if (b < 2 * n_tiles + n_super) n_largerec += c8[k];
            else n_tilerec += c8[k];                 // wide MEDIUM discs: tile pairs, rendered by k_large
        }
    }
    if (threadIdx.x < 4) s_cls[threadIdx.x] = 0u;
    __syncthreads();
    {   // class counts: every thread sums a strided share of the per-block counts
        unsigned int c[4] = {0u, 0u, 0u, 0u};
        for (int r = threadIdx.x; r < nrows; r += kScanThreads) {
            const uint4 v = *reinterpret_cast<const uint4 *>(cls_counts + 4 * r);
            c[0] += v.x; c[1] += v.y; c[2] += v.z; c[3] += v.w;
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const unsigned int t = __reduce_add_sync(0xffffffffu, c[k]);
            if ((threadIdx.x & 31) == 0 && t) atomicAdd(&s_cls[k], t);
        }
    }
    const unsigned long long off_all = block_excl_scan_256(u_all, s_warp, &s_tot_all);
    (void)block_excl_scan_256(u_tiles, s_warp, &s_tot_tiles);
    (void)block_excl_scan_256(n_small, s_warp, &s_tot_small);
    const unsigned long long tile_records = block_excl_scan_256(n_tilerec, s_warp, &s_tot_items) * 0ull + s_tot_items;
    const unsigned long long large_records = block_excl_scan_256(n_largerec, s_warp, &s_tot_items) * 0ull + s_tot_items;
    // chunk size of this frame, in units: about 128 chunks per SM (work items are taken from an atomic counter; many
    // small ones keep the tail short when their costs differ), between kChunkMin and kChunkMax
    unsigned long long cs = (s_tot_tiles + (unsigned long long)n_sm * 128 - 1) / ((unsigned long long)n_sm * 128);
    cs = cs >= 1024 ? (cs + 511) / 512 * 512 : (cs + 127) / 128 * 128;      // small frames: short chunks, they are latency bound
    cs = min((unsigned long long)kChunkMax, max((unsigned long long)kChunkMin, cs));
    const unsigned int K = (unsigned int)cs;
    // capacity counts true record units; the padding of bins and runs has its own allowance in the workspace
    const bool overflow = 2ull * (tile_records - s_tot_small) + s_tot_small + 2ull * large_records > capacity_units || s_tot_all > 0xffff0000ull;
    unsigned long long run = off_all;
    for (int bb = b0; bb < b1; bb += 8) {            // eight independent loads per round (this block is latency bound)
        unsigned int c8[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) c8[k] = (bb + k < b1) ? __ldcg(bin_count + bb + k) : 0u;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            if (bb + k < b1) vstart[bb + k] = (unsigned int)run;
            run += (c8[k] * bin_unit_size(bb + k, n_tiles) + 1u) & ~1u;
        }
    }
    if (threadIdx.x == kScanThreads - 1) vstart[nbins] = (unsigned int)s_tot_all;
    {   // work items of k_large: (chunk of a super-tile's records) x (block of the super-tile), exclusive prefix over the super-tiles
        // regions: the super-tiles (large_blocks blocks each), then the tiles' bins of wide MEDIUM discs (the tile is the one block)
        const int n_reg = nbins - 2 * n_tiles;
        const int sper = (n_reg + kScanThreads - 1) / kScanThreads;
        const int s0 = min(n_reg, (int)threadIdx.x * sper), s1 = min(n_reg, s0 + sper);
        unsigned long long items = 0;
        for (int sb = s0; sb < s1; ++sb) items += (unsigned long long)((__ldcg(bin_count + 2 * n_tiles + sb) + large_chunk - 1) / large_chunk) * (sb < n_super ? large_blocks : 1u);
        unsigned long long irun = block_excl_scan_256(items, s_warp, &s_tot_items);
        for (int sb = s0; sb < s1; ++sb) {
            large_off[sb] = overflow ? 0u : (unsigned int)irun;
            irun += (unsigned long long)((__ldcg(bin_count + 2 * n_tiles + sb) + large_chunk - 1) / large_chunk) * (sb < n_super ? large_blocks : 1u);
        }
        if (threadIdx.x == kScanThreads - 1) large_off[n_reg] = overflow ? 0u : (unsigned int)irun;
    }
    if (threadIdx.x == 0) {
        // slabs of about 96 MB, at most 32 and at most one per row
        unsigned int G = (unsigned int)((s_tot_all * 16ull + kSlabBytes - 1) / kSlabBytes);
        G = max(1u, min(min(G, (unsigned int)kMaxSlabs), (unsigned int)nrows));
        const unsigned int cps = ((unsigned int)nrows + G - 1) / G;
        stats->slabs = ((unsigned int)nrows + cps - 1) / cps;
        stats->rows_per_slab = cps;
        stats->tile_units = overflow ? 0u : (unsigned int)s_tot_tiles;
        stats->total_units = overflow ? 0u : (unsigned int)s_tot_all;
        stats->count[0] = (unsigned long long)s_cls[0] - s_tot_small - s_cls[2] - s_cls[3];
        stats->count[1] = s_tot_small;
        stats->count[2] = s_cls[2];
        stats->count[3] = s_cls[3];
        stats->pairs = tile_records;
        stats->small_pairs = s_tot_small;
        stats->large_pairs = large_records;
        stats->chunks = overflow ? 0ull : (s_tot_tiles + K - 1) / K;
        stats->capacity = capacity_units / 2;
        stats->overflow = overflow ? 1u : 0u;
        stats->work_counter = 0u;
        stats->chunk_size = K;
        stats->scan_done = 0u;
        // totals of the frame (the only chunk of a one-shot frame, or this chunk added to the earlier ones)
        stats->f_count[0] += stats->count[0]; stats->f_count[1] += s_tot_small; stats->f_count[2] += s_cls[2]; stats->f_count[3] += s_cls[3];
        stats->f_pairs += tile_records; stats->f_large_pairs += large_records;
        stats->f_chunks += stats->chunks;
        stats->f_overflow |= overflow ? 1u : 0u;
    }
}

// Chunked frames: the fixed-point unit of the tiles' sums follows the largest record amplitude seen so far.  When a chunk
// raises it, the sums of the earlier chunks are shifted to the new unit (rounded to nearest) before the chunk is added.
__global__ void __launch_bounds__(256)
k_rescale(long long *__restrict__ accum, size_t n, const DeviceStats *__restrict__ stats);
__global__ void k_rescale_done(DeviceStats *stats);

// One block per slab s (blocks beyond the frame's slab count leave at once): the slab's runs.  Run (s, bin) holds the
// bin's records that the rows of slab s produce: cnt = P[(s + 1) rows_per_slab][bin] - P[s rows_per_slab][bin] with P the
// exclusive row prefixes k_scan left in `counts`; the runs of a slab follow each other in bin order, each padded to an
// even number of units.  run[bin * 32 + s] = {first unit inside the slab, records}; the last block to finish turns the slab
// sizes into slab_base[] (DeviceStats).
constexpr int kLayoutThreads = 1024;

__global__ void __launch_bounds__(kLayoutThreads)
k_layout(const unsigned int *__restrict__ counts, const unsigned int *__restrict__ bin_count, int nrows, int nbins, int n_tiles,
         uint2 *__restrict__ run, DeviceStats *__restrict__ stats)
{
    __shared__ unsigned int s_warp[32], s_total;
    __shared__ unsigned int s_ticket;
    const unsigned int G = stats->slabs, cps = stats->rows_per_slab;
    const unsigned int s = blockIdx.x;
    if (s < G) {
        const unsigned int rlo = s * cps, rhi = (s + 1) * cps;
        const unsigned int *plo = counts + (size_t)rlo * nbins;
        const unsigned int *phi = rhi < (unsigned int)nrows ? counts + (size_t)rhi * nbins : bin_count;
        const int per = (nbins + kLayoutThreads - 1) / kLayoutThreads;
        const int b0 = min(nbins, (int)threadIdx.x * per), b1 = min(nbins, b0 + per);
        unsigned int sum = 0u;
        for (int b = b0; b < b1; ++b) sum += ((__ldcg(phi + b) - __ldcg(plo + b)) * bin_unit_size(b, n_tiles) + 1u) & ~1u;
        const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        unsigned int inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_warp[w] = inc;
        __syncthreads();
        if (w == 0) {
            const unsigned int c = s_warp[lane];
            unsigned int ci = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned int t = __shfl_up_sync(0xffffffffu, ci, o);
                if (lane >= o) ci += t;
            }
            s_warp[lane] = ci - c;
            if (lane == 31) s_total = ci;
        }
        __syncthreads();
        unsigned int off = s_warp[w] + inc - sum;
        for (int b = b0; b < b1; ++b) {
            const unsigned int cnt = __ldcg(phi + b) - __ldcg(plo + b);
            run[(size_t)b * kMaxSlabs + s] = make_uint2(off, cnt);
            off += (cnt * bin_unit_size(b, n_tiles) + 1u) & ~1u;
        }
        if (threadIdx.x == 0) stats->slab_base[s] = s_total;        // the slab's size for now
    } else {
        for (int b = threadIdx.x; b < nbins; b += kLayoutThreads) run[(size_t)b * kMaxSlabs + s] = make_uint2(0u, 0u);   // no such run
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_ticket = atomicAdd(&stats->layout_done, 1u);
    __syncthreads();
    if (s_ticket != gridDim.x - 1) return;
    __threadfence();
    if (threadIdx.x == 0) {
        unsigned int base = 0u;
        for (unsigned int k = 0; k < (unsigned int)kMaxSlabs; ++k) {
            const unsigned int sz = k < G ? *(volatile unsigned int *)&stats->slab_base[k] : 0u;
            stats->slab_base[k] = base;
            base += sz;
        }
        stats->layout_done = 0u;
    }
}

// ---- pre-processing: normalisation range found from the data (PAPER.md:76, :166 fn. 1) ----------------------------
// Floats as unsigned keys whose order is the order of the values, so that atomicMin / atomicMax reduce them.
__device__ __forceinline__ unsigned int float_key(float v) { const unsigned int b = __float_as_uint(v); return (b & 0x80000000u) ? ~b : b | 0x80000000u; }
__device__ __forceinline__ float key_float(unsigned int k) { return __uint_as_float((k & 0x80000000u) ? k & 0x7fffffffu : ~k); }

struct RangeRaw { unsigned int kmin, kmax; };            // per species; k_range_init sets {0xffffffff, 0}

__global__ void k_range_init(RangeRaw *raw) { if (threadIdx.x < kMaxSpecies) raw[threadIdx.x] = RangeRaw{0xffffffffu, 0u}; }

// min / max of the finite values of v[0, n) (log10 first when asked), reduced into raw[s]
__global__ void __launch_bounds__(512)
k_minmax(const float *__restrict__ v, unsigned long long n, int use_log10, RangeRaw *__restrict__ raw, int s)
{
    unsigned int kmin = 0xffffffffu, kmax = 0u;
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (unsigned long long)gridDim.x * blockDim.x) {
        float x = __ldg(v + i);
        if (use_log10) x = log10f(x);
        if (x >= -3.0e38f && x <= 3.0e38f) { const unsigned int k = float_key(x); kmin = min(kmin, k); kmax = max(kmax, k); }
    }
    kmin = __reduce_min_sync(0xffffffffu, kmin); kmax = __reduce_max_sync(0xffffffffu, kmax);
    if ((threadIdx.x & 31) == 0 && kmin <= kmax) { atomicMin(&raw[s].kmin, kmin); atomicMax(&raw[s].kmax, kmax); }
}

// {min, 1 / (max - min)} per species; a species without a finite value gets the range (0, 1)
__global__ void k_range_finish(const RangeRaw *__restrict__ raw, float2 *__restrict__ out)
{
    if (threadIdx.x < kMaxSpecies) {
        const RangeRaw r = raw[threadIdx.x];
        const float lo = r.kmin <= r.kmax ? key_float(r.kmin) : 0.0f, hi = r.kmin <= r.kmax ? key_float(r.kmax) : 1.0f;
        out[threadIdx.x] = make_float2(lo, __fdiv_rn(1.0f, __fsub_rn(hi, lo)));
    }
}

// ---- A2: colour + amplitude (PAPER.md:76 normalisation/log, :85 look-up table) -------------------------------
__device__ __forceinline__ int species_of(unsigned int i, const FrameParams &fp)
{
    int s = 0;
#pragma unroll
    for (int k = 1; k < kMaxSpecies; ++k) s += (k < fp.n_species && i >= fp.sp_begin[k]);
    return s;
}

// lut: the species' table (shared or global memory), lut_n entries.  Colour and amplitude are continuous in the
// inputs (no integer is decided here beyond the table cell), so plain float32 with a reciprocal range is enough.
__device__ __forceinline__ float3 colour_of(float scalar, const SpeciesDev &S, const float4 *lut, float2 rng, float3 vec)
{
    float r = S.fixed_r, g = S.fixed_g, b = S.fixed_b;
    if (S.vector) {                                // rho^R = v_x, rho^G = v_y, rho^B = v_z, normalised like the scalar
        const float tr = (vec.x - rng.x) * rng.y, tg = (vec.y - rng.x) * rng.y, tb = (vec.z - rng.x) * rng.y;
        r = fminf(tr > 0.0f ? tr : 0.0f, 1.0f);
        g = fminf(tg > 0.0f ? tg : 0.0f, 1.0f);
        b = fminf(tb > 0.0f ? tb : 0.0f, 1.0f);
    } else if (S.use_colormap) {
        float v = scalar;
        if (S.use_log10) v = log10f(v);
        float t = (v - rng.x) * rng.y;
        t = (t > 0.0f) ? t : 0.0f;                 // NaN clamps to 0
        t = fminf(t, 1.0f);
        const float u = t * S.lut_nm1;             // 0 <= u <= lut_n - 1 <= 1023
        float ru;
        int i0 = rint_small(u, ru);
        const bool up = ru > u;                    // rint rounded up: floor is one below
        i0 = min(i0 - (up ? 1 : 0), S.lut_n - 2);
        const float f0 = fminf(ru - (up ? 1.0f : 0.0f), S.lut_nm2);
        const float fr = u - f0;
        const float4 a = lut[i0];
        const float4 c = lut[i0 + 1];
        r = fmaf(fr, c.x - a.x, a.x);
        g = fmaf(fr, c.y - a.y, a.y);
        b = fmaf(fr, c.z - a.z, a.z);
    }
    return make_float3(r, g, b);
}

// normalisation range of a species: the caller's, or the one found on the device (k_minmax / k_range_finish)
__device__ __forceinline__ float2 species_range(const FrameParams &fp, int s)
{
    return fp.sp[s].auto_range ? fp.dev_range[s] : make_float2(fp.sp[s].smin, fp.sp[s].inv_range);
}

// E_p * (column constant) = b_s * colour * sqrt(pi) h I (R12, R13)
__device__ __forceinline__ float3 amplitude(float I, float scalar, float h, const SpeciesDev &S, const float4 *lut, float2 rng, float3 vec)
{
    const float3 c = colour_of(scalar, S, lut, rng, vec);
    const float col = S.brightness * (1.7724538509055160273f * h * I);   // b_s * sqrt(pi) h I
    return make_float3(c.x * col, c.y * col, c.z * col);
}

// Render records.
//   MEDIUM / LARGE, 32 bytes: {px, py, c, r2} {aR, aG, aB, box}
//     c = -log2(e) / sp^2, r2 = rp^2 (float32, the C1 inside test compares d2 with it), a = E * col.
//     box: the particle's pixel box clipped to the bin it is filed under, relative to the bin's origin.  Tile bins
//     (MEDIUM): x0 | y0 << 6 | (x1 - x0) << 12 | (y1 - y0) << 18.  Super-tile bins (LARGE): x0 | y0 << 8 | x1 << 16 |
//     y1 << 24.  The renderers never round a float again.
//   SMALL, 16 bytes: {pixel, aR, aG, aB}: pixel = y * T + x inside the tile, a = E * col * pi sp^2 (1 - exp(-chi^2)),
//     the whole clipped flux (R6): a SMALL particle needs "only its location".
// A record whose amplitude is not finite (I or scalar = Inf / NaN) carries amplitude 0.
// box of the particle clipped to bin (bx, by), relative to the bin's origin
__device__ __forceinline__ unsigned int pack_box(const Geo &g, int bx, int by, int sh, bool large)
{
    const int ox = bx << sh, oy = by << sh, m = (1 << sh) - 1;
    const int cx0 = max(g.x0 - ox, 0), cx1 = min(g.x1 - ox, m), cy0 = max(g.y0 - oy, 0), cy1 = min(g.y1 - oy, m);
    return large ? ((unsigned int)cx0 | ((unsigned int)cy0 << 8) | ((unsigned int)cx1 << 16) | ((unsigned int)cy1 << 24))
                 : ((unsigned int)cx0 | ((unsigned int)cy0 << 6) | ((unsigned int)(cx1 - cx0) << 12) | ((unsigned int)(cy1 - cy0) << 18));
}

// next free unit of a bin's run: shared-memory cursor, or the block's row of the count matrix (see hist_inc)
template <bool GHIST>
__device__ __forceinline__ unsigned int cursor_take(unsigned int *p, unsigned int units)
{
    return atomicAdd(p, units);
}

template <bool ALIGNED, bool GHIST, bool BTILE>
__global__ void __launch_bounds__(kBinThreads, 1)
k_scatter(const float *__restrict__ x, const float *__restrict__ y, const float *__restrict__ z,
          const float *__restrict__ h, const float *__restrict__ I, const float *__restrict__ scalar,
          unsigned long long n, unsigned long long per, const __grid_constant__ FrameParams fp,
          const unsigned int *__restrict__ counts, unsigned int *__restrict__ cursor_rows, const uint2 *__restrict__ run,
          DeviceStats *__restrict__ stats, float4 *__restrict__ records)
{
    extern __shared__ unsigned int cursor_s[];               // nbins cursors, then the packed colour tables
    __shared__ float s_amax[kBinThreads / 32];
    __shared__ float2 s_rng[kMaxSpecies];
    if (stats->overflow) return;
    if (threadIdx.x < kMaxSpecies) s_rng[threadIdx.x] = threadIdx.x < fp.n_species ? species_range(fp, threadIdx.x) : make_float2(0.0f, 0.0f);
    float4 *s_lut = reinterpret_cast<float4 *>(cursor_s + (GHIST ? 0 : ((fp.nbins + 3) & ~3)));
    // this block's cursors: slab base + the run's first unit + the units of the slab's rows before this one
    const unsigned int *row = counts + (size_t)blockIdx.x * fp.nbins;
    unsigned int *cursor = GHIST ? cursor_rows + (size_t)blockIdx.x * fp.nbins : cursor_s;     // GHIST: a row of its own in global memory
    {
        const unsigned int cps = stats->rows_per_slab, s = blockIdx.x / cps;
        const unsigned int base = stats->slab_base[s];
        const unsigned int *row0 = counts + (size_t)(s * cps) * fp.nbins;
        const bool first = blockIdx.x == s * cps;
        for (int i = threadIdx.x; i < fp.nbins; i += kBinThreads) {
            const unsigned int before = first ? 0u : row[i] - row0[i];
            cursor[i] = base + run[(size_t)i * kMaxSlabs + s].x + before * bin_unit_size(i, fp.n_tiles);
        }
    }
    if (fp.lut_total > 0) {
        for (int s = 0; s < fp.n_species; ++s)
            if (fp.sp[s].use_colormap)
                for (int i = threadIdx.x; i < fp.sp[s].lut_n; i += kBinThreads)
                    s_lut[fp.sp[s].lut_off + i] = fp.lut[s * kMaxLut + i];
    }
    __syncthreads();
    const unsigned long long lo = (unsigned long long)blockIdx.x * per;
    const unsigned int len = lo < n ? (unsigned int)min(n - lo, per) : 0u;
    const unsigned int lo32 = (unsigned int)lo;
    x += lo; y += lo; z += lo; h += lo; I += lo; scalar += lo;
    // species of the block's first and last particle: most blocks lie inside one species
    const int s_first = species_of(lo32, fp), s_last = species_of(lo32 + (len ? len - 1 : 0), fp);
    float amax = 0.0f;
    const bool one_species = s_first == s_last;
    const int ts = fp.tshift, tmask = fp.T - 1;
    const unsigned int lane4 = 4u * (threadIdx.x & 31u);
    for (unsigned int iw = 4u * (threadIdx.x & ~31u); iw < len; iw += 4u * kBinThreads) {
        const unsigned int i = iw + lane4;
        float xs[4], ys[4], zs[4], hs[4], Is[4], ss[4];
        load4<ALIGNED>(x, i, len, xs);
        load4<ALIGNED>(y, i, len, ys);
        load4<ALIGNED>(z, i, len, zs);
        load4<ALIGNED>(h, i, len, hs);
        load4<ALIGNED>(I, i, len, Is);
        load4<ALIGNED>(scalar, i, len, ss);
        float vr[4] = {0.f, 0.f, 0.f, 0.f}, vg[4] = {0.f, 0.f, 0.f, 0.f}, vb[4] = {0.f, 0.f, 0.f, 0.f};
        if (fp.any_vector) {
            load4<false>(fp.vec[0] + lo, i, len, vr);
            load4<false>(fp.vec[1] + lo, i, len, vg);
            load4<false>(fp.vec[2] + lo, i, len, vb);
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const Geo g = geometry(xs[j], ys[j], zs[j], hs[j], fp);
            const int cls = (i + j < len) ? g.cls : CULLED;
            const int s = one_species ? s_first : species_of(min(lo32 + i + j, lo32 + len - 1), fp);
            const SpeciesDev &S = fp.sp[s];
            const float4 *lut = fp.lut_total > 0 ? s_lut + S.lut_off : fp.lut + s * kMaxLut;
            float3 a = amplitude(Is[j], ss[j], hs[j], S, lut, s_rng[s], make_float3(vr[j], vg[j], vb[j]));
            const bool small = cls == SMALL;
            const float sp2 = __fmul_rn(g.sp, g.sp);
            const float wsm = small ? fp.csmall * sp2 : 1.0f;
            a.x *= wsm; a.y *= wsm; a.z *= wsm;
            const float am = fmaxf(fabsf(a.x), fmaxf(fabsf(a.y), fabsf(a.z)));
            if (!(am <= 3.0e38f)) a = make_float3(0.0f, 0.0f, 0.0f);             // Inf / NaN amplitude
            else if (cls != CULLED) amax = fmaxf(amax, am);
            const BinWalk w = bin_walk<BTILE>(g, cls, fp);
            if (small) {
                if (BTILE) {       // the paper's scheme: SMALL particles go straight to the small-particle partial image
                    float *o = fp.btile_planes + 4 * (3 * (size_t)fp.W * fp.H) + 3 * ((size_t)g.y0 * fp.W + g.x0);
                    asm volatile("red.global.add.f32 [%0], %1;" :: "l"(o), "f"(a.x) : "memory");
                    asm volatile("red.global.add.f32 [%0], %1;" :: "l"(o + 1), "f"(a.y) : "memory");
                    asm volatile("red.global.add.f32 [%0], %1;" :: "l"(o + 2), "f"(a.z) : "memory");
                } else {
                    const unsigned int pix = (unsigned int)(((g.y0 & tmask) << ts) | (g.x0 & tmask));
                    const unsigned int u = cursor_take<GHIST>(cursor + (2 * (w.by0 * fp.ntx + w.bx0) + 1), 1u);
                    asm volatile("st.global.v4.f32 [%0], {%1,%2,%3,%4};" :: "l"(records + u), "f"(__uint_as_float(pix)), "f"(a.x), "f"(a.y), "f"(a.z) : "memory");
                }
            }
            // MEDIUM and LARGE: one 32-byte record per bin of the box.  Boxes wider than 2 x 2 bins are walked by the whole warp
            // (coop_bin_walk), the record travelling from its lane by shuffles
            const int nrec = (cls == MEDIUM || cls == LARGE) ? w.n : 0;
            if (__any_sync(0xffffffffu, nrec > 0)) {
                const float4 ra = make_float4(g.px, g.py, __fdividef(-1.4426950408889634f, sp2), __fmul_rn(g.rp, g.rp));
                // boxes inside 2 x 2 bins (nearly all, outside cfg3): their lane writes the records, one warp-uniform loop of at most four steps
                const bool wide = nrec > 0 && (w.bx1 - w.bx0 > 1 || w.by1 - w.by0 > 1);
                const int nown = wide ? 0 : nrec;
                const int nmax = __reduce_max_sync(0xffffffffu, nown);
                int bx = w.bx0, by = w.by0;
#pragma unroll 1
                for (int t = 0; t < nmax; ++t) {
                    if (t < nown) {
                        unsigned int box;
                        if (BTILE && cls == MEDIUM) {      // box relative to the home tile's Btile (body + boundary of r_0)
                            const int ox = (bx << ts) - fp.btile_r0, oy = (by << ts) - fp.btile_r0;
                            box = (unsigned int)(g.x0 - ox) | ((unsigned int)(g.y0 - oy) << 6) | ((unsigned int)(g.x1 - g.x0) << 12) | ((unsigned int)(g.y1 - g.y0) << 18);
                        } else {
                            box = pack_box(g, bx, by, w.sh, w.route != 0);
                        }
                        st_record(records, cursor_take<GHIST>(cursor + (w.base + w.mult * (by * w.pitch + bx)), 2u), ra,
                                  make_float4(a.x, a.y, a.z, __uint_as_float(box)));
                    }
                    const bool wrap = bx == w.bx1;
                    bx = wrap ? w.bx0 : bx + 1;
                    by += wrap;
                }
                if (__any_sync(0xffffffffu, wide)) {
                    const unsigned int xx = (unsigned int)g.x0 | ((unsigned int)g.x1 << 16), yy = (unsigned int)g.y0 | ((unsigned int)g.y1 << 16);
                    coop_bin_walk(wide, w, (int)(threadIdx.x & 31u), [&](bool ok, int sl, int bx, int by, int route) {
                        const float4 sa = make_float4(__shfl_sync(0xffffffffu, ra.x, sl), __shfl_sync(0xffffffffu, ra.y, sl),
                                                      __shfl_sync(0xffffffffu, ra.z, sl), __shfl_sync(0xffffffffu, ra.w, sl));
                        const float s_r = __shfl_sync(0xffffffffu, a.x, sl), s_g = __shfl_sync(0xffffffffu, a.y, sl), s_b = __shfl_sync(0xffffffffu, a.z, sl);
                        const unsigned int sxx = __shfl_sync(0xffffffffu, xx, sl), syy = __shfl_sync(0xffffffffu, yy, sl);
                        if (ok) {
                            Geo sg;
                            sg.x0 = (int)(sxx & 0xffffu); sg.x1 = (int)(sxx >> 16); sg.y0 = (int)(syy & 0xffffu); sg.y1 = (int)(syy >> 16);
                            const unsigned int box = pack_box(sg, bx, by, route == 1 ? fp.sshift : fp.tshift, route != 0);
                            st_record(records, cursor_take<GHIST>(cursor + routed_bin(route, bx, by, fp), 2u), sa, make_float4(s_r, s_g, s_b, __uint_as_float(box)));
                        }
                    });
                }
            }
        }
    }
    // largest record amplitude of the frame: fixes the fixed-point scale of k_splat and k_large
    amax = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(amax)));   // amax >= 0: bit order = value order
    if ((threadIdx.x & 31) == 0) s_amax[threadIdx.x >> 5] = amax;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < kBinThreads / 32; ++w) amax = fmaxf(amax, s_amax[w]);
        if (amax > 0.0f) atomicMax(&stats->amax_bits, __float_as_uint(amax));
    }
}

// ---- A5: tile renderer for SMALL + MEDIUM records -------------------------------------------------------------
__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float pow2i(int e) { return __int_as_float((e + 127) << 23); }   // -126 <= e <= 127

// Fixed-point exponent of the frame: contributions are accumulated in units of 2^-e, with the largest record
// amplitude in [2^(kFixedBits-1), 2^kFixedBits).  Integer sums are exact and independent of the summation order.
__device__ __forceinline__ int fixed_exponent(unsigned int amax_bits)
{
    if (amax_bits == 0u) return 0;
    int ex = (int)(amax_bits >> 23) - 126;              // amax = m 2^ex, m in [0.5, 1) (subnormals: ex = -126, fine)
    return kFixedBits - ex;
}

__global__ void __launch_bounds__(256)
k_rescale(long long *__restrict__ accum, size_t n, const DeviceStats *__restrict__ stats)
{
    const int e_new = fixed_exponent(stats->amax_bits);
    const int sh = stats->accum_exp_set ? stats->accum_exp - e_new : 0;     // > 0: the unit grew by 2^sh
    if (sh <= 0) return;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const long long v = accum[i];
        accum[i] = sh >= 63 ? 0ll : (v + (1ll << (sh - 1))) >> sh;
    }
}

__global__ void k_rescale_done(DeviceStats *stats)
{
    stats->accum_exp = fixed_exponent(stats->amax_bits);
    stats->accum_exp_set = 1u;
}

// ---- packed float32 pairs (Blackwell FADD2 / FMUL2 / FFMA2: two IEEE round-to-nearest results per issue slot) ----
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk2(f32x2 v, float &a, float &b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f32x2 fadd2(f32x2 a, f32x2 b) { f32x2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fmul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 ffma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
// c += a * b with the sum pinned to its register pair (a separate result register made ptxas copy 24 accumulator registers per record)
__device__ __forceinline__ void ffma2_acc(f32x2 &c, f32x2 a, f32x2 b) { asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(c) : "l"(a), "l"(b)); }

// Framebuffer of a tile in shared memory, fixed point: per channel a low plane (sums of the low 16 bits of each
// contribution, unsigned) and a high plane (sums of the signed upper bits).  value = hi * 65536 + lo, in units of
// 2^-e.  A segment holds at most kChunkMax = 32768 records and a record touches a pixel once, so neither plane can
// wrap.  Updates are native 32-bit shared-memory atomics without a return value (64-bit and float atomics on shared
// memory are CAS loops on sm_100).  Integer sums are exact and independent of the order.
__device__ __forceinline__ void fixed_add(unsigned int *lo, unsigned int *hi, float value)
{
    const int v = __float2int_rn(value);                // |v| <= 2^kFixedBits
    const int up = v >> 16;
    const unsigned int alo = (unsigned int)__cvta_generic_to_shared(lo), ahi = (unsigned int)__cvta_generic_to_shared(hi);
    asm volatile("{\n\t.reg .pred p;\n\tred.shared.add.u32 [%0], %2;\n\tsetp.ne.s32 p, %3, 0;\n\t@p red.shared.add.u32 [%1], %3;\n\t}"
                 :: "r"(alo), "r"(ahi), "r"((unsigned int)v & 0xffffu), "r"(up) : "memory");
}

// Geometry of the tile renderer: a warp owns a strip of the tile (8 x 8 pixels; 64 x 4 for T = 64; a box of 3 x 3 pixels straddles
// fewer square strips than 16 x 4 ones: cfg2 k_splat 2.50 -> 2.34 ms), a
// lane owns kNP pairs of horizontally adjacent pixels of it and keeps their RGB sums in registers as packed pairs.
template <int T> struct SplatCfg {
    static constexpr int kPix = T * T;
    static constexpr int kNP = T == 64 ? 4 : 1;          // pixel pairs per lane
    static constexpr int kSW = T == 64 ? 64 : 8;                     // strip width
    static constexpr int kSH = 64 * kNP / kSW;           // strip height
    static constexpr int kStripsX = T / kSW, kStripsY = T / kSH;
    static constexpr int kWarps = kStripsX * kStripsY;   // 1, 4, 16, 16 for T = 8, 16, 32, 64
    static constexpr int kThreads = 32 * kWarps;         // one record per thread and batch
    static constexpr int kFoldBatches = 1024 / kThreads > 0 ? 1024 / kThreads : 1;   // fold the sub-sums every ~1024 records
};

// k_splat itself lives in splotch_splat.cuh.

// ---- A8: epilogue -------------------------------------------------------------------------------------------------
// One CTA per tile: the tile's 64-bit fixed-point sums (fed by k_splat and k_large) become the float32 image, S or
// 1 - exp(-S) (the exact E = A solution); every pixel is written exactly once (:216-219, :238).
template <int T>
__global__ void __launch_bounds__(256)
k_compose(const unsigned long long *__restrict__ accum, const DeviceStats *__restrict__ stats,
          const __grid_constant__ FrameParams fp, float *__restrict__ image)
{
    constexpr int kPix = T * T;
    const int tile = blockIdx.x;
    const int tx0 = (tile % fp.ntx) * T, ty0 = (tile / fp.ntx) * T;
    const bool ok = stats->f_overflow == 0u;
    const double unit = ldexp(1.0, -fixed_exponent(stats->amax_bits));       // one fixed-point unit
    for (int p = threadIdx.x; p < kPix; p += 256) {
        const int ix = tx0 + p % T, iy = ty0 + p / T;
        if (ix < fp.W && iy < fp.H) {
            const unsigned long long *q = accum + (size_t)tile * (3 * kPix) + p;
            float *o = image + 3ull * ((size_t)iy * fp.W + ix);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float v = ok ? (float)((double)(long long)__ldg(q + c * kPix) * unit) : 0.0f;
                o[c] = fp.apply_transfer ? -expm1f(-v) : v;
            }
        }
    }
}

// ---- A8 for a particle-sharded frame: the shards' fixed-point tile sums -> the image, in one kernel ------------------------------
// Every shard (a GPU of a multi-GPU frame, or a part of the set rendered into its own workspace) leaves exact
// 64-bit sums in units of its own 2^-e.  The sum over the shards is taken per pixel in double precision (integers times powers of
// two: exact up to 2^53 units), so the result does not depend on the order of the shards; the pointers may be peer-mapped device
// memory of other GPUs (loads over NVLink), which fuses the image reduction of the sharded frame into the epilogue: no float
// partial images, no separate all-reduce.  Tiles [tile0, tile1): a rank may compose its share of the image only.
constexpr int kMaxShards = 16;
struct ShardPtrs {
    const unsigned long long *accum[kMaxShards];
    const DeviceStats *stats[kMaxShards];
    int n;
};

template <int T>
__global__ void __launch_bounds__(256)
k_compose_shards(const __grid_constant__ ShardPtrs sh, const __grid_constant__ FrameParams fp, int tile0, int apply_transfer,
                 float *__restrict__ image)
{
    constexpr int kPix = T * T;
    __shared__ double s_unit[kMaxShards];
    __shared__ int s_ok;
    if (threadIdx.x == 0) {
        int ok = 1;
        for (int k = 0; k < sh.n; ++k) {
            ok &= sh.stats[k]->f_overflow == 0u;
            s_unit[k] = ldexp(1.0, -fixed_exponent(sh.stats[k]->amax_bits));
        }
        s_ok = ok;
    }
    __syncthreads();
    const int tile = tile0 + blockIdx.x;
    const int tx0 = (tile % fp.ntx) * T, ty0 = (tile / fp.ntx) * T;
    for (int p = threadIdx.x; p < kPix; p += 256) {
        const int ix = tx0 + p % T, iy = ty0 + p / T;
        if (ix < fp.W && iy < fp.H) {
            float *o = image + 3ull * ((size_t)iy * fp.W + ix);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double v = 0.0;
                for (int k = 0; k < sh.n; ++k) v += (double)(long long)__ldg(sh.accum[k] + (size_t)tile * (3 * kPix) + c * kPix + p) * s_unit[k];
                const float f = s_ok ? (float)v : 0.0f;
                o[c] = apply_transfer ? -expm1f(-f) : f;
            }
        }
    }
}

// ---- 1 - exp(-S) on a finished image: the transfer of a frame whose partial images were summed elsewhere (multi-GPU) ----
__global__ void __launch_bounds__(256)
k_apply_transfer(float *__restrict__ image, size_t n)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) image[i] = -expm1f(-image[i]);
}

// ---- test hook: per-tile pair counts (SMALL + MEDIUM bins of every tile) ---------------------------------------------
__global__ void __launch_bounds__(256)
k_tile_counts(const unsigned int *__restrict__ bin_count, int n_tiles, int n_super, int n_big, unsigned int *__restrict__ out)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n_tiles) out[t] = bin_count[2 * t] + bin_count[2 * t + 1] + (n_big ? bin_count[2 * n_tiles + n_super + t] : 0u);
}

// ---- test hook: per-particle classification results -----------------------------------------------------------
__global__ void __launch_bounds__(256)
k_debug_geometry(const float *__restrict__ x, const float *__restrict__ y, const float *__restrict__ z,
                 const float *__restrict__ h, unsigned long long n, const __grid_constant__ FrameParams fp, int8_t *cls, float *px, float *py,
                 float *sp, float *rp, float *zc, int4 *pbox, int4 *tbox, int *ilabel)
{
    const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const Geo g = geometry(x[i], y[i], z[i], h[i], fp);
    if (cls) cls[i] = (int8_t)g.cls;
    if (px) px[i] = g.px;
    if (py) py[i] = g.py;
    if (sp) sp[i] = g.sp;
    if (rp) rp[i] = g.rp;
    if (zc) zc[i] = g.zc;
    if (pbox) pbox[i] = make_int4(g.x0, g.x1, g.y0, g.y1);
    if (tbox) {
        if (g.cls == CULLED) tbox[i] = make_int4(0, -1, 0, -1);
        else tbox[i] = make_int4(g.x0 >> fp.tshift, g.x1 >> fp.tshift, g.y0 >> fp.tshift, g.y1 >> fp.tshift);
    }
    if (ilabel) ilabel[i] = paper_label(g, fp);
}

}  // namespace splotch
