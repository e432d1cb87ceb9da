// splotch_kernels.cuh -- device code of the B200-native Splotch rendering path (sm_100a).
//
// Stage map (paper passages in PAPER.md):
//   k_count    A1+A3+A4a  roto-translate, project, classify (:76, :138, :156-173) and count (particle, bin) pairs
//   k_colscan  A4b        per-bin exclusive scan over the count matrix rows (replaces thrust::reduce_by_key, :203)
//   k_binscan  A4c        exclusive scan over bins, chunk table, frame statistics (replaces inclusive_scan, :205)
//   k_scatter  A1-A3+A2+A4d  recompute geometry, colourise (:76, :85), write render records in bin order
//                            (replaces copy_if + sort_by_key, :196-202)
//   k_splat    A5         small + medium particles of one chunk of one tile into warp-private shared-memory
//                         framebuffers (the paper's medium-particle kernel, :183, :224-228, without its halo copies)
//   k_compose  A6+A8      per tile: sum chunk partials, gather the LARGE particles of the tile's super-tile
//                         (the paper renders these on the CPU, :232-238), optional 1-exp(-S), write the image
//
// Canonical float32 geometry: every operation that decides an integer (class, pixel box, tile box, the inside
// test) is written with round-to-nearest intrinsics (__fmul_rn, __fmaf_rn, __fdiv_rn ...) which nvcc never
// contracts or reorders, so the values equal those of any IEEE-754 binary32 implementation of the same sequence.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace splotch {

constexpr int kMaxSpecies   = 8;
constexpr int kMaxLut       = 1024;
constexpr int kChunk        = 4096;   // records per work item of k_splat
constexpr int kSplatWarps   = 8;
constexpr int kBinThreads   = 512;    // k_count / k_scatter block size
constexpr int kSuperShift   = 3;      // super-tile = 8 x 8 tiles (LARGE particles are binned to super-tiles)

enum { CULLED = 0, SMALL = 1, MEDIUM = 2, LARGE = 3 };

struct SpeciesDev {
    float brightness, absorb;
    float fixed_r, fixed_g, fixed_b;
    float smin, range;
    int   use_colormap, use_log10, lut_n, pad;
};

struct FrameParams {
    float cam[16];               // r[3] u[3] f[3] eye[3] s cx cy 0
    float chi, r_small, r_large, z_near;
    float fW, fH;
    float csmall;                // pi (1 - exp(-chi^2)): flux of the clipped unit Gaussian per sigma_px^2
    int   W, H, T, tshift;
    int   ntx, nty, n_tiles;
    int   sshift, nsx, nsy, n_super, nbins;
    int   additive, apply_transfer;
    int   n_species;
    unsigned long long sp_begin[kMaxSpecies + 1];
    SpeciesDev sp[kMaxSpecies];
    const float4 *lut;           // [kMaxSpecies][kMaxLut] rgb0
};

struct DeviceStats {             // written by k_binscan, read back by splotch_get_stats
    unsigned long long count[4];
    unsigned long long pairs, large_pairs, chunks, capacity;
    unsigned int overflow, work_counter, pad0, pad1;
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

// C1 of DESIGN.md: the canonical float32 sequence (PAPER.md:76 projection, Eq. 7 :138 radius, :156-160 classes).
__device__ __forceinline__ Geo geometry(float x, float y, float z, float h, const FrameParams &fp)
{
    Geo g;
    const float dx = __fsub_rn(x, fp.cam[9]), dy = __fsub_rn(y, fp.cam[10]), dz = __fsub_rn(z, fp.cam[11]);
    const float xc = dot3(fp.cam + 0, dx, dy, dz);
    const float yc = dot3(fp.cam + 3, dx, dy, dz);
    g.zc = dot3(fp.cam + 6, dx, dy, dz);
    g.cls = CULLED;
    g.px = g.py = g.sp = g.rp = 0.0f;
    g.x0 = g.y0 = 0;
    g.x1 = g.y1 = -1;
    if (g.zc > fp.z_near) {
        const float k = __fdiv_rn(fp.cam[12], g.zc);
        g.px = __fmaf_rn(xc, k, fp.cam[13]);
        g.py = __fmaf_rn(-yc, k, fp.cam[14]);
        g.sp = __fmul_rn(h, k);
        g.rp = __fmul_rn(fp.chi, g.sp);
        if (g.rp >= 0.0f && g.rp <= 3.0e38f) {
            if (g.rp <= fp.r_small) {
                if (g.px >= 0.0f && g.px < fp.fW && g.py >= 0.0f && g.py < fp.fH) {
                    g.cls = SMALL;
                    g.x0 = g.x1 = (int)floorf(g.px);
                    g.y0 = g.y1 = (int)floorf(g.py);
                }
            } else {
                const float fx0 = fmaxf(ceilf(__fsub_rn(__fsub_rn(g.px, g.rp), 0.5f)), 0.0f);
                const float fx1 = fmaxf(fminf(floorf(__fsub_rn(__fadd_rn(g.px, g.rp), 0.5f)), __fsub_rn(fp.fW, 1.0f)), -1.0f);
                const float fy0 = fmaxf(ceilf(__fsub_rn(__fsub_rn(g.py, g.rp), 0.5f)), 0.0f);
                const float fy1 = fmaxf(fminf(floorf(__fsub_rn(__fadd_rn(g.py, g.rp), 0.5f)), __fsub_rn(fp.fH, 1.0f)), -1.0f);
                if (fx0 <= fx1 && fy0 <= fy1) {
                    g.cls = (g.rp <= fp.r_large) ? MEDIUM : LARGE;
                    g.x0 = (int)fx0; g.x1 = (int)fx1;
                    g.y0 = (int)fy0; g.y1 = (int)fy1;
                }
            }
        }
    }
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

// Visit every bin a particle is assigned to: its tile (SMALL), the tiles of its pixel box (MEDIUM) or the
// super-tiles of its pixel box (LARGE, bins n_tiles ...).  k_count and k_scatter share this traversal.
template <class F>
__device__ __forceinline__ void for_each_bin(const Geo &g, const FrameParams &fp, F &&f)
{
    if (g.cls == CULLED) return;
    if (g.cls == LARGE) {
        const int sx0 = g.x0 >> fp.sshift, sx1 = g.x1 >> fp.sshift;
        const int sy0 = g.y0 >> fp.sshift, sy1 = g.y1 >> fp.sshift;
        for (int sy = sy0; sy <= sy1; ++sy)
            for (int sx = sx0; sx <= sx1; ++sx) f(fp.n_tiles + sy * fp.nsx + sx);
        return;
    }
    const int tx0 = g.x0 >> fp.tshift, tx1 = g.x1 >> fp.tshift;
    const int ty0 = g.y0 >> fp.tshift, ty1 = g.y1 >> fp.tshift;
    for (int ty = ty0; ty <= ty1; ++ty)
        for (int tx = tx0; tx <= tx1; ++tx) f(ty * fp.ntx + tx);
}

// ---- streaming loads: four consecutive particles of one field ------------------------------------------------
__device__ __forceinline__ float4 ldg_stream4(const float *p)
{
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

template <bool ALIGNED>
__device__ __forceinline__ void load4(const float *__restrict__ a, unsigned long long i, unsigned long long hi, float (&v)[4])
{
    if (ALIGNED && i + 4 <= hi) {
        const float4 q = ldg_stream4(a + i);
        v[0] = q.x; v[1] = q.y; v[2] = q.z; v[3] = q.w;
    } else {
#pragma unroll
        for (int j = 0; j < 4; ++j) v[j] = (i + j < hi) ? __ldg(a + i + j) : 0.0f;
    }
}

__device__ __forceinline__ unsigned int warp_sum(unsigned int v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// ---- A1 + A3 + A4a: classify and count ------------------------------------------------------------------------
// Block b owns the particle range [b*per, (b+1)*per) and a private histogram over all bins in shared memory;
// row b of `counts` receives it, so the count stage needs no global atomics and is deterministic.
template <bool ALIGNED>
__global__ void __launch_bounds__(kBinThreads)
k_count(const float *__restrict__ x, const float *__restrict__ y, const float *__restrict__ z,
        const float *__restrict__ h, unsigned long long n, unsigned long long per, const __grid_constant__ FrameParams fp,
        unsigned int *__restrict__ counts, unsigned int *__restrict__ cls_counts)
{
    extern __shared__ unsigned int hist[];
    __shared__ unsigned int s_cls[4];
    for (int i = threadIdx.x; i < fp.nbins; i += blockDim.x) hist[i] = 0u;
    if (threadIdx.x < 4) s_cls[threadIdx.x] = 0u;
    __syncthreads();
    const unsigned long long lo = (unsigned long long)blockIdx.x * per;
    const unsigned long long hi = min(n, lo + per);
    unsigned int c1 = 0, c2 = 0, c3 = 0, call = 0;
    for (unsigned long long i = lo + 4ull * threadIdx.x; i < hi; i += 4ull * blockDim.x) {
        float xs[4], ys[4], zs[4], hs[4];
        load4<ALIGNED>(x, i, hi, xs);
        load4<ALIGNED>(y, i, hi, ys);
        load4<ALIGNED>(z, i, hi, zs);
        load4<ALIGNED>(h, i, hi, hs);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (i + j < hi) {
                const Geo g = geometry(xs[j], ys[j], zs[j], hs[j], fp);
                ++call;
                c1 += (g.cls == SMALL); c2 += (g.cls == MEDIUM); c3 += (g.cls == LARGE);
                for_each_bin(g, fp, [&](int bin) { atomicAdd(&hist[bin], 1u); });
            }
        }
    }
    c1 = warp_sum(c1); c2 = warp_sum(c2); c3 = warp_sum(c3); call = warp_sum(call);
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&s_cls[0], call - c1 - c2 - c3);
        atomicAdd(&s_cls[1], c1); atomicAdd(&s_cls[2], c2); atomicAdd(&s_cls[3], c3);
    }
    __syncthreads();
    unsigned int *row = counts + (size_t)blockIdx.x * fp.nbins;
    for (int i = threadIdx.x; i < fp.nbins; i += blockDim.x) row[i] = hist[i];
    if (threadIdx.x < 4) cls_counts[blockIdx.x * 4 + threadIdx.x] = s_cls[threadIdx.x];
}

// ---- A4b: per bin, exclusive scan down the rows of the count matrix -----------------------------------------
__global__ void __launch_bounds__(256)
k_colscan(unsigned int *__restrict__ counts, int nrows, int nbins, unsigned int *__restrict__ bin_count)
{
    const int bin = blockIdx.x * blockDim.x + threadIdx.x;
    if (bin >= nbins) return;
    unsigned int run = 0;
    int b = 0;
    for (; b + 8 <= nrows; b += 8) {
        unsigned int c[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) c[k] = counts[(size_t)(b + k) * nbins + bin];
#pragma unroll
        for (int k = 0; k < 8; ++k) { counts[(size_t)(b + k) * nbins + bin] = run; run += c[k]; }
    }
    for (; b < nrows; ++b) {
        const unsigned int c = counts[(size_t)b * nbins + bin];
        counts[(size_t)b * nbins + bin] = run;
        run += c;
    }
    bin_count[bin] = run;
}

// ---- A4c: scan over bins, chunk table, statistics (one block) ------------------------------------------------
__device__ __forceinline__ unsigned long long block_excl_scan_1024(unsigned long long v, unsigned long long *s_warp,
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
    if (w == 0) {
        unsigned long long ws = s_warp[lane], winc = ws;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long t = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += t;
        }
        s_warp[lane] = winc - ws;
        if (lane == 31) *total = winc;
    }
    __syncthreads();
    const unsigned long long r = s_warp[w] + inc - v;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(1024)
k_binscan(const unsigned int *__restrict__ bin_count, int n_tiles, int nbins, unsigned int *__restrict__ bin_start,
          unsigned int *__restrict__ chunk_start, uint2 *__restrict__ chunk_desc,
          const unsigned int *__restrict__ cls_counts, int nrows, unsigned long long capacity,
          unsigned long long max_chunks, DeviceStats *__restrict__ stats)
{
    __shared__ unsigned long long s_warp[32];
    __shared__ unsigned long long s_tot_pairs, s_tot_all, s_tot_chunks;
    const int per = (nbins + 1023) / 1024;
    const int b0 = min(nbins, (int)threadIdx.x * per), b1 = min(nbins, b0 + per);
    unsigned long long sum_all = 0, sum_tiles = 0, sum_chunks = 0;
    for (int b = b0; b < b1; ++b) {
        const unsigned int c = bin_count[b];
        sum_all += c;
        if (b < n_tiles) { sum_tiles += c; sum_chunks += (c + kChunk - 1) / kChunk; }
    }
    const unsigned long long off_all = block_excl_scan_1024(sum_all, s_warp, &s_tot_all);
    const unsigned long long off_chunks = block_excl_scan_1024(sum_chunks, s_warp, &s_tot_chunks);
    (void)block_excl_scan_1024(sum_tiles, s_warp, &s_tot_pairs);
    const bool overflow = s_tot_all > capacity || s_tot_chunks > max_chunks;
    unsigned long long run = off_all, crun = off_chunks;
    for (int b = b0; b < b1; ++b) {
        const unsigned int c = bin_count[b];
        bin_start[b] = (unsigned int)run;
        if (b < n_tiles) {
            chunk_start[b] = (unsigned int)crun;
            const unsigned int nc = (c + kChunk - 1) / kChunk;
            if (!overflow)
                for (unsigned int k = 0; k < nc; ++k) chunk_desc[crun + k] = make_uint2((unsigned int)b, k);
            crun += nc;
        }
        run += c;
    }
    if (threadIdx.x == 1023) {
        bin_start[nbins] = (unsigned int)s_tot_all;
        chunk_start[n_tiles] = (unsigned int)s_tot_chunks;
    }
    if (threadIdx.x < 4) {
        unsigned long long c = 0;
        for (int r = 0; r < nrows; ++r) c += cls_counts[r * 4 + threadIdx.x];
        stats->count[threadIdx.x] = c;
    }
    if (threadIdx.x == 0) {
        stats->pairs = s_tot_pairs;
        stats->large_pairs = s_tot_all - s_tot_pairs;
        stats->chunks = overflow ? 0ull : s_tot_chunks;
        stats->capacity = capacity;
        stats->overflow = overflow ? 1u : 0u;
        stats->work_counter = 0u;
    }
}

// ---- A2: colour + amplitude (PAPER.md:76 normalisation/log, :85 look-up table) -------------------------------
__device__ __forceinline__ int species_of(unsigned long long i, const FrameParams &fp)
{
    int s = 0;
#pragma unroll
    for (int k = 1; k < kMaxSpecies; ++k) s += (k < fp.n_species && i >= fp.sp_begin[k]);
    return s;
}

__device__ __forceinline__ float3 amplitude(float I, float scalar, float h, int s, const FrameParams &fp)
{
    const SpeciesDev &S = fp.sp[s];
    float r = S.fixed_r, g = S.fixed_g, b = S.fixed_b;
    if (S.use_colormap) {
        float v = scalar;
        if (S.use_log10) v = log10f(v);
        float t = (v - S.smin) / S.range;
        t = (t > 0.0f) ? t : 0.0f;                 // NaN clamps to 0
        t = fminf(t, 1.0f);
        const float u = t * (float)(S.lut_n - 1);
        const int i0 = min((int)floorf(u), S.lut_n - 2);
        const float fr = u - (float)i0;
        const float4 a = __ldg(fp.lut + s * kMaxLut + i0);
        const float4 c = __ldg(fp.lut + s * kMaxLut + i0 + 1);
        r = fmaf(fr, c.x - a.x, a.x);
        g = fmaf(fr, c.y - a.y, a.y);
        b = fmaf(fr, c.z - a.z, a.z);
    }
    const float col = S.brightness * (1.7724538509055160273f * h * I);   // b_s * sqrt(pi) h I
    return make_float3(r * col, g * col, b * col);
}

// Render record, 32 bytes: {px, py, c = -log2(e)/sp^2, rp | -1 for SMALL} {aR, aG, aB, zc}
// MEDIUM / LARGE: a = E * col.   SMALL: a = E * col * pi sp^2 (1 - exp(-chi^2)) (the whole clipped flux).
__device__ __forceinline__ void st_record(float4 *rec, unsigned int slot, float4 a, float4 b)
{
    rec[2ull * slot] = a;
    rec[2ull * slot + 1] = b;
}

template <bool ALIGNED>
__global__ void __launch_bounds__(kBinThreads)
k_scatter(const float *__restrict__ x, const float *__restrict__ y, const float *__restrict__ z,
          const float *__restrict__ h, const float *__restrict__ I, const float *__restrict__ scalar,
          unsigned long long n, unsigned long long per, const __grid_constant__ FrameParams fp,
          const unsigned int *__restrict__ counts, const unsigned int *__restrict__ bin_start,
          const DeviceStats *__restrict__ stats, float4 *__restrict__ records)
{
    extern __shared__ unsigned int cursor[];
    if (stats->overflow) return;
    const unsigned int *row = counts + (size_t)blockIdx.x * fp.nbins;
    for (int i = threadIdx.x; i < fp.nbins; i += blockDim.x) cursor[i] = bin_start[i] + row[i];
    __syncthreads();
    const unsigned long long lo = (unsigned long long)blockIdx.x * per;
    const unsigned long long hi = min(n, lo + per);
    for (unsigned long long i = lo + 4ull * threadIdx.x; i < hi; i += 4ull * blockDim.x) {
        float xs[4], ys[4], zs[4], hs[4], Is[4], ss[4];
        load4<ALIGNED>(x, i, hi, xs);
        load4<ALIGNED>(y, i, hi, ys);
        load4<ALIGNED>(z, i, hi, zs);
        load4<ALIGNED>(h, i, hi, hs);
        load4<ALIGNED>(I, i, hi, Is);
        load4<ALIGNED>(scalar, i, hi, ss);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (i + j < hi) {
                const Geo g = geometry(xs[j], ys[j], zs[j], hs[j], fp);
                if (g.cls != CULLED) {
                    float3 a = amplitude(Is[j], ss[j], hs[j], species_of(i + j, fp), fp);
                    float4 ra, rb;
                    ra.x = g.px; ra.y = g.py;
                    if (g.cls == SMALL) {
                        const float w = fp.csmall * (g.sp * g.sp);
                        a.x *= w; a.y *= w; a.z *= w;
                        ra.z = 0.0f; ra.w = -1.0f;
                    } else {
                        ra.z = __fdiv_rn(-1.4426950408889634f, __fmul_rn(g.sp, g.sp));
                        ra.w = g.rp;
                    }
                    rb = make_float4(a.x, a.y, a.z, g.zc);
                    for_each_bin(g, fp, [&](int bin) {
                        const unsigned int slot = atomicAdd(&cursor[bin], 1u);
                        st_record(records, slot, ra, rb);
                    });
                }
            }
        }
    }
}

// ---- A5: tile renderer for SMALL + MEDIUM records -------------------------------------------------------------
__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int T> struct SplatCfg {
    static constexpr int kStride = T + 3;                       // float4 per framebuffer row (bank spreading)
    static constexpr int kFbElems = T * kStride;                // float4 per warp-private framebuffer
    static constexpr int kWarps = (T == 32) ? 4 : kSplatWarps;
    static constexpr size_t kSmemBytes = sizeof(float4) * (size_t)kFbElems * kWarps;
};

// One work item = up to kChunk consecutive records of one tile.  Every warp owns a private T x T RGB
// framebuffer in shared memory and walks its share of the records: SMALL records are deposited one lane per
// particle (lanes that hit the same pixel take turns), MEDIUM records one particle at a time with the lanes
// spread over the pixels of its box, so there is never a concurrent update of one pixel and no atomics.
// The warps' framebuffers are summed into the chunk's partial tile.
template <int T>
__global__ void __launch_bounds__(SplatCfg<T>::kWarps * 32)
k_splat(const float4 *__restrict__ records, const unsigned int *__restrict__ bin_start,
        const uint2 *__restrict__ chunk_desc, DeviceStats *__restrict__ stats, float4 *__restrict__ partials,
        const __grid_constant__ FrameParams fp)
{
    using Cfg = SplatCfg<T>;
    constexpr int kStride = Cfg::kStride, kWarps = Cfg::kWarps, kThreads = kWarps * 32;
    extern __shared__ float4 fb_all[];
    __shared__ unsigned int s_chunk;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float4 *fb = fb_all + warp * Cfg::kFbElems;
    const unsigned int total = (unsigned int)stats->chunks;
    for (;;) {
        if (threadIdx.x == 0) s_chunk = atomicAdd(&stats->work_counter, 1u);
        for (int i = threadIdx.x; i < Cfg::kFbElems * kWarps; i += kThreads) fb_all[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        __syncthreads();
        const unsigned int chunk = s_chunk;
        if (chunk >= total) break;
        const uint2 d = chunk_desc[chunk];
        const int tile = (int)d.x;
        const unsigned int begin = bin_start[tile] + d.y * kChunk;
        const unsigned int end = min(begin + (unsigned int)kChunk, bin_start[tile + 1]);
        const int tx0 = (tile % fp.ntx) * T, ty0 = (tile / fp.ntx) * T;
        const float ftx0 = (float)tx0, fty0 = (float)ty0;
        const float ftx1 = (float)min(tx0 + T - 1, fp.W - 1), fty1 = (float)min(ty0 + T - 1, fp.H - 1);
        for (unsigned int base = begin + warp * 32; base < end; base += kThreads) {
            const unsigned int idx = base + lane;
            const bool valid = idx < end;
            float4 ra = make_float4(0.f, 0.f, 0.f, 0.f), rb = ra;
            if (valid) { ra = __ldg(records + 2ull * idx); rb = __ldg(records + 2ull * idx + 1); }
            const bool is_small = valid && ra.w < 0.0f;
            // ---- SMALL: one lane per particle; equal pixels within the warp take turns
            if (__any_sync(0xffffffffu, is_small)) {
                const int pix = is_small ? ((int)floorf(ra.y) - ty0) * kStride + ((int)floorf(ra.x) - tx0)
                                         : (0x100000 + lane);
                unsigned int grp = __match_any_sync(0xffffffffu, pix);
                bool pending = is_small;
                while (__any_sync(0xffffffffu, pending)) {
                    const int leader = __ffs(grp) - 1;            // lowest lane of my pixel group still waiting
                    if (pending && lane == leader) {
                        float4 v = fb[pix];
                        v.x += rb.x; v.y += rb.y; v.z += rb.z;
                        fb[pix] = v;
                        pending = false;
                    }
                    grp &= grp - 1u;                              // drop that lane (no-op once the group is empty)
                    __syncwarp();
                }
            }
            // ---- MEDIUM: clip the pixel box to the tile (same float32 formulas as the classification stage)
            int bx0 = 0, by0 = 0, bw = 0, bh = 0;
            if (valid && !is_small) {
                const float fx0 = fmaxf(ceilf(__fsub_rn(__fsub_rn(ra.x, ra.w), 0.5f)), ftx0);
                const float fx1 = fminf(floorf(__fsub_rn(__fadd_rn(ra.x, ra.w), 0.5f)), ftx1);
                const float fy0 = fmaxf(ceilf(__fsub_rn(__fsub_rn(ra.y, ra.w), 0.5f)), fty0);
                const float fy1 = fminf(floorf(__fsub_rn(__fadd_rn(ra.y, ra.w), 0.5f)), fty1);
                if (fx0 <= fx1 && fy0 <= fy1) {
                    bx0 = (int)fx0; by0 = (int)fy0;
                    bw = (int)fx1 - bx0 + 1; bh = (int)fy1 - by0 + 1;
                }
            }
            const int packed = (bx0 - tx0) | ((by0 - ty0) << 8) | (bw << 16) | (bh << 24);
            unsigned int med = __ballot_sync(0xffffffffu, bw > 0);
            while (med) {
                const int src = __ffs(med) - 1;
                med &= med - 1;
                const float ppx = __shfl_sync(0xffffffffu, ra.x, src);
                const float ppy = __shfl_sync(0xffffffffu, ra.y, src);
                const float pc = __shfl_sync(0xffffffffu, ra.z, src);
                const float prp = __shfl_sync(0xffffffffu, ra.w, src);
                const float aR = __shfl_sync(0xffffffffu, rb.x, src);
                const float aG = __shfl_sync(0xffffffffu, rb.y, src);
                const float aB = __shfl_sync(0xffffffffu, rb.z, src);
                const int pk = __shfl_sync(0xffffffffu, packed, src);
                const int lx0 = pk & 0xff, ly0 = (pk >> 8) & 0xff, w = (pk >> 16) & 0xff, hgt = (pk >> 24) & 0xff;
                const int npx = w * hgt;
                const float inv_w = 1.0f / (float)w;
                const float r2 = __fmul_rn(prp, prp);
                for (int k = lane; k < npx; k += 32) {
                    const int j = (int)(((float)k + 0.5f) * inv_w);
                    const int i = k - j * w;
                    const int lx = lx0 + i, ly = ly0 + j;
                    const float dxf = __fsub_rn(__fadd_rn((float)(tx0 + lx), 0.5f), ppx);
                    const float dyf = __fsub_rn(__fadd_rn((float)(ty0 + ly), 0.5f), ppy);
                    const float d2 = __fmaf_rn(dxf, dxf, __fmul_rn(dyf, dyf));
                    if (d2 <= r2) {
                        const float wgt = ex2_approx(d2 * pc);
                        float4 *q = fb + ly * kStride + lx;
                        float4 v = *q;
                        v.x = fmaf(aR, wgt, v.x); v.y = fmaf(aG, wgt, v.y); v.z = fmaf(aB, wgt, v.z);
                        *q = v;
                    }
                }
                __syncwarp();
            }
        }
        __syncthreads();
        float4 *out = partials + (size_t)chunk * (T * T);
        for (int p = threadIdx.x; p < T * T; p += kThreads) {
            const int yy = p / T, xx = p % T;
            float4 s = fb_all[yy * kStride + xx];
#pragma unroll
            for (int w = 1; w < kWarps; ++w) {
                const float4 v = fb_all[w * Cfg::kFbElems + yy * kStride + xx];
                s.x += v.x; s.y += v.y; s.z += v.z;
            }
            out[p] = s;
        }
        __syncthreads();
    }
}

// ---- A6 + A8: compose one tile ----------------------------------------------------------------------------------
// Thread t owns pixels t, t+256, ... of the tile (registers).  Sums the chunk partials in chunk order, then
// gathers the LARGE records of the tile's super-tile (each record is tested against the tile, survivors are
// staged in shared memory and evaluated by every pixel owner), in two-level float32 accumulation.
template <int T>
__global__ void __launch_bounds__(256)
k_compose(const float4 *__restrict__ partials, const unsigned int *__restrict__ chunk_start,
          const float4 *__restrict__ records, const unsigned int *__restrict__ bin_start,
          const DeviceStats *__restrict__ stats, const __grid_constant__ FrameParams fp,
          float *__restrict__ image)
{
    constexpr int kPix = T * T;
    constexpr int kPpt = (kPix + 255) / 256;
    __shared__ float4 sA[256], sB[256];
    __shared__ int s_woff[8], s_cnt;
    const int tile = blockIdx.x;
    const int tx = tile % fp.ntx, ty = tile / fp.ntx;
    const int tx0 = tx * T, ty0 = ty * T;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float acc[kPpt][3], sub[kPpt][3], fxc[kPpt], fyc[kPpt];
#pragma unroll
    for (int k = 0; k < kPpt; ++k) {
        const int p = threadIdx.x + k * 256;
        acc[k][0] = acc[k][1] = acc[k][2] = 0.0f;
        sub[k][0] = sub[k][1] = sub[k][2] = 0.0f;
        fxc[k] = __fadd_rn((float)(tx0 + p % T), 0.5f);
        fyc[k] = __fadd_rn((float)(ty0 + p / T), 0.5f);
    }
    const bool ok = stats->overflow == 0u;
    if (ok) {
        const unsigned int c0 = chunk_start[tile], c1 = chunk_start[tile + 1];
        for (unsigned int ch = c0; ch < c1; ++ch) {
#pragma unroll
            for (int k = 0; k < kPpt; ++k) {
                const int p = threadIdx.x + k * 256;
                if (p < kPix) {
                    const float4 v = __ldg(partials + (size_t)ch * kPix + p);
                    acc[k][0] += v.x; acc[k][1] += v.y; acc[k][2] += v.z;
                }
            }
        }
        const int sbin = fp.n_tiles + (ty >> kSuperShift) * fp.nsx + (tx >> kSuperShift);
        const unsigned int lb = bin_start[sbin], le = bin_start[sbin + 1];
        const float ftx0 = (float)tx0, fty0 = (float)ty0;
        const float ftx1 = (float)min(tx0 + T - 1, fp.W - 1), fty1 = (float)min(ty0 + T - 1, fp.H - 1);
        int batch = 0;
        for (unsigned int base = lb; base < le; base += 256, ++batch) {
            const unsigned int idx = base + threadIdx.x;
            bool hit = false;
            float4 ra, rb;
            if (idx < le) {
                ra = __ldg(records + 2ull * idx);
                rb = __ldg(records + 2ull * idx + 1);
                const float fx0 = ceilf(__fsub_rn(__fsub_rn(ra.x, ra.w), 0.5f));
                const float fx1 = floorf(__fsub_rn(__fadd_rn(ra.x, ra.w), 0.5f));
                const float fy0 = ceilf(__fsub_rn(__fsub_rn(ra.y, ra.w), 0.5f));
                const float fy1 = floorf(__fsub_rn(__fadd_rn(ra.y, ra.w), 0.5f));
                hit = fx0 <= ftx1 && fx1 >= ftx0 && fy0 <= fty1 && fy1 >= fty0;
            }
            const unsigned int bal = __ballot_sync(0xffffffffu, hit);
            if (lane == 0) s_woff[warp] = __popc(bal);
            __syncthreads();
            if (threadIdx.x == 0) {
                int run = 0;
                for (int w = 0; w < 8; ++w) { const int c = s_woff[w]; s_woff[w] = run; run += c; }
                s_cnt = run;
            }
            __syncthreads();
            if (hit) {
                const int pos = s_woff[warp] + __popc(bal & ((1u << lane) - 1u));
                sA[pos] = ra; sB[pos] = rb;
            }
            __syncthreads();
            const int cnt = s_cnt;
            for (int m = 0; m < cnt; ++m) {
                const float4 a = sA[m], b = sB[m];
                const float r2 = __fmul_rn(a.w, a.w);
#pragma unroll
                for (int k = 0; k < kPpt; ++k) {
                    const float dxf = __fsub_rn(fxc[k], a.x), dyf = __fsub_rn(fyc[k], a.y);
                    const float d2 = __fmaf_rn(dxf, dxf, __fmul_rn(dyf, dyf));
                    if (d2 <= r2) {
                        const float wgt = ex2_approx(d2 * a.z);
                        sub[k][0] = fmaf(b.x, wgt, sub[k][0]);
                        sub[k][1] = fmaf(b.y, wgt, sub[k][1]);
                        sub[k][2] = fmaf(b.z, wgt, sub[k][2]);
                    }
                }
            }
            if ((batch & 3) == 3) {
#pragma unroll
                for (int k = 0; k < kPpt; ++k)
#pragma unroll
                    for (int c = 0; c < 3; ++c) { acc[k][c] += sub[k][c]; sub[k][c] = 0.0f; }
            }
            __syncthreads();
        }
#pragma unroll
        for (int k = 0; k < kPpt; ++k)
#pragma unroll
            for (int c = 0; c < 3; ++c) acc[k][c] += sub[k][c];
    }
#pragma unroll
    for (int k = 0; k < kPpt; ++k) {
        const int p = threadIdx.x + k * 256;
        const int ix = tx0 + p % T, iy = ty0 + p / T;
        if (p < kPix && ix < fp.W && iy < fp.H) {
            float *o = image + 3ull * ((size_t)iy * fp.W + ix);
#pragma unroll
            for (int c = 0; c < 3; ++c) o[c] = fp.apply_transfer ? -expm1f(-acc[k][c]) : acc[k][c];
        }
    }
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
