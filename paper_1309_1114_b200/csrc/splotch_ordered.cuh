// splotch_ordered.cuh -- device code of the ordered (E_p != A_p) mode, step A7 of DESIGN.md (sm_100a).
//
// Eq. 1 for one particle is linear in I: crossing particle p maps I -> I + (E_p/A_p - I)(1 - exp(-A_p tau_p)),
// tau_p = rho_0 sqrt(pi) sigma w_p(pixel) from Eq. 2 (:83).  With E_p != A_p the result depends on the order in which
// the particles are crossed (:85 sets that case aside; reading R15 of DESIGN.md: far to near by the float32 camera
// depth z_c, ties by lower particle index first).  The additive path's unordered binning cannot give that order, so
// this mode has its own pipeline:
//   k_ocount    A1+A3      classify, count the (particle, tile) pairs of every block of 2048 particles
//   k_oscan     A4         exclusive scan of the block totals, frame statistics
//   k_opairs    A1-A3+A2   one 32-byte record per particle (index order) and its pairs, in index order:
//                          key = tile << 32 | ~bits(z_c), value = particle index
//   k_rs_*      A4/A7      stable least-significant-digit radix sort of the pairs, 8 bits per pass (4 passes for the
//                          depth, 1-3 for the tile); equal keys keep index order, which is the tie rule of R15.
//                          Replaces thrust::sort_by_key (:201); hand-written: histogram, one linear scan of the
//                          digit-major count matrix, rank by warp match + shared-memory reordering
//   k_obounds   A4         tile start offsets from the sorted keys (replaces reduce_by_key + inclusive_scan, :203-205)
//   k_orender   A7         a CTA walks a chunk of the sorted pairs tile by tile; per pixel it composes the particles'
//                          affine maps I -> t I + c in order, into one (t, c_R, c_G, c_B) per pixel and segment
//   k_ocombine  A7+A8      per tile: fold the segments' maps in order from I = 0 (composition is associative), write
//                          the image
#pragma once
#include "splotch_kernels.cuh"

namespace splotch {

constexpr int kOThreads = 512;                 // k_ocount / k_opairs: 4 consecutive particles per thread
constexpr int kOBlockParticles = 4 * kOThreads;
constexpr int kRsThreads = 512;                // radix sort: 8 elements per thread
constexpr int kRsItems = 8;
constexpr int kRsTile = kRsThreads * kRsItems; // 4096 elements per block and pass
constexpr int kRsWarps = kRsThreads / 32;
constexpr int kOChunkMin = 256;                // records per work item of k_orender (lower bound)

__device__ __forceinline__ int tile_pairs(const Geo &g, const FrameParams &fp)
{
    if (g.cls == CULLED) return 0;
    return ((g.x1 >> fp.tshift) - (g.x0 >> fp.tshift) + 1) * ((g.y1 >> fp.tshift) - (g.y0 >> fp.tshift) + 1);
}

// ---- classify and count pairs per block -------------------------------------------------------------------------
template <bool ALIGNED>
__global__ void __launch_bounds__(kOThreads)
k_ocount(const float *__restrict__ x, const float *__restrict__ y, const float *__restrict__ z, const float *__restrict__ h,
         unsigned long long n, const __grid_constant__ FrameParams fp, unsigned int *__restrict__ blk_pairs,
         DeviceStats *__restrict__ stats)
{
    __shared__ unsigned int s_sum[4], s_z[2];
    if (threadIdx.x < 4) s_sum[threadIdx.x] = 0u;
    if (threadIdx.x < 2) s_z[threadIdx.x] = 0u;
    __syncthreads();
    const unsigned long long lo = (unsigned long long)blockIdx.x * kOBlockParticles;
    const unsigned int len = (unsigned int)min(n - lo, (unsigned long long)kOBlockParticles);
    x += lo; y += lo; z += lo; h += lo;
    const unsigned int i = 4u * threadIdx.x;
    float xs[4], ys[4], zs[4], hs[4];
    load4<ALIGNED>(x, i, len, xs);
    load4<ALIGNED>(y, i, len, ys);
    load4<ALIGNED>(z, i, len, zs);
    load4<ALIGNED>(h, i, len, hs);
    unsigned int pairs = 0u, c1 = 0u, c2 = 0u, c3 = 0u, zmax = 0u, nzmax = 0u;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        Geo g = geometry(xs[j], ys[j], zs[j], hs[j], fp);
        if (!(i + j < len)) g.cls = CULLED;
        if (g.cls != CULLED) { const unsigned int zk = ~__float_as_uint(g.zc); zmax = max(zmax, zk); nzmax = max(nzmax, ~zk); }
        pairs += (unsigned int)tile_pairs(g, fp);
        c1 += g.cls == SMALL; c2 += g.cls == MEDIUM; c3 += g.cls == LARGE;
    }
    pairs = warp_sum(pairs);
    const unsigned int cc = warp_sum(c1 | (c2 << 10) | (c3 << 20));        // at most 128 per field and warp
    zmax = __reduce_max_sync(0xffffffffu, zmax); nzmax = __reduce_max_sync(0xffffffffu, nzmax);
    if ((threadIdx.x & 31) == 0 && zmax) { atomicMax(&s_z[0], zmax); atomicMax(&s_z[1], nzmax); }
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(&s_sum[0], pairs);
        atomicAdd(&s_sum[1], cc & 1023u); atomicAdd(&s_sum[2], (cc >> 10) & 1023u); atomicAdd(&s_sum[3], cc >> 20);
    }
    __syncthreads();
    if (threadIdx.x == 0) blk_pairs[blockIdx.x] = s_sum[0];
    if (threadIdx.x >= 1 && threadIdx.x < 4 && s_sum[threadIdx.x]) atomicAdd(&stats->count[threadIdx.x], (unsigned long long)s_sum[threadIdx.x]);
    if (threadIdx.x == 4 && s_z[0]) { atomicMax(&stats->zkey_max, s_z[0]); atomicMax(&stats->nzkey_max, s_z[1]); }
}

// ---- exclusive scan of the block totals (one block) ---------------------------------------------------------------
constexpr int kOScanThreads = 1024;

__global__ void __launch_bounds__(kOScanThreads)
k_oscan(unsigned int *__restrict__ blk_pairs, int nblk, unsigned long long n, unsigned long long capacity, int n_sm,
        int n_tiles, DeviceStats *__restrict__ stats)
{
    __shared__ unsigned long long s_warp[kOScanThreads / 32];
    __shared__ unsigned long long s_total;
    const int per = (nblk + kOScanThreads - 1) / kOScanThreads;
    const int b0 = min(nblk, (int)threadIdx.x * per), b1 = min(nblk, b0 + per);
    unsigned long long sum = 0;
    for (int b = b0; b < b1; ++b) sum += blk_pairs[b];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned long long inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_warp[w] = inc;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long run = 0;
        for (int k = 0; k < kOScanThreads / 32; ++k) { const unsigned long long c = s_warp[k]; s_warp[k] = run; run += c; }
        s_total = run;
    }
    __syncthreads();
    unsigned long long run = s_warp[w] + inc - sum;
    const unsigned long long total = s_total;
    const bool overflow = total > capacity;
    for (int b = b0; b < b1; ++b) { const unsigned int c = blk_pairs[b]; blk_pairs[b] = (unsigned int)run; run += c; }
    if (threadIdx.x == 0) {
        unsigned long long cs = (total + (unsigned long long)n_sm * 128 - 1) / ((unsigned long long)n_sm * 128);
        cs = (cs + 255) / 256 * 256;             // so that chunks <= 128 n_sm (or capacity / kChunkMax): bounds the segment slots
        cs = min((unsigned long long)4096, max((unsigned long long)kOChunkMin, cs));          // kOChunkMax (k_orender)
        stats->pairs = total;
        stats->large_pairs = 0ull;
        stats->sort_n = overflow ? 0ull : total;         // the sort and the renderers see an empty frame on overflow
        stats->chunks = overflow ? 0ull : (total + cs - 1) / cs;
        stats->capacity = capacity;
        stats->overflow = overflow ? 1u : 0u;
        stats->work_counter = 0u;
        stats->chunk_size = (unsigned int)cs;
        stats->count[0] = n - stats->count[1] - stats->count[2] - stats->count[3];
        // key layout of this frame: depth keys relative to the smallest one, only as many bits as their range needs
        const unsigned int zmin = ~stats->nzkey_max, zrange = stats->zkey_max >= zmin ? stats->zkey_max - zmin : 0u;
        const unsigned int zbits = zrange ? 32u - (unsigned int)__clz(zrange) : 0u;
        const unsigned int tbits = n_tiles > 1 ? 32u - (unsigned int)__clz((unsigned int)n_tiles - 1u) : 0u;
        stats->zkey_min = zmin; stats->zbits = zbits; stats->key_bits = zbits + tbits;
    }
}

// ---- records and pairs in index order -----------------------------------------------------------------------------
// Ordered-mode record, 32 bytes, one per particle: {px, py, c, r2 | flag} {q_R, q_G, q_B, ak}
//   MEDIUM / LARGE: c = -log2(e) / sp^2, r2 = rp^2 (the C1 inside test).  SMALL: (px, py) = the centre of its pixel,
//   c = 0, r2 = 0.25: only that pixel passes the inside test, with weight exp2(0) = 1.
//   kappa > 0: q = E / kappa (the fixed point of Eq. 1 inside the particle), ak = kappa * col [* pi sp^2 (1 - e^-chi^2)
//   for SMALL], so that 1 - exp(-A tau) = 1 - exp(-ak w).   kappa == 0 (flag = sign bit of r2): q = E * col [* ...],
//   I += q w.  Non-finite amplitudes give a record without effect.
template <bool ALIGNED>
__global__ void __launch_bounds__(kOThreads)
k_opairs(const float *__restrict__ x, const float *__restrict__ y, const float *__restrict__ z, const float *__restrict__ h,
         const float *__restrict__ I, const float *__restrict__ scalar, unsigned long long n,
         const __grid_constant__ FrameParams fp, const unsigned int *__restrict__ blk_off, const DeviceStats *__restrict__ stats,
         float4 *__restrict__ rec, unsigned long long *__restrict__ keys, unsigned int *__restrict__ vals)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *s_lut = reinterpret_cast<float4 *>(smem_raw);
    __shared__ unsigned int s_w[kOThreads / 32];
    if (stats->overflow) return;
    const unsigned int zkey_min = stats->zkey_min, zbits = stats->zbits;
    if (fp.lut_total > 0) {
        for (int s = 0; s < fp.n_species; ++s)
            if (fp.sp[s].use_colormap)
                for (int i = threadIdx.x; i < fp.sp[s].lut_n; i += kOThreads)
                    s_lut[fp.sp[s].lut_off + i] = fp.lut[s * kMaxLut + i];
    }
    const unsigned long long lo = (unsigned long long)blockIdx.x * kOBlockParticles;
    const unsigned int len = (unsigned int)min(n - lo, (unsigned long long)kOBlockParticles);
    const unsigned int lo32 = (unsigned int)lo;
    x += lo; y += lo; z += lo; h += lo; I += lo; scalar += lo;
    const unsigned int i = 4u * threadIdx.x;
    float xs[4], ys[4], zs[4], hs[4], Is[4], ss[4];
    load4<ALIGNED>(x, i, len, xs);
    load4<ALIGNED>(y, i, len, ys);
    load4<ALIGNED>(z, i, len, zs);
    load4<ALIGNED>(h, i, len, hs);
    load4<ALIGNED>(I, i, len, Is);
    load4<ALIGNED>(scalar, i, len, ss);
    Geo g[4];
    unsigned int cnt = 0u;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        g[j] = geometry(xs[j], ys[j], zs[j], hs[j], fp);
        if (!(i + j < len)) g[j].cls = CULLED;
        cnt += (unsigned int)tile_pairs(g[j], fp);
    }
    // position of this thread's first pair: block offset + exclusive scan over the threads (index order)
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned int inc = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_w[w] = inc;
    __syncthreads();                                   // also: colour tables staged
    unsigned int woff = 0u;
    for (int k = 0; k < w; ++k) woff += s_w[k];
    unsigned long long pos = (unsigned long long)blk_off[blockIdx.x] + woff + inc - cnt;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if (g[j].cls == CULLED) continue;
        const unsigned int idx = lo32 + i + j;
        const int s = species_of(idx, fp);
        const SpeciesDev &S = fp.sp[s];
        const float4 *lut = fp.lut_total > 0 ? s_lut + S.lut_off : fp.lut + s * kMaxLut;
        float3 vv = make_float3(0.0f, 0.0f, 0.0f);
        if (fp.any_vector && idx < n) vv = make_float3(__ldg(fp.vec[0] + idx), __ldg(fp.vec[1] + idx), __ldg(fp.vec[2] + idx));
        const float3 rgb = colour_of(ss[j], S, lut, species_range(fp, s), vv);
        const float3 E = make_float3(S.brightness * rgb.x, S.brightness * rgb.y, S.brightness * rgb.z);
        const bool small = g[j].cls == SMALL;
        const float sp2 = __fmul_rn(g[j].sp, g[j].sp);
        const float col = 1.7724538509055160273f * hs[j] * Is[j] * (small ? fp.csmall * sp2 : 1.0f);   // tau at weight 1
        float4 ra, rb;
        if (small) {
            ra.x = __fadd_rn((float)g[j].x0, 0.5f); ra.y = __fadd_rn((float)g[j].y0, 0.5f);
            ra.z = 0.0f; ra.w = 0.25f;
        } else {
            ra.x = g[j].px; ra.y = g[j].py;
            ra.z = __fdividef(-1.4426950408889634f, sp2);
            ra.w = __fmul_rn(g[j].rp, g[j].rp);
        }
        const float kappa = S.absorb;
        if (kappa > 0.0f) {
            const float inv = 1.0f / kappa;
            rb = make_float4(E.x * inv, E.y * inv, E.z * inv, kappa * col);
        } else {
            rb = make_float4(E.x * col, E.y * col, E.z * col, 0.0f);
            ra.w = -ra.w;                              // flag: pure emission, I += q w
        }
        const float am = fmaxf(fmaxf(fabsf(rb.x), fabsf(rb.y)), fmaxf(fabsf(rb.z), fabsf(rb.w)));
        if (!(am <= 3.0e38f)) rb = make_float4(0.0f, 0.0f, 0.0f, 0.0f);   // Inf / NaN: a record without effect
        st_record(rec + (size_t)idx, idx, ra, rb);      // 32-byte record idx = units 2 idx
        const unsigned long long zkey = (unsigned long long)(~__float_as_uint(g[j].zc) - zkey_min);
        const int tx0 = g[j].x0 >> fp.tshift, tx1 = g[j].x1 >> fp.tshift;
        const int ty0 = g[j].y0 >> fp.tshift, ty1 = g[j].y1 >> fp.tshift;
        for (int ty = ty0; ty <= ty1; ++ty)
            for (int tx = tx0; tx <= tx1; ++tx) {
                keys[pos] = ((unsigned long long)(unsigned int)(ty * fp.ntx + tx) << zbits) | zkey;
                vals[pos] = idx;
                ++pos;
            }
    }
}

// ---- stable LSD radix sort, 8 bits per pass, 64-bit keys + 32-bit values -----------------------------------------
__device__ __forceinline__ unsigned int rs_digit(unsigned long long key, int shift) { return (unsigned int)(key >> shift) & 255u; }

// hist is digit-major: hist[d * nblk + b]; one linear exclusive scan over it gives every block's output offsets.
__global__ void __launch_bounds__(kRsThreads)
k_rs_count(const unsigned long long *__restrict__ keys, const DeviceStats *__restrict__ stats, int shift, int nblk,
           unsigned int *__restrict__ hist)
{
    __shared__ unsigned int s_h[256];
    if ((unsigned int)shift >= stats->key_bits) return;          // this frame's keys have no bit left for this pass
    if (threadIdx.x < 256) s_h[threadIdx.x] = 0u;
    __syncthreads();
    const unsigned long long P = stats->sort_n;
    const unsigned long long seg = (unsigned long long)blockIdx.x * kRsTile;
    if (seg < P) {
        const unsigned int cnt = (unsigned int)min(P - seg, (unsigned long long)kRsTile);
        // A thread takes 8 CONSECUTIVE keys and adds one shared-memory atomic per run of equal digits.  The low depth digits are spread
        // evenly (8 atomics per thread on different counters), but a block's high depth digit and its tile digits take few values
        // (the pairs are sorted by the lower digits, or still in index order): there plain atomics piled up on a few counters
        // (0.66 ms a pass on cfg4) and warp aggregation by match.any cost 0.59 ms, against 0.17 ms for the spread digits.
        const unsigned int p0 = threadIdx.x * kRsItems;
        unsigned long long k[kRsItems];
        if (p0 + kRsItems <= cnt) {
            const ulonglong2 *src = reinterpret_cast<const ulonglong2 *>(keys + seg + p0);
#pragma unroll
            for (int i = 0; i < kRsItems / 2; ++i) { const ulonglong2 v = __ldg(src + i); k[2 * i] = v.x; k[2 * i + 1] = v.y; }
        } else {
#pragma unroll
            for (int i = 0; i < kRsItems; ++i) k[i] = p0 + i < cnt ? __ldg(keys + seg + p0 + i) : 0ull;
        }
        unsigned int dprev = 256u, run = 0u;
#pragma unroll
        for (int i = 0; i < kRsItems; ++i) {
            const unsigned int d = p0 + i < cnt ? rs_digit(k[i], shift) : 256u;
            if (d != dprev) {
                if (run) atomicAdd(&s_h[dprev], run);
                dprev = d; run = 0u;
            }
            run += d < 256u ? 1u : 0u;
        }
        if (run) atomicAdd(&s_h[dprev], run);
    }
    __syncthreads();
    if (threadIdx.x < 256) hist[(size_t)threadIdx.x * nblk + blockIdx.x] = s_h[threadIdx.x];
}

// exclusive scan of m unsigned ints in place, three launches: block sums, scan of the sums (one block), apply
constexpr int kScThreads = 512, kScItems = 8, kScTile = kScThreads * kScItems;

__device__ __forceinline__ unsigned int block_excl_scan_u32(unsigned int v, unsigned int *s_warp, unsigned int *total)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    unsigned int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_warp[w] = inc;
    __syncthreads();
    if (w == 0) {
        const unsigned int c = lane < nw ? s_warp[lane] : 0u;
        unsigned int ci = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int t = __shfl_up_sync(0xffffffffu, ci, o);
            if (lane >= o) ci += t;
        }
        if (lane < nw) s_warp[lane] = ci - c;
        if (lane == 31) *total = ci;
    }
    __syncthreads();
    const unsigned int r = s_warp[w] + inc - v;
    __syncthreads();
    return r;
}

__global__ void __launch_bounds__(kScThreads)
k_sc_reduce(const unsigned int *__restrict__ a, unsigned int m, unsigned int *__restrict__ sums,
            const DeviceStats *__restrict__ stats, int shift)
{
    __shared__ unsigned int s_warp[32], s_total;
    if ((unsigned int)shift >= stats->key_bits) return;
    const unsigned int base = blockIdx.x * kScTile + threadIdx.x * kScItems;
    unsigned int s = 0u;
    if (base + kScItems <= m) {
        const uint4 u = *reinterpret_cast<const uint4 *>(a + base), v = *reinterpret_cast<const uint4 *>(a + base + 4);
        s = u.x + u.y + u.z + u.w + v.x + v.y + v.z + v.w;
    } else {
        for (int k = 0; k < kScItems; ++k) if (base + k < m) s += a[base + k];
    }
    (void)block_excl_scan_u32(s, s_warp, &s_total);
    if (threadIdx.x == 0) sums[blockIdx.x] = s_total;
}

__global__ void __launch_bounds__(1024)
k_sc_top(unsigned int *__restrict__ sums, int ng, const DeviceStats *__restrict__ stats, int shift)
{
    __shared__ unsigned int s_warp[32], s_total;
    if ((unsigned int)shift >= stats->key_bits) return;
    const int per = (ng + 1023) / 1024;
    const int b0 = min(ng, (int)threadIdx.x * per), b1 = min(ng, b0 + per);
    unsigned int s = 0u;
    for (int b = b0; b < b1; ++b) s += sums[b];
    unsigned int run = block_excl_scan_u32(s, s_warp, &s_total);
    for (int b = b0; b < b1; ++b) { const unsigned int c = sums[b]; sums[b] = run; run += c; }
}

__global__ void __launch_bounds__(kScThreads)
k_sc_apply(unsigned int *__restrict__ a, unsigned int m, const unsigned int *__restrict__ sums,
           const DeviceStats *__restrict__ stats, int shift)
{
    __shared__ unsigned int s_warp[32], s_total;
    if ((unsigned int)shift >= stats->key_bits) return;
    const unsigned int base = blockIdx.x * kScTile + threadIdx.x * kScItems;
    unsigned int v[kScItems];
    unsigned int s = 0u;
#pragma unroll
    for (int k = 0; k < kScItems; ++k) { v[k] = base + k < m ? a[base + k] : 0u; s += v[k]; }
    unsigned int run = block_excl_scan_u32(s, s_warp, &s_total) + sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < kScItems; ++k) {
        if (base + k < m) a[base + k] = run;
        run += v[k];
    }
}

struct RsSmem {
    unsigned long long keys[kRsTile];
    unsigned int vals[kRsTile];
    unsigned int wcount[kRsWarps][257];
    unsigned int dstart[256];
    unsigned int gbase[256];
    unsigned int warp_tmp[32];
    unsigned int total;
};

// One block moves its 4096 elements to their places of this pass.  Element order inside the block is (warp, item,
// lane) = position order; ranks among equal digits are taken in that order (warp match + per-warp counters, then an
// exclusive prefix over the warps), so the pass is stable.  The elements are first reordered in shared memory, then
// written out position by position: consecutive threads write consecutive addresses of a digit's run.
__global__ void __launch_bounds__(kRsThreads)
k_rs_scatter(const unsigned long long *__restrict__ keys_in, const unsigned int *__restrict__ vals_in,
             unsigned long long *__restrict__ keys_out, unsigned int *__restrict__ vals_out,
             const DeviceStats *__restrict__ stats, int shift, int nblk, const unsigned int *__restrict__ hist)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    RsSmem &S = *reinterpret_cast<RsSmem *>(smem_raw);
    const unsigned long long P = stats->sort_n;
    const unsigned long long seg = (unsigned long long)blockIdx.x * kRsTile;
    if (seg >= P || (unsigned int)shift >= stats->key_bits) return;
    const unsigned int cnt = (unsigned int)min(P - seg, (unsigned long long)kRsTile);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < kRsWarps * 257; i += kRsThreads) (&S.wcount[0][0])[i] = 0u;
    unsigned long long key[kRsItems];
    unsigned int val[kRsItems], rank[kRsItems];
    const unsigned int wbase = w * (32 * kRsItems) + lane;
#pragma unroll
    for (int i = 0; i < kRsItems; ++i) {
        const unsigned int p = wbase + i * 32;
        key[i] = p < cnt ? __ldg(keys_in + seg + p) : ~0ull;
        val[i] = p < cnt ? __ldg(vals_in + seg + p) : 0u;
    }
    __syncthreads();
    // the eight matches first (independent, their latency overlaps), then the counter rounds, which depend on each other
    unsigned int dig[kRsItems], peers[kRsItems];
#pragma unroll
    for (int i = 0; i < kRsItems; ++i) {
        dig[i] = wbase + i * 32 < cnt ? rs_digit(key[i], shift) : 256u;
        peers[i] = __match_any_sync(0xffffffffu, dig[i]);
    }
#pragma unroll
    for (int i = 0; i < kRsItems; ++i) {
        const int leader = __ffs(peers[i]) - 1;
        unsigned int old = 0u;
        if (lane == leader) { old = S.wcount[w][dig[i]]; S.wcount[w][dig[i]] = old + (unsigned int)__popc(peers[i]); }
        old = __shfl_sync(0xffffffffu, old, leader);
        rank[i] = old + (unsigned int)__popc(peers[i] & ((1u << lane) - 1u));
        __syncwarp();
    }
    __syncthreads();
    unsigned int tot = 0u;
    if (threadIdx.x < 256) {
        for (int k = 0; k < kRsWarps; ++k) { const unsigned int c = S.wcount[k][threadIdx.x]; S.wcount[k][threadIdx.x] = tot; tot += c; }
    }
    const unsigned int ds = block_excl_scan_u32(tot, S.warp_tmp, &S.total);      // threads >= 256 contribute 0
    if (threadIdx.x < 256) {
        S.dstart[threadIdx.x] = ds;
        S.gbase[threadIdx.x] = hist[(size_t)threadIdx.x * nblk + blockIdx.x] - ds;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < kRsItems; ++i) {
        const unsigned int p = wbase + i * 32;
        if (p < cnt) {
            const unsigned int d = rs_digit(key[i], shift);
            const unsigned int lp = S.dstart[d] + S.wcount[w][d] + rank[i];
            S.keys[lp] = key[i];
            S.vals[lp] = val[i];
        }
    }
    __syncthreads();
    for (unsigned int j = threadIdx.x; j < cnt; j += kRsThreads) {
        const unsigned long long k = S.keys[j];
        const unsigned int o = S.gbase[rs_digit(k, shift)] + j;
        keys_out[o] = k;
        vals_out[o] = S.vals[j];
    }
}

// ---- tile start offsets from the sorted keys ----------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_obounds(const unsigned long long *__restrict__ keys0, const unsigned long long *__restrict__ keys1,
          const DeviceStats *__restrict__ stats, int n_tiles, unsigned int *__restrict__ tile_start)
{
    const unsigned long long P = stats->sort_n;
    const unsigned long long p0 = 4ull * ((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x);     // four consecutive pairs per thread
    if (P == 0ull) {
        for (unsigned long long p = p0; p < p0 + 4ull; ++p) if (p <= (unsigned long long)n_tiles) tile_start[p] = 0u;
        return;
    }
    if (p0 >= P) return;
    // the sorted pairs are in buffer (number of passes that ran) & 1
    const unsigned long long *keys = (((stats->key_bits + 7u) >> 3) & 1u) ? keys1 : keys0;
    const unsigned int zbits = stats->zbits;
    unsigned long long k[4];
    if (p0 + 4ull <= P) {
        const ulonglong2 a = *reinterpret_cast<const ulonglong2 *>(keys + p0), b = *reinterpret_cast<const ulonglong2 *>(keys + p0 + 2);
        k[0] = a.x; k[1] = a.y; k[2] = b.x; k[3] = b.y;
    } else {
        for (int j = 0; j < 4; ++j) k[j] = p0 + j < P ? keys[p0 + j] : keys[P - 1];
    }
    int tp = p0 > 0 ? (int)(__ldg(keys + p0 - 1) >> zbits) : -1;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const unsigned long long p = p0 + j;
        if (p < P) {
            const int t = (int)(k[j] >> zbits);
            for (int u = tp + 1; u <= t; ++u) tile_start[u] = (unsigned int)p;
            if (p == P - 1) for (int u = t + 1; u <= n_tiles; ++u) tile_start[u] = (unsigned int)P;
            tp = t;
        }
    }
}

__global__ void __launch_bounds__(256)
k_odiff(const unsigned int *__restrict__ tile_start, int n_tiles, unsigned int *__restrict__ out)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n_tiles) out[t] = tile_start[t + 1] - tile_start[t];
}

// ---- A7: ordered compositing of one chunk -------------------------------------------------------------------------
// a = 1 - exp(-x) and e = exp(-x) for the optical depth x of one particle at one pixel.  |x| < 0.25: a from the
// Taylor series to x^8 (relative error < 2e-8), e = 1 - a; otherwise e = 2^(-x log2 e) (ex2.approx), a = 1 - e.
__device__ __forceinline__ void absorb_pair(float x, float &a, float &e)
{
    // (1 - exp(-x)) / x = sum_k (-x)^k / (k + 1)!, k = 0 .. 7, by Horner's rule in y = -x
    const float y = -x;
    float p = 2.48015873e-5f;                       // 1 / 8!
    p = fmaf(p, y, 1.98412698e-4f);                 // 1 / 7!
    p = fmaf(p, y, 1.38888889e-3f);                 // 1 / 6!
    p = fmaf(p, y, 8.33333333e-3f);                 // 1 / 5!
    p = fmaf(p, y, 4.16666667e-2f);                 // 1 / 4!
    p = fmaf(p, y, 1.66666667e-1f);                 // 1 / 3!
    p = fmaf(p, y, 0.5f);
    p = fmaf(p, y, 1.0f);
    const float as = x * p;
    const float el = ex2_approx(x * -1.4426950408889634f);
    const bool small = fabsf(x) < 0.25f;
    a = small ? as : 1.0f - el;
    e = small ? 1.0f - as : el;
}

// floor of v as an int, for any float (clamped to +-1e9 first; NaN gives -1e9)
__device__ __forceinline__ int floor_clamped(float v) { return __float2int_rd(fminf(fmaxf(v, -1.0e9f), 1.0e9f)); }

// A segment (the records of one tile inside one chunk of the sorted list) is cut into four consecutive quarters, one per
// warp.  A warp keeps a private map (t, c_R, c_G, c_B) per pixel of the tile in shared memory and crosses its records in
// order, 32 FRAGMENTS (record, pixel of its box inside the tile) at a time: a SMALL record is one fragment, the others one per
// pixel of their box, so all lanes work whatever the mix (the first version gave every record to the 32 lanes that own a
// strip of 64 pixels: 16 of 32 lanes active, 111 warp instructions per pair, profiles/r2_step1_*).  Fragments of one batch that
// fall on the same pixel are applied in rounds, lower lane (earlier record) first: the order per pixel is the sorted order.
// At the end of the segment the four maps are composed in order (composition is associative) into the segment's map.
constexpr int kORThreads = 128;
constexpr int kORWarps = kORThreads / 32;
constexpr int kOChunkMax = 4096;               // records per chunk: a warp composes at most 1024 records in float32

template <int T> struct ORenderSmem {
    float4 map[kORWarps][T * T];
    unsigned int owner[kORWarps][T * T];       // per pixel: the lowest lane that wants it in the current round (0xffffffff: free)
    float4 recA[kORWarps][32], recB[kORWarps][32];
    uint4 box[kORWarps][32];                   // {x0 | y0 << 8 | (width - 1) << 16 | (height - 1) << 24 (tile-relative), first fragment, 65536 / width rounded up, -}
    unsigned int chunk;
    int tile;
};

template <int T>
__global__ void __launch_bounds__(kORThreads)
k_orender(const float4 *__restrict__ rec, const unsigned int *__restrict__ vals0, const unsigned int *__restrict__ vals1,
          const unsigned int *__restrict__ tile_start, DeviceStats *__restrict__ stats, float4 *__restrict__ seg,
          const __grid_constant__ FrameParams fp)
{
    constexpr int kPix = T * T;
    extern __shared__ __align__(16) unsigned char orender_smem_raw[];
    ORenderSmem<T> &S = *reinterpret_cast<ORenderSmem<T> *>(orender_smem_raw);
    const unsigned int *__restrict__ vals = (((stats->key_bits + 7u) >> 3) & 1u) ? vals1 : vals0;   // the sorted values
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned int lt = (1u << lane) - 1u;
    const unsigned int total = (unsigned int)stats->chunks;
    const unsigned int K = stats->chunk_size;
    const unsigned int pairs = (unsigned int)stats->sort_n;
    float4 *map = S.map[warp];
    for (;;) {
        __syncthreads();
        if (warp == 0) {
            unsigned int c = 0u;
            if (lane == 0) c = atomicAdd(&stats->work_counter, 1u);
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c < total) {
                const unsigned int r = c * K;
                int lo = 0, n = fp.n_tiles;
                while (n > 1) {
                    const int step = (n + 31) / 32;
                    const int t = lo + lane * step;
                    const bool le = t < lo + n && __ldg(tile_start + t) <= r;
                    const int k = __popc(__ballot_sync(0xffffffffu, le)) - 1;
                    lo += k * step;
                    n = min(step, n - k * step);
                }
                if (lane == 0) S.tile = lo;
            }
            if (lane == 0) S.chunk = c;
        }
        __syncthreads();
        const unsigned int chunk = S.chunk;
        if (chunk >= total) break;
        const unsigned int r0 = chunk * K, r1 = min(r0 + K, pairs);
        int tile = S.tile;
        unsigned int tb = tile_start[tile], te = tile_start[tile + 1];
        for (;;) {
            const unsigned int begin = max(tb, r0), end = min(te, r1);
            const int tx0 = (tile % fp.ntx) * T, ty0 = (tile / fp.ntx) * T;
            // this warp's quarter of the segment, in whole batches of 32 records
            const unsigned int nb = (end - begin + 31u) / 32u, per = (nb + kORWarps - 1u) / kORWarps;
            const unsigned int wb = min(end, begin + 32u * per * (unsigned int)warp), we = min(end, wb + 32u * per);
            for (int i = lane; i < kPix; i += 32) { map[i] = make_float4(1.0f, 0.0f, 0.0f, 0.0f); S.owner[warp][i] = 0xffffffffu; }
            __syncwarp();
            // the records of a batch are gathered through the sorted values; the next batch's records and the following batch's
            // values are requested before the current batch is composed
            unsigned int vnext = wb + 32u + lane < we ? __ldg(vals + wb + 32u + lane) : 0u;
            float4 nra = make_float4(0.f, 0.f, 0.f, 0.f), nrb = nra;
            if (wb + lane < we) ld_record(rec, __ldg(vals + wb + lane), nra, nrb);
            for (unsigned int base = wb; base < we; base += 32u) {
                const float4 ra = nra, rb = nrb;
                const bool valid = base + lane < we;
                {
                    const unsigned int nxt = base + 32u + lane;
                    nra = make_float4(0.f, 0.f, 0.f, 0.f); nrb = nra;
                    if (nxt < we) ld_record(rec, vnext, nra, nrb);
                    if (nxt + 32u < we) vnext = __ldg(vals + nxt + 32u);
                }
                // pixel box of the record inside the tile: exact for SMALL records (c = 0: the one pixel of the centre), one pixel of
                // slack for the others (the C1 inside test decides)
                unsigned int nfrag = 0u, bx = 0u;
                if (valid) {
                    // C1's box is ceil((p - rp) - 0.5) .. floor((p + rp) - 0.5); rp is recovered from r2 = rp^2 to a few ulp, so the bounds
                    // are widened by a relative 1e-4 (never narrower than C1's box, one pixel wider only next to an integer)
                    const float r2 = fabsf(ra.w);
                    const bool point = ra.z == 0.0f;                  // SMALL: the record holds the centre of its pixel
                    const float rr = point ? 0.0f : sqrtf(r2) * 1.0001f + 1.0e-4f;
                    const float lo_off = point ? 0.0f : 0.5f;         // ceil(v) = floor(v - eps) + 1, done as floor(v + 0.5 - eps) for v = p - rp - 0.5 + 0.5
                    const int x0 = max(floor_clamped(ra.x - rr + lo_off) - tx0, 0), x1 = min(floor_clamped(ra.x + rr - lo_off) - tx0, T - 1);
                    const int y0 = max(floor_clamped(ra.y - rr + lo_off) - ty0, 0), y1 = min(floor_clamped(ra.y + rr - lo_off) - ty0, T - 1);
                    if (x0 <= x1 && y0 <= y1) {
                        nfrag = (unsigned int)((x1 - x0 + 1) * (y1 - y0 + 1));
                        bx = (unsigned int)x0 | ((unsigned int)y0 << 8) | ((unsigned int)(x1 - x0) << 16) | ((unsigned int)(y1 - y0) << 24);
                    }
                }
                unsigned int inc = nfrag;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const unsigned int t = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += t;
                }
                const unsigned int nf = __shfl_sync(0xffffffffu, inc, 31);
                const bool single = __all_sync(0xffffffffu, nfrag <= 1u);        // every record is one fragment (or none): lane = record
                // otherwise the records that have fragments are staged in shared memory, packed: source c starts at fragment first_c
                const unsigned int has = __ballot_sync(0xffffffffu, nfrag > 0u);
                unsigned int my_first = 0xffffffffu;               // lane c: first fragment of packed source c
                if (!single) {
                    if (nfrag > 0u) {
                        const int c = __popc(has & lt);
                        const unsigned int bw = ((bx >> 16) & 255u) + 1u;
                        S.recA[warp][c] = ra; S.recB[warp][c] = rb;
                        S.box[warp][c] = make_uint4(bx, inc - nfrag, (65536u + bw - 1u) / bw, 0u);
                    }
                    __syncwarp();
                    if (lane < __popc(has)) my_first = S.box[warp][lane].y;
                }
                for (unsigned int f0 = 0u; f0 < (single ? 1u : nf); f0 += 32u) {
                    float4 A = ra, B = rb;
                    unsigned int box = bx, k = 0u, inv = 65536u;
                    bool act = nfrag == 1u;
                    if (!single) {
                        const unsigned int f = f0 + lane;
                        act = f < nf;
                        // source of fragment f: the last packed source that starts at or before f.  `cover` sources start at or before f0;
                        // the starts inside this window are one bit each, counted up to this lane
                        const int cover = __popc(__ballot_sync(0xffffffffu, my_first <= f0));
                        const unsigned int rel = my_first - f0;
                        const unsigned int starts = __reduce_or_sync(0xffffffffu, (rel >= 1u && rel < 32u) ? (1u << rel) : 0u);
                        const int sl = cover - 1 + __popc(starts & ((2u << lane) - 1u));
                        const uint4 bq = S.box[warp][sl];
                        A = S.recA[warp][sl]; B = S.recB[warp][sl];
                        box = bq.x; k = f - bq.y; inv = bq.z;
                    }
                    const unsigned int bw = ((box >> 16) & 255u) + 1u;
                    const unsigned int ky = (k * inv) >> 16, kx = k - ky * bw;      // k / bw, k % bw (exact for k < 1024, bw <= 32)
                    const int lx = (int)((box & 255u) + kx), ly = (int)(((box >> 8) & 255u) + ky);
                    const float dxf = __fsub_rn(__fadd_rn((float)(tx0 + lx), 0.5f), A.x);
                    const float dyf = __fsub_rn(__fadd_rn((float)(ty0 + ly), 0.5f), A.y);
                    const float d2 = __fmaf_rn(dxf, dxf, __fmul_rn(dyf, dyf));
                    act = act && d2 <= fabsf(A.w);
                    const float wgt = ex2_approx(d2 * A.z);
                    const bool emit_only = A.w < 0.0f;
                    float a, e;
                    absorb_pair(B.w * wgt, a, e);
                    // I -> e I + g with g = q a (absorbing) or q w (pure emitter, e = 1)
                    const float ga = emit_only ? wgt : a;
                    e = emit_only ? 1.0f : e;
                    const float gr = B.x * ga, gg = B.y * ga, gb = B.z * ga;
                    const int pix = ly * T + lx;
                    // Fragments of this step that fall on the same pixel are applied in rounds, lower lane (earlier record) first: every
                    // pending lane bids for its pixel with a shared-memory atomicMin of its lane number, the winners apply and free the
                    // pixel.  (First version: match.any, 37 % of the stall samples; second: one vote per bit of the pixel index, 25
                    // instructions per step; a round of bids costs about 10 and most steps need one.)
                    unsigned int *own = S.owner[warp];
                    bool pending = act;
                    while (__any_sync(0xffffffffu, pending)) {
                        if (pending) atomicMin(own + pix, (unsigned int)lane);
                        __syncwarp();
                        const bool win = pending && own[pix] == (unsigned int)lane;
                        __syncwarp();
                        if (win) {
                            float4 m = map[pix];
                            m.x *= e; m.y = fmaf(m.y, e, gr); m.z = fmaf(m.z, e, gg); m.w = fmaf(m.w, e, gb);
                            map[pix] = m;
                            own[pix] = 0xffffffffu;
                            pending = false;
                        }
                        __syncwarp();
                    }
                }
                __syncwarp();
            }
            __syncthreads();                  // the four maps of the segment are complete
            {   // compose them in order: slot = chunk + tile (segments of a tile are consecutive chunks)
                float4 *out = seg + ((size_t)chunk + (size_t)tile) * kPix;
                for (int p = threadIdx.x; p < kPix; p += kORThreads) {
                    double t = 1.0, cr = 0.0, cg = 0.0, cb = 0.0;
#pragma unroll
                    for (int w = 0; w < kORWarps; ++w) {
                        const float4 m = S.map[w][p];
                        const double mt = (double)m.x;
                        t *= mt; cr = fma(cr, mt, (double)m.y); cg = fma(cg, mt, (double)m.z); cb = fma(cb, mt, (double)m.w);
                    }
                    out[p] = make_float4((float)t, (float)cr, (float)cg, (float)cb);
                }
            }
            if (te >= r1) break;
            do { ++tile; tb = te; te = tile_start[tile + 1]; } while (te == tb);
            __syncthreads();                  // the maps are rewritten for the next tile
        }
    }
}

// ---- A7 + A8: fold the segments of a tile in order, write the image -------------------------------------------------
// A CTA folds the segments of 64 pixels of one tile: four slices of the segment range are composed in parallel by 64
// threads each (composition of the maps (t, c) is associative), the four partial maps are then applied in order.  A
// halo-core tile has more than a thousand segments: one thread per pixel walking them alone was latency bound.
constexpr int kCombinePix = 64, kCombineSlices = 4;

template <int T>
__global__ void __launch_bounds__(kCombinePix * kCombineSlices)
k_ocombine(const float4 *__restrict__ seg, const unsigned int *__restrict__ tile_start, const DeviceStats *__restrict__ stats,
           const __grid_constant__ FrameParams fp, float *__restrict__ image)
{
    constexpr int kPix = T * T, kGroups = kPix / kCombinePix;
    __shared__ double s_map[kCombineSlices][4][kCombinePix];
    const int tile = blockIdx.x / kGroups;
    const int p = (blockIdx.x % kGroups) * kCombinePix + (threadIdx.x % kCombinePix);
    const int slice = threadIdx.x / kCombinePix;
    const int tx0 = (tile % fp.ntx) * T, ty0 = (tile / fp.ntx) * T;
    const unsigned int tb = tile_start[tile], te = tile_start[tile + 1];
    const unsigned int K = stats->chunk_size;
    const bool any = te > tb && stats->overflow == 0u;
    const unsigned int c0 = any ? tb / K : 1u, c1 = any ? (te - 1u) / K : 0u;
    const unsigned int nseg = any ? c1 - c0 + 1u : 0u, per = (nseg + kCombineSlices - 1) / kCombineSlices;
    const unsigned int s0 = c0 + slice * per, s1 = min(s0 + per, c1 + 1u);       // this slice's segments [s0, s1)
    double t = 1.0, cr = 0.0, cg = 0.0, cb = 0.0;
    for (unsigned int c = s0; c < s1 && any; c += 8) {          // eight maps in flight, composed in order
        float4 m[8];
#pragma unroll
        for (int k = 0; k < 8; ++k)
            m[k] = c + k < s1 ? __ldg(seg + ((size_t)(c + k) + (size_t)tile) * kPix + p) : make_float4(1.0f, 0.0f, 0.0f, 0.0f);
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const double mt = (double)m[k].x;
            t *= mt;
            cr = fma(cr, mt, (double)m[k].y);
            cg = fma(cg, mt, (double)m[k].z);
            cb = fma(cb, mt, (double)m[k].w);
        }
    }
    const int q = threadIdx.x % kCombinePix;
    s_map[slice][0][q] = t; s_map[slice][1][q] = cr; s_map[slice][2][q] = cg; s_map[slice][3][q] = cb;
    __syncthreads();
    if (slice == 0) {
        double I[3] = {0.0, 0.0, 0.0};                          // background (reading R16)
#pragma unroll
        for (int s = 0; s < kCombineSlices; ++s) {
            const double mt = s_map[s][0][q];
            I[0] = fma(I[0], mt, s_map[s][1][q]);
            I[1] = fma(I[1], mt, s_map[s][2][q]);
            I[2] = fma(I[2], mt, s_map[s][3][q]);
        }
        const int ix = tx0 + p % T, iy = ty0 + p / T;
        if (ix < fp.W && iy < fp.H) {
            float *o = image + 3ull * ((size_t)iy * fp.W + ix);
            o[0] = (float)I[0]; o[1] = (float)I[1]; o[2] = (float)I[2];
        }
    }
}

}  // namespace splotch
