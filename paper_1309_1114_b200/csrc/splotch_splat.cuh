// splotch_splat.cuh -- A5, the tile renderer for SMALL + MEDIUM records (sm_100a).
//
// The paper's medium-particle kernel (a CUDA block owns a tile in shared memory, particles are
// staged n_p at a time, one pixel per thread) redesigned for B200:
//   * a work item is a chunk of consecutive bin-sorted records, cut into segments at tile boundaries, so a heavy tile
//     is shared by many CTAs (the load-imbalance problem of :242);
//   * records stream from HBM into shared memory with 1-D bulk copies (cp.async.bulk, the TMA engine) that complete
//     on an mbarrier: two windows of 256 records per CTA, the next one in flight while the current one is rendered,
//     no registers and no thread stalls spent on the copy (the first version loaded a batch into registers, waited
//     for it and barriered twice per 128 records: 0.18 of its 0.48 ms on cfg1 were that skeleton alone,
//     profiles/r1_step3_*);
//   * records whose box is at most 2 x 2 pixels (every SMALL record) are splatted by the thread that decodes them,
//     into fixed-point planes in shared memory (native integer red.shared);
//   * all others are evaluated by pixel owners: a warp owns a 64-pixel strip, a lane two adjacent pixels, sums live in
//     registers as packed float32 pairs (FADD2 / FFMA2 / FMUL2), no atomics;
//   * at the end of a segment everything is added to the tile's 64-bit fixed-point sums in L2 (exact, commutative).
#pragma once
#include "splotch_kernels.cuh"

namespace splotch {

template <int T> struct Splat2Cfg {
    using Base = SplatCfg<T>;
    static constexpr int kPix = Base::kPix, kThreads = Base::kThreads;
    static constexpr int kWin = kThreads > 256 ? kThreads : 256;     // records per bulk copy
    static constexpr int kStages = 2;
    static constexpr int kFoldRecords = 1024;                        // fold the register sub-sums about this often
    static constexpr size_t kStageBytes = 32u * kWin;
    static constexpr size_t kSmemBytes = kStageBytes * kStages + sizeof(unsigned int) * (6 * kPix + 2 * kWin) + 8 * kStages +
                                         sizeof(unsigned short) * kWin * Base::kWarps;
};

__device__ __forceinline__ unsigned int smem_u32(const void *p) { return (unsigned int)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned int bar, unsigned int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned int bar, unsigned int bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(unsigned int dst, const void *src, unsigned int bytes, unsigned int bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned int bar, unsigned int parity)
{
    unsigned int ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}

template <int T>
__global__ void __launch_bounds__(SplatCfg<T>::kThreads)
k_splat(const float4 *__restrict__ records, const unsigned int *__restrict__ bin_start, DeviceStats *__restrict__ stats,
        unsigned long long *__restrict__ accum, const __grid_constant__ FrameParams fp)
{
    using Cfg = Splat2Cfg<T>;
    using Geo = SplatCfg<T>;
    constexpr int kPix = Cfg::kPix, kThreads = Cfg::kThreads, kWin = Cfg::kWin, kStages = Cfg::kStages;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4 *stage = reinterpret_cast<float4 *>(smem_raw);                                   // [kStages][kWin][2]
    unsigned int *fb = reinterpret_cast<unsigned int *>(smem_raw + Cfg::kStageBytes * kStages);   // lo R G B, hi R G B
    unsigned int *stM = fb + 6 * kPix;                                                      // [2][kWin] strip masks
    unsigned long long *mbar = reinterpret_cast<unsigned long long *>(stM + 2 * kWin);
    unsigned short *hits = reinterpret_cast<unsigned short *>(mbar + kStages);              // [warps][kWin] per-warp hit lists
    __shared__ unsigned int s_chunk;
    __shared__ int s_tile;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sx = warp % Geo::kStripsX, sy = warp / Geo::kStripsX;
    const int lx = sx * Geo::kSW + 2 * (lane % (Geo::kSW / 2)), ly = sy * Geo::kSH + lane / (Geo::kSW / 2);
    const unsigned int my_strip = (1u << (16 + sx)) | (1u << sy);
    const unsigned int total = (unsigned int)stats->chunks;
    const unsigned int K = stats->chunk_size;
    const unsigned int pairs = (unsigned int)stats->pairs;
    const int e = fixed_exponent(stats->amax_bits);
    const float sc1 = pow2i(e / 2), sc2 = pow2i(e - e / 2);
    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(smem_u32(mbar + s), 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    unsigned int wcount = 0u;      // windows consumed by this CTA so far: stage = wcount % kStages, parity from wcount / kStages
    unsigned int sub = 0u;         // sub-ranges so far: mask buffer = sub & 1
    // window j of the current chunk -> stage (wbase + j) % kStages
    auto issue = [&](unsigned int wbase, unsigned int j, unsigned int r0, unsigned int r1) {
        const unsigned int s = (wbase + j) % kStages;
        const unsigned int wb = r0 + j * kWin, bytes = 32u * (min(wb + kWin, r1) - wb);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(smem_u32(mbar + s), bytes);
        bulk_copy_g2s(smem_u32(stage + 2 * kWin * s), records + 2ull * wb, bytes, smem_u32(mbar + s));
    };
    for (;;) {
        __syncthreads();
        if (warp == 0) {
            // next chunk, and the tile that holds its first record: the last tile t with bin_start[t] <= r0, found
            // by a 32-way search over bin_start (three or four rounds of 32 probes)
            unsigned int c = 0u;
            if (lane == 0) c = atomicAdd(&stats->work_counter, 1u);
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c < total) {
                const unsigned int r = c * K;
                int lo = 0, n = fp.n_tiles;
                while (n > 1) {
                    const int step = (n + 31) / 32;
                    const int t = lo + lane * step;
                    const bool le = t < lo + n && __ldg(bin_start + t) <= r;
                    const int k = __popc(__ballot_sync(0xffffffffu, le)) - 1;
                    lo += k * step;
                    n = min(step, n - k * step);
                }
                if (lane == 0) s_tile = lo;
            }
            if (lane == 0) s_chunk = c;
        }
        __syncthreads();
        const unsigned int chunk = s_chunk;
        if (chunk >= total) break;
        const unsigned int r0 = chunk * K, r1 = min(r0 + K, pairs);
        const unsigned int nwin = (r1 - r0 + kWin - 1) / kWin;
        const unsigned int wbase = wcount;
        if (threadIdx.x == 0)
            for (unsigned int j = 0; j < min(nwin, (unsigned int)kStages); ++j) issue(wbase, j, r0, r1);
        int tile = s_tile;
        unsigned int te = bin_start[tile + 1];
        bool open = false;
        float fx = 0.0f, fy = 0.0f;
        int tx0 = 0, ty0 = 0;
        f32x2 fxp = 0ull, accR = 0ull, accG = 0ull, accB = 0ull, subR = 0ull, subG = 0ull, subB = 0ull;
        unsigned int since = 0u;
        // ---- segment end: register sums and planes -> the tile's 64-bit sums in global memory
        auto flush = [&]() {
            accR = fadd2(accR, subR); accG = fadd2(accG, subG); accB = fadd2(accB, subB);
            __syncthreads();                             // all direct-path atomics of the segment have landed
            float v[6];
            upk2(accR, v[0], v[1]); upk2(accG, v[2], v[3]); upk2(accB, v[4], v[5]);
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int q = 0; q < 2; ++q) {            // this lane's own two pixels: no other thread touches them now
                    const long long f = __float2ll_rn(v[2 * c + q] * sc1 * sc2);
                    unsigned int *q0 = fb + c * kPix + ly * T + lx + q;
                    q0[0] += (unsigned int)(f & 0xffffll);
                    q0[3 * kPix] += (unsigned int)(int)(f >> 16);
                }
            __syncthreads();
            unsigned long long *out = accum + (size_t)tile * (3 * kPix);
            for (int i = threadIdx.x; i < 3 * kPix; i += kThreads) {
                const long long s = (long long)(int)fb[3 * kPix + i] * 65536ll + (long long)fb[i];
                if (s != 0ll) atomicAdd(out + i, (unsigned long long)s);
            }
        };
        for (unsigned int k = 0; k < nwin; ++k, ++wcount) {
            const unsigned int st = wcount % kStages;
            mbar_wait(smem_u32(mbar + st), (wcount / kStages) & 1u);
            const float4 *win = stage + 2 * kWin * st;
            const unsigned int wb = r0 + k * kWin, we = min(wb + kWin, r1);
            unsigned int pos = wb;
            bool first = true;
            while (pos < we) {
                if (!open) {
                    // ---- segment begin: clear the planes (each thread clears the words it read in flush) and the sums
                    for (int i = threadIdx.x; i < 6 * kPix; i += kThreads) fb[i] = 0u;
                    tx0 = (tile % fp.ntx) * T; ty0 = (tile / fp.ntx) * T;
                    fx = __fadd_rn((float)(tx0 + lx), 0.5f); fy = __fadd_rn((float)(ty0 + ly), 0.5f);
                    fxp = pk2(fx, __fadd_rn(fx, 1.0f));
                    accR = accG = accB = subR = subG = subB = 0ull;
                    since = 0u;
                    open = true;
                    __syncthreads();
                }
                const unsigned int end = min(we, te), cnt = end - pos, off = pos - wb;
                unsigned int *mask = stM + (sub & 1u) * kWin;
                // ---- decode: direct splat of boxes up to 2 x 2, strip masks for the others
                for (unsigned int i = threadIdx.x; i < ((cnt + 31u) & ~31u); i += kThreads) {
                    unsigned int touch = 0u;
                    if (i < cnt) {
                        const float4 ra = win[2 * (off + i)], rb = win[2 * (off + i) + 1];
                        const unsigned int box = __float_as_uint(rb.w);
                        const int bx0 = (int)(box & 31u), by0 = (int)((box >> 5) & 31u);
                        const int bw1 = (int)((box >> 10) & 31u), bh1 = (int)((box >> 15) & 31u);     // width - 1, height - 1
                        if (bw1 <= 1 && bh1 <= 1) {
                            const float ax = rb.x * sc1 * sc2, ay = rb.y * sc1 * sc2, az = rb.z * sc1 * sc2;
                            const float fx0 = __fadd_rn((float)(tx0 + bx0), 0.5f), fy0 = __fadd_rn((float)(ty0 + by0), 0.5f);
#pragma unroll
                            for (int q = 0; q < 4; ++q) {
                                const int qx = q & 1, qy = q >> 1;
                                if (qx <= bw1 && qy <= bh1) {
                                    const float dxf = __fsub_rn(qx ? __fadd_rn(fx0, 1.0f) : fx0, ra.x);
                                    const float dyf = __fsub_rn(qy ? __fadd_rn(fy0, 1.0f) : fy0, ra.y);
                                    const float d2 = __fmaf_rn(dxf, dxf, __fmul_rn(dyf, dyf));
                                    if (d2 <= ra.w) {
                                        const float wgt = ex2_approx(d2 * ra.z);
                                        unsigned int *q0 = fb + (by0 + qy) * T + bx0 + qx;
                                        fixed_add(q0, q0 + 3 * kPix, ax * wgt);
                                        fixed_add(q0 + kPix, q0 + 4 * kPix, ay * wgt);
                                        fixed_add(q0 + 2 * kPix, q0 + 5 * kPix, az * wgt);
                                    }
                                }
                            }
                        } else {
                            const int x1 = bx0 + bw1, y1 = by0 + bh1;
                            const unsigned int xm = (2u << (x1 / Geo::kSW)) - (1u << (bx0 / Geo::kSW));
                            const unsigned int ym = (2u << (y1 / Geo::kSH)) - (1u << (by0 / Geo::kSH));
                            touch = (xm << 16) | ym;
                        }
                    }
                    mask[i] = touch;
                }
                __syncthreads();                         // masks visible; every warp is done with the previous sub-range
                if (first && k >= 1u && threadIdx.x == 0 && k - 1u + kStages < nwin) issue(wbase, k - 1u + kStages, r0, r1);
                first = false;
                // ---- pixel owners: every warp walks the records that touch its strip (the paper's "one pixel per
                //      thread, particles in sequence", :226, with a 64-pixel warp strip and a box test in front)
                const float4 *recs = win + 2 * off;
                // compact the records that touch this warp's strip into the warp's hit list, then evaluate them two at a
                // time: the two dependent chains (LDS -> d2 -> ex2 -> FFMA2) interleave, which halves the exposed latency
                unsigned short *hl = hits + warp * kWin;
                unsigned int nh = 0u;
#pragma unroll 1
                for (unsigned int g = 0; g < cnt; g += 32) {
                    const unsigned int t = mask[g + lane];
                    const bool hit = (t & my_strip & 0xffff0000u) && (t & my_strip & 0xffffu);
                    const unsigned int m = __ballot_sync(0xffffffffu, hit);
                    if (hit) hl[nh + __popc(m & ((1u << lane) - 1u))] = (unsigned short)(g + lane);
                    nh += __popc(m);
                }
                __syncwarp();
                auto weights = [&](const float4 &A) -> f32x2 {
                    const float dyf = __fsub_rn(fy, A.y);
                    const f32x2 dx = fadd2(fxp, pk2(-A.x, -A.x));
                    const float t2 = __fmul_rn(dyf, dyf);
                    const f32x2 d2 = ffma2(dx, dx, pk2(t2, t2));
                    const f32x2 arg = fmul2(d2, pk2(A.z, A.z));
                    float d20, d21, a0, a1;
                    upk2(d2, d20, d21); upk2(arg, a0, a1);
                    const float w0 = d20 <= A.w ? ex2_approx(a0) : 0.0f;
                    const float w1 = d21 <= A.w ? ex2_approx(a1) : 0.0f;
                    return pk2(w0, w1);
                };
                unsigned int j = 0u;
#pragma unroll 1
                for (; j + 1u < nh; j += 2u) {
                    const unsigned int pr = *reinterpret_cast<const unsigned int *>(hl + j);
                    const float4 A0 = recs[2 * (pr & 0xffffu)], B0 = recs[2 * (pr & 0xffffu) + 1];
                    const float4 A1 = recs[2 * (pr >> 16)], B1 = recs[2 * (pr >> 16) + 1];
                    const f32x2 w0 = weights(A0), w1 = weights(A1);
                    subR = ffma2(pk2(B0.x, B0.x), w0, subR); subG = ffma2(pk2(B0.y, B0.y), w0, subG); subB = ffma2(pk2(B0.z, B0.z), w0, subB);
                    subR = ffma2(pk2(B1.x, B1.x), w1, subR); subG = ffma2(pk2(B1.y, B1.y), w1, subG); subB = ffma2(pk2(B1.z, B1.z), w1, subB);
                }
                if (j < nh) {
                    const unsigned int r = hl[j];
                    const float4 A0 = recs[2 * r], B0 = recs[2 * r + 1];
                    const f32x2 w0 = weights(A0);
                    subR = ffma2(pk2(B0.x, B0.x), w0, subR); subG = ffma2(pk2(B0.y, B0.y), w0, subG); subB = ffma2(pk2(B0.z, B0.z), w0, subB);
                }
                __syncwarp();                            // the list is rewritten in the next sub-range
                since += cnt;
                if (since >= (unsigned int)Cfg::kFoldRecords) {      // two-level sums: float32 stays accurate to ~1e-6
                    since = 0u;
                    accR = fadd2(accR, subR); accG = fadd2(accG, subG); accB = fadd2(accB, subB);
                    subR = subG = subB = 0ull;
                }
                pos = end;
                ++sub;
                if (pos == te) {                         // the tile's records end here
                    flush();
                    open = false;
                    if (pos < r1) { do { ++tile; te = bin_start[tile + 1]; } while (te == pos); }
                }
            }
        }
        if (open) flush();                               // the chunk ends inside a tile
    }
}

}  // namespace splotch
