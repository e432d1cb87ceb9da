// splotch_splat.cuh -- A5, the tile renderer for SMALL + MEDIUM records (sm_100a).
//
// The paper's medium-particle kernel (a CUDA block owns a tile in shared memory, particles are
// staged n_p at a time, one pixel per thread) and its small-particle path (:179: fragment buffer + reduce_by_key)
// redesigned for B200 as ONE persistent, warp-specialised kernel:
//   * a work item is a chunk of the virtual record order (bin after bin, see k_scan), cut into segments at tile
//     boundaries, so a heavy tile is shared by many CTAs (the load-imbalance problem of :242);
//   * a PRODUCER warp takes chunks from an atomic counter and streams their records into a ring of shared-memory
//     windows with 1-D bulk copies (cp.async.bulk, the TMA engine) that complete on mbarriers.  A bin is stored as up
//     to 32 runs, one per slab of the record array (k_layout): lane s of the producer owns run s, and every lane
//     copies the intersection of its run with the window, so gathering a window costs a handful of instructions
//     whatever the number of runs.  The producer never waits for the consumers except for a free window, and runs
//     on into the next chunk while the consumers still render the previous one;
//   * CONSUMER warps render the windows:
//       - SMALL records (16 bytes: pixel + three amplitudes) are added by one thread per record straight into the
//         tile's fixed-point planes in shared memory (native integer red.shared; no weights, no masks, no lists);
//       - MEDIUM records whose box is at most 2 x 2 pixels are splatted by the thread that decodes them, the same way;
//       - the others are evaluated by pixel owners: a warp owns a strip of the tile, a lane 2 (T = 64: 8) adjacent
//         pixels, sums live in registers as packed float32 pairs (FADD2 / FFMA2 / FMUL2), no atomics;
//   * at the end of a segment everything is added to the tile's 64-bit fixed-point sums in L2 (exact, commutative).
#pragma once
#include "splotch_kernels.cuh"

namespace splotch {

constexpr int kSplatStages = 3;
constexpr int kSplatMaxSub = 16;           // sub-ranges (runs of one bin) a window may hold
constexpr int kSplatEndChunk = 1, kSplatExit = 2;

struct SplatWin {                          // what the producer tells the consumers about a window
    int n_sub, flags;
    int bin[kSplatMaxSub];
    unsigned short off[kSplatMaxSub], cnt[kSplatMaxSub];     // first unit inside the window, records
};

template <int T> struct Splat2Cfg {
    using Base = SplatCfg<T>;
    static constexpr int kPix = Base::kPix, kConsumers = Base::kThreads, kThreads = Base::kThreads + 32;
    // 16-byte units per window: 256 MEDIUM or 512 SMALL records for the 4-warp tiles, twice that for the 16-warp ones
    // (one record per consumer thread and decode round, as many records per barrier)
    static constexpr int kWinUnits = T >= 32 ? 1024 : 512;
    static constexpr int kMaxRec = kWinUnits / 2;                    // MEDIUM records per sub-range
    static constexpr size_t kStageBytes = 16u * kWinUnits;
    static constexpr int kMinBlocks = T == 8 ? 12 : (T == 16 ? 6 : (T == 32 ? 2 : 1));     // T = 32: two 17-warp CTAs per SM need <= 60 registers
    static constexpr size_t kSmemBytes = kStageBytes * kSplatStages + sizeof(unsigned int) * (6 * kPix + 2 * kMaxRec) +
                                         sizeof(unsigned short) * kMaxRec * Base::kWarps * 2 + sizeof(SplatWin) * kSplatStages + 16 * kSplatStages;
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
__device__ __forceinline__ void mbar_arrive(unsigned int bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
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

// One warp copies units [rel0, rel0 + take) of bin `bin` (unpadded concatenation of the bin's runs) to `dst`: lane s
// holds run s = {first unit inside slab s, records}; every lane copies the part of its run inside the range.
// Returns the bin's unpadded units.  All 32 lanes must call.
__device__ __forceinline__ unsigned int gather_bin(const float4 *__restrict__ records, uint2 myrun, unsigned int slab_base_l,
                                                   unsigned int usz, unsigned int rel0, unsigned int take, unsigned int dst,
                                                   unsigned int bar, int lane)
{
    const unsigned int units = myrun.y * usz;
    unsigned int pe = units;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, pe, o);
        if (lane >= o) pe += t;
    }
    const unsigned int total = __shfl_sync(0xffffffffu, pe, 31);
    const unsigned int pb = pe - units;
    const unsigned int lo = max(pb, rel0), hi = min(pe, rel0 + take);
    if (lo < hi) bulk_copy_g2s(dst + 16u * (lo - rel0), records + slab_base_l + myrun.x + (lo - pb), 16u * (hi - lo), bar);
    return total;
}

// the producer's wait for a free window: it is usually far ahead of the consumers, so it must not take issue slots from them.
// try_wait with a suspend-time hint parks the warp in hardware until the phase completes or the time is up (a sleep-and-poll loop
// of 256 ns was still 13 % of k_splat's instructions on cfg2, profiles/r2_step1_*)
__device__ __forceinline__ void mbar_wait_relaxed(unsigned int bar, unsigned int parity)
{
    unsigned int ok;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity), "r"(20000u) : "memory");
    } while (!ok);
}

template <int T>
__global__ void __launch_bounds__(Splat2Cfg<T>::kThreads, Splat2Cfg<T>::kMinBlocks)
k_splat(const float4 *__restrict__ records, const unsigned int *__restrict__ vstart, const uint2 *__restrict__ run,
        DeviceStats *__restrict__ stats, unsigned long long *__restrict__ accum, const __grid_constant__ FrameParams fp)
{
    using Cfg = Splat2Cfg<T>;
    using Geo = SplatCfg<T>;
    constexpr int kPix = Cfg::kPix, kConsumers = Cfg::kConsumers, kMaxRec = Cfg::kMaxRec, kNP = Geo::kNP, kSplatWinUnits = Cfg::kWinUnits;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4 *stage = reinterpret_cast<float4 *>(smem_raw);                                        // [kSplatStages][kSplatWinUnits]
    unsigned int *fb = reinterpret_cast<unsigned int *>(stage + kSplatStages * kSplatWinUnits);  // lo R G B, hi R G B
    unsigned int *stM = fb + 6 * kPix;                                                           // [2][warps] lengths of the hit lists (room for 2 kMaxRec words)
    unsigned short *hits = reinterpret_cast<unsigned short *>(stM + 2 * kMaxRec);                // [2][warps][kMaxRec] per-strip hit lists, double buffered
    SplatWin *wins = reinterpret_cast<SplatWin *>(hits + 2 * kMaxRec * Geo::kWarps);
    unsigned long long *full = reinterpret_cast<unsigned long long *>(wins + kSplatStages), *empty = full + kSplatStages;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x < 2 * Geo::kWarps) stM[threadIdx.x] = 0u;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kSplatStages; ++s) { mbar_init(smem_u32(full + s), 1u); mbar_init(smem_u32(empty + s), Geo::kWarps); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const unsigned int total = (unsigned int)stats->chunks;
    const unsigned int K = stats->chunk_size;
    const unsigned int tile_units = stats->tile_units;
    if (warp == Geo::kWarps) {
        // ================================= producer warp =================================
        const unsigned int slab_base_l = stats->slab_base[lane];
        const int nb2 = 2 * fp.n_tiles;
        unsigned int it = 0u;                           // windows posted so far
        for (;;) {
            unsigned int c = 0u;
            if (lane == 0) c = atomicAdd(&stats->work_counter, 1u);
            c = __shfl_sync(0xffffffffu, c, 0);
            if (c >= total) break;
            const unsigned int v0 = c * K, v1 = min(v0 + K, tile_units);
            // the bin that holds unit v0: the last b with vstart[b] <= v0, by a 32-way search
            int bin;
            {
                int lo = 0, n = nb2;
                while (n > 1) {
                    const int step = (n + 31) / 32;
                    const int t = lo + lane * step;
                    const bool le = t < lo + n && __ldg(vstart + t) <= v0;
                    const int k = __popc(__ballot_sync(0xffffffffu, le)) - 1;
                    lo += k * step;
                    n = min(step, n - k * step);
                }
                bin = lo;
            }
            unsigned int pos = v0;
            unsigned int vs = __ldg(vstart + bin), ve = __ldg(vstart + bin + 1);
            uint2 myrun = __ldg(run + (size_t)bin * kMaxSlabs + lane);
            while (pos < v1) {
                const unsigned int st = it % kSplatStages;
                mbar_wait_relaxed(smem_u32(empty + st), ((it / kSplatStages) & 1u) ^ 1u);
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                SplatWin *wd = wins + st;
                unsigned int fill = 0u;
                int nsub = 0;
                while (pos < v1 && nsub < kSplatMaxSub) {
                    const unsigned int usz = (unsigned int)(2 - (bin & 1));
                    unsigned int room = (unsigned int)kSplatWinUnits - fill;
                    if (usz == 2u) room &= ~1u;
                    if (room == 0u) break;
                    const unsigned int rel0 = pos - vs;
                    // units of this bin inside the chunk, from rel0 on; the bin's padding unit (if any) is skipped below
                    const unsigned int want = min(min(ve, v1) - pos, room);
                    const unsigned int tu = gather_bin(records, myrun, slab_base_l, usz, rel0, want, smem_u32(stage + st * kSplatWinUnits) + 16u * fill,
                                                       smem_u32(full + st), lane);
                    const unsigned int got = rel0 < tu ? min(want, tu - rel0) : 0u;       // true units copied
                    if (got > 0u) {
                        if (lane == 0) { wd->bin[nsub] = bin; wd->off[nsub] = (unsigned short)fill; wd->cnt[nsub] = (unsigned short)(got / usz); }
                        ++nsub;
                        fill += got;
                    }
                    pos += want;
                    if (rel0 + want >= tu) pos = min(ve, v1);            // only padding is left in this bin
                    if (pos >= ve && pos < v1) {                        // next bin
                        ++bin;
                        vs = ve; ve = __ldg(vstart + bin + 1);
                        myrun = __ldg(run + (size_t)bin * kMaxSlabs + lane);
                    }
                }
                if (lane == 0) {
                    wd->n_sub = nsub;
                    wd->flags = pos >= v1 ? kSplatEndChunk : 0;
                    mbar_expect_tx(smem_u32(full + st), 16u * fill);
                }
                __syncwarp();
                ++it;
            }
        }
        // no chunk is left: tell the consumers
        const unsigned int st = it % kSplatStages;
        mbar_wait_relaxed(smem_u32(empty + st), ((it / kSplatStages) & 1u) ^ 1u);
        if (lane == 0) { wins[st].n_sub = 0; wins[st].flags = kSplatExit; mbar_arrive(smem_u32(full + st)); }
        return;
    }
    // ===================================== consumer warps =====================================
    constexpr int kLPR = Geo::kSW / (2 * kNP);          // lanes per strip row
    const int sx = warp % Geo::kStripsX, sy = warp / Geo::kStripsX;
    const int lx = sx * Geo::kSW + 2 * kNP * (lane % kLPR), ly = sy * Geo::kSH + lane / kLPR;
    const int e = fixed_exponent(stats->amax_bits);
    const float sc1 = pow2i(e / 2), sc2 = pow2i(e - e / 2);
    auto cbar = [&]() { asm volatile("bar.sync 1, %0;" :: "n"(kConsumers) : "memory"); };
    int tile = -1;                 // tile of the open segment, -1: none
    float fy = 0.0f;
    int tx0 = 0, ty0 = 0;
    f32x2 fxp[kNP], acc[kNP][3], sub[kNP][3];
    unsigned int since = 0u, nsubs = 0u;
    // ---- segment end: register sums and planes -> the tile's 64-bit sums in global memory
    auto flush = [&]() {
        cbar();                                      // all direct-path atomics of the segment have landed
#pragma unroll
        for (int p = 0; p < kNP; ++p)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                float v0, v1;
                upk2(fadd2(acc[p][c], sub[p][c]), v0, v1);
                unsigned int *q0 = fb + c * kPix + ly * T + lx + 2 * p;       // this lane's own pixels: no other thread touches them now
                const long long f0 = __float2ll_rn(v0 * sc1 * sc2), f1 = __float2ll_rn(v1 * sc1 * sc2);
                q0[0] += (unsigned int)(f0 & 0xffffll); q0[3 * kPix] += (unsigned int)(int)(f0 >> 16);
                q0[1] += (unsigned int)(f1 & 0xffffll); q0[3 * kPix + 1] += (unsigned int)(int)(f1 >> 16);
            }
        cbar();
        unsigned long long *out = accum + (size_t)tile * (3 * kPix);
        for (int i = threadIdx.x; i < 3 * kPix; i += kConsumers) {
            const long long s = (long long)(int)fb[3 * kPix + i] * 65536ll + (long long)fb[i];
            if (s != 0ll) atomicAdd(out + i, (unsigned long long)s);
        }
        tile = -1;
    };
    for (unsigned int it = 0u;; ++it) {
        const unsigned int st = it % kSplatStages;
        mbar_wait(smem_u32(full + st), (it / kSplatStages) & 1u);
        const SplatWin *wd = wins + st;
        const int n_sub = wd->n_sub, flags = wd->flags;
        if (flags & kSplatExit) break;
        const float4 *win = stage + st * kSplatWinUnits;
        for (int k = 0; k < n_sub; ++k) {
            const int bin = wd->bin[k];
            const unsigned int off = wd->off[k], cnt = wd->cnt[k];
            if (tile >= 0 && (bin >> 1) != tile) flush();
            if (tile < 0) {
                // ---- segment begin: clear the planes and the sums
                tile = bin >> 1;
                cbar();                              // every thread is done reading the planes (flush of the previous segment)
                for (int i = threadIdx.x; i < 6 * kPix; i += kConsumers) fb[i] = 0u;
                tx0 = (tile % fp.ntx) * T; ty0 = (tile / fp.ntx) * T;
                fy = __fadd_rn((float)(ty0 + ly), 0.5f);
#pragma unroll
                for (int p = 0; p < kNP; ++p) {
                    fxp[p] = pk2(__fadd_rn((float)(tx0 + lx + 2 * p), 0.5f), __fadd_rn((float)(tx0 + lx + 2 * p + 1), 0.5f));
#pragma unroll
                    for (int c = 0; c < 3; ++c) acc[p][c] = sub[p][c] = 0ull;
                }
                since = 0u;
                cbar();
            }
            if (bin & 1) {
                // ---- SMALL records: one thread per record, three fixed-point additions
                for (unsigned int i = threadIdx.x; i < cnt; i += kConsumers) {
                    const float4 r = win[off + i];
                    unsigned int *q0 = fb + (__float_as_uint(r.x) & (kPix - 1));
                    fixed_add(q0, q0 + 3 * kPix, r.y * sc1 * sc2);
                    fixed_add(q0 + kPix, q0 + 4 * kPix, r.z * sc1 * sc2);
                    fixed_add(q0 + 2 * kPix, q0 + 5 * kPix, r.w * sc1 * sc2);
                }
                continue;
            }
            // ---- MEDIUM records.  Decode: direct splat of boxes up to 2 x 2, strip masks for the others
            const float4 *recs = win + off;
            // the decoding thread appends the record to the hit list of every strip its box touches (one shared-memory atomic per strip:
            // every warp scanning a mask word per record cost 16 scans per record with 32-px tiles).  Lists and lengths are double
            // buffered: a warp that is done with this sub-range decodes the next one while others still evaluate this one
            unsigned int *cnts = stM + (nsubs & 1u) * Geo::kWarps;
            unsigned short *lists = hits + (nsubs & 1u) * (kMaxRec * Geo::kWarps);
            ++nsubs;
            for (unsigned int i = threadIdx.x; i < cnt; i += kConsumers) {
                {
                    const float4 ra = recs[2 * i], rb = recs[2 * i + 1];
                    const unsigned int box = __float_as_uint(rb.w);
                    const int bx0 = (int)(box & 63u), by0 = (int)((box >> 6) & 63u);
                    const int bw1 = (int)((box >> 12) & 63u), bh1 = (int)((box >> 18) & 63u);     // width - 1, height - 1
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
                        const int sx0 = bx0 / Geo::kSW, sx1 = (bx0 + bw1) / Geo::kSW, sy0 = by0 / Geo::kSH, sy1 = (by0 + bh1) / Geo::kSH;
                        for (int yy = sy0; yy <= sy1; ++yy)
                            for (int xx = sx0; xx <= sx1; ++xx) {
                                const int wq = yy * Geo::kStripsX + xx;
                                lists[wq * kMaxRec + atomicAdd(&cnts[wq], 1u)] = (unsigned short)i;
                            }
                    }
                }
            }
            cbar();                                  // lists visible; every warp is done with the sub-range before the previous one
            // ---- pixel owners: every warp compacts the records that touch its strip into its hit list (the paper's "one
            //      pixel per thread, particles in sequence", :226, with a warp strip and a box test in front), then evaluates
            //      them two at a time: the two dependent chains (LDS -> d2 -> ex2 -> FFMA2) interleave
            const unsigned short *hl = lists + warp * kMaxRec;
            const unsigned int nh = cnts[warp];
            auto eval = [&](unsigned int r) {
                const float4 A = recs[2 * r], B = recs[2 * r + 1];
                const float dyf = __fsub_rn(fy, A.y);
                const float t2 = __fmul_rn(dyf, dyf);
                const f32x2 NX = pk2(-A.x, -A.x), T2 = pk2(t2, t2), C = pk2(A.z, A.z);
                const f32x2 BR = pk2(B.x, B.x), BG = pk2(B.y, B.y), BB = pk2(B.z, B.z);
#pragma unroll
                for (int p = 0; p < kNP; ++p) {
                    const f32x2 dx = fadd2(fxp[p], NX);
                    const f32x2 d2 = ffma2(dx, dx, T2);
                    const f32x2 arg = fmul2(d2, C);
                    float d20, d21, a0, a1;
                    upk2(d2, d20, d21); upk2(arg, a0, a1);
                    const float w0 = d20 <= A.w ? ex2_approx(a0) : 0.0f;
                    const float w1 = d21 <= A.w ? ex2_approx(a1) : 0.0f;
                    const f32x2 W = pk2(w0, w1);
                    sub[p][0] = ffma2(BR, W, sub[p][0]); sub[p][1] = ffma2(BG, W, sub[p][1]); sub[p][2] = ffma2(BB, W, sub[p][2]);
                }
            };
            unsigned int j = 0u;
#pragma unroll 1
            for (; j + 3u < nh; j += 4u) {           // four hits per round: one 64-bit read of the list, four independent chains
                const uint2 pr = *reinterpret_cast<const uint2 *>(hl + j);
                eval(pr.x & 0xffffu); eval(pr.x >> 16); eval(pr.y & 0xffffu); eval(pr.y >> 16);
            }
            for (; j < nh; ++j) eval(hl[j]);
            __syncwarp();
            if (lane == 0) cnts[warp] = 0u;          // this buffer is filled again in the sub-range after next
            since += cnt;
            if (since >= 1024u) {                    // two-level sums: float32 stays accurate to ~1e-6
                since = 0u;
#pragma unroll
                for (int p = 0; p < kNP; ++p)
#pragma unroll
                    for (int c = 0; c < 3; ++c) { acc[p][c] = fadd2(acc[p][c], sub[p][c]); sub[p][c] = 0ull; }
            }
        }
        if ((flags & kSplatEndChunk) && tile >= 0) flush();      // the chunk ends inside a tile
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(empty + st));        // this warp is done with the window
    }
}

}  // namespace splotch
