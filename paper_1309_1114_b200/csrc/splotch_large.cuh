// splotch_large.cuh -- A6, the cooperative path for LARGE particles (r(p) > r_0) (sm_100a).
//
// The paper renders large particles on the CPU while the GPU works on the rest and names the
// resulting imbalance as its bottleneck for R_0 > 2 (:324).  Here they stay on the GPU: k_scatter files each LARGE
// particle under every super-tile (128 x 128 px) its box touches, and k_large splits the work into items of
// (chunk of a super-tile's records) x (32 x 32-pixel block of that super-tile) that CTAs take from an atomic counter,
// so a region covered by hundreds of thousands of large discs (camera inside a halo, cfg3) is shared by many CTAs.
// With 32-px tiles the same kernel renders the MEDIUM discs wider than kRouteRadius: they sit in a third bin of their tile
// (splotch_kernels.cuh), a region of one block, the tile itself.
//   * the chunk's records stream through shared memory with bulk copies on mbarriers, as in k_splat;
//   * every thread tests two records per window against the block's four bands of 8 rows x 32 pixels and files the record
//     in up to two lists: bands that lie wholly inside the clip disc, bands the edge of the disc crosses (with one index list
//     per band, so a warp meets only the records that cross its band);
//   * bands inside the disc: no pixel is clipped and the Gaussian is separable, exp2(c d^2) = exp2(c dx^2) exp2(c dy^2), so
//     the sum over the records is a dense contraction D[(colour, y)][x] = sum_p A[(colour, y)][p] B[p][x] with
//     A = a_colour exp2(c dy^2) (zero in the rows of the record's other bands), B = exp2(c dx^2).  It runs on the
//     5th-generation tensor cores: tcgen05.mma kind::tf32, M = 128 (three colours x 32 rows), N = 32, K = 8 records per
//     instruction, accumulator in tensor memory.  TF32 keeps 10 mantissa bits (the hardware truncates), so every float32
//     operand is split into a high and a low part and three products are added (hi hi + hi lo + lo hi: relative error 2^-21).
//     A is written straight to tensor memory by the lane that owns the row (tcgen05.st), B to shared memory (K-major core
//     matrices, no swizzle), in groups of 16 records with two operand buffers; tcgen05.commit on an mbarrier frees a
//     buffer.  The tensor cores add with truncation (measured: -1.7e-8 relative per accumulated record), so an accumulator
//     takes 64 records, then the other one takes over and the first is folded into float32 second-level sums;
//   * bands the edge crosses: pixel owners (a thread owns 8 adjacent pixels of a row, sums in registers as packed pairs)
//     evaluate the C1 inside test of every pixel (bit-exact packed d2), one ex2 per pixel inside;
//   * sums go to the tiles' 64-bit fixed-point sums in L2 (exact, commutative), the same sums k_splat feeds; k_compose
//     turns them into the float32 image.
// Blocks are 32 x 32 px whatever the tile side T is.  Measured on cfg3 (9.5e11 LARGE fragments): round 1 397 ms (one ex2 per
// pixel), row recurrence 296 ms, tensor-core bands 282 ms, 128-px super-tiles 245 ms; with the wide MEDIUM discs (1.05e12
// fragments) 292 ms, per-band lists 274 ms, padded list and items of 8192 records 266 ms, per-pixel loop unrolled four times 253 ms.
#pragma once
#include "splotch_kernels.cuh"
#include "splotch_splat.cuh"

namespace splotch {

constexpr int kLargeThreads = 128;
constexpr int kLargeWin = 256;            // records per bulk copy; every thread tests two of them
constexpr int kLargeStages = 2;
constexpr int kLargeChunk = 8192;         // records per work item
constexpr int kLargeBlock = 32;           // block side in px
constexpr int kLargePpt = 8;              // pixels per thread (one row segment) on the cutting-disc path
constexpr int kGemmGroup = 16;            // records per operand buffer: two K-steps of 8 (tcgen05.mma kind::tf32 has K = 8)
constexpr int kGemmSpan = 64;             // records accumulated in tensor memory before the sums are folded into registers
constexpr unsigned int kLargeTmemCols = 128;   // D0, D1 (32 columns each), A0, A1 (two K-steps x (8 hi + 8 lo) columns each)

// ---- tcgen05 (5th-generation tensor cores, tensor memory): the few PTX forms k_large needs -----------------------
// Shared-memory matrix descriptor of a K-major operand without swizzle: core matrices of 8 rows x 16 bytes (4 tf32),
// the two core matrices of a K-step 128 bytes apart (leading byte offset), groups of 8 rows 256 bytes apart (stride byte
// offset); bits 46-47 = 1 (sm_100 descriptor version).
__device__ __forceinline__ unsigned long long umma_desc_kmajor(unsigned int saddr)
{
    return (unsigned long long)((saddr & 0x3ffffu) >> 4) | ((unsigned long long)(128u >> 4) << 16) | ((unsigned long long)(256u >> 4) << 32) | (1ull << 46);
}
// instruction descriptor: D = F32, A = B = TF32, both K-major, N = 32, M = 128
constexpr unsigned int kUmmaIdesc = (1u << 4) | (2u << 7) | (2u << 10) | ((32u >> 3) << 17) | ((128u >> 4) << 24);

// D[128 x 32] (+)= A[128 x 8] B[8 x 32]: A in tensor memory (lane = row, one 32-bit column per k), B in shared memory
__device__ __forceinline__ void umma_tf32_ts(unsigned int d_tmem, unsigned int a_tmem, unsigned long long b_desc, unsigned int accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
                 :: "r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(kUmmaIdesc), "r"(accumulate) : "memory");
}
// the mbarrier receives one arrival when every tcgen05.mma issued so far by this thread has completed
__device__ __forceinline__ void umma_commit(unsigned int bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// 16 consecutive 32-bit columns of this thread's lane
__device__ __forceinline__ void tmem_st16(unsigned int addr, const unsigned int (&v)[16])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
                 :: "r"(addr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
                    "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void tmem_ld16(unsigned int addr, unsigned int (&v)[16])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
                   "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]) : "r"(addr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// shared memory of k_large (dynamic: more than the 48 KB a kernel may declare statically)
struct LargeSmem {
    float4 stage[kLargeStages][kLargeWin][2];      // records of two windows (bulk copies)
    float  bop[2][2][2][256];                      // B operand: [buffer][K-step][hi, lo][(x / 8, k / 4, x % 8, k % 4)]
    float  acc2[32][96];                           // second-level sums of the tensor-core path: [x][(colour, y)], threads of warps 0-2
    float4 gA[kLargeWin + kGemmGroup], gB[kLargeWin + kGemmGroup];   // tensor-core list (+ padding to whole groups): {px, py, c, r2} {a_R, a_G, a_B, row-band mask}
    float4 cA[kLargeWin], cB[kLargeWin];           // per-pixel list
    unsigned char clist[kLargeThreads / 32][kLargeWin];   // per band (warp): the entries of the per-pixel list it evaluates
    unsigned int ccnt[kLargeThreads / 32];
    unsigned long long mbar[kLargeStages], gbar[2];
    int cnt[kLargeThreads / 32][2];
    unsigned int item, tmem;
    int sup;
};

__global__ void __launch_bounds__(kLargeThreads, 4)
k_large(const float4 *__restrict__ records, const unsigned int *__restrict__ bin_count, const uint2 *__restrict__ run,
        const unsigned int *__restrict__ large_off, DeviceStats *__restrict__ stats,
        unsigned long long *__restrict__ accum, const __grid_constant__ FrameParams fp)
{
    extern __shared__ __align__(1024) unsigned char large_smem_raw[];
    LargeSmem &S = *reinterpret_cast<LargeSmem *>(large_smem_raw);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (stats->overflow) return;
    // regions: the super-tiles (LARGE records, blocks of 32 x 32 px), then, with 32-px tiles, the tiles' bins of wide MEDIUM discs (the
    // tile is the one block); record boxes are relative to the region's origin in both
    const int n_super = fp.n_super, n_reg = fp.n_super + fp.n_big;
    const unsigned int total = large_off[n_reg];
    if (total == 0u) return;                                             // nothing for this kernel in this frame
    if (threadIdx.x == 0) {
        for (int s = 0; s < kLargeStages; ++s) mbar_init(smem_u32(S.mbar + s), 1u);
        mbar_init(smem_u32(S.gbar + 0), 1u); mbar_init(smem_u32(S.gbar + 1), 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {                 // tensor memory of this CTA (at most four CTAs per SM: 4 x 128 of the SM's 512 columns)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&S.tmem)), "n"(kLargeTmemCols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (warp < 3) {
#pragma unroll
        for (int j = 0; j < 32; ++j) S.acc2[j][threadIdx.x] = 0.0f;
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const unsigned int tmem = S.tmem;
    const unsigned int tlane = tmem + ((unsigned int)(warp * 32) << 16);     // this warp's quarter of the 128 lanes
    const int e = fixed_exponent(stats->amax_bits);
    const float sc1 = pow2i(e / 2), sc2 = pow2i(e - e / 2);
    const int bps = 1 << (fp.sshift - 5);                               // blocks per super-tile side
    const int nblk = bps * bps;
    const int T = fp.T, tmask = T - 1, kPix = T * T;
    // this thread's pixels inside the block on the per-pixel path: 8 adjacent ones of one row
    const int row = threadIdx.x >> 2, col0 = (threadIdx.x & 3) * kLargePpt;
    unsigned int wcount = 0u;
    unsigned int g_issued0 = 0u, g_issued1 = 0u, g_waited0 = 0u, g_waited1 = 0u;   // operand buffers: commits issued / phases seen (the same in every thread)
    unsigned int ngroups = 0u;
    const unsigned int slab_base_l = stats->slab_base[lane];
    uint2 myrun = make_uint2(0u, 0u);            // warp 0: lane s holds run s of the item's super-tile bin
    // window j of the current item (records [r0, r1) of the bin, counted over its runs) -> stage (wbase + j) % kLargeStages;
    // called by all lanes of warp 0: every lane copies the part of its run inside the window
    auto issue = [&](unsigned int wbase, unsigned int j, unsigned int r0, unsigned int r1) {
        const unsigned int s = (wbase + j) % kLargeStages;
        const unsigned int wb = r0 + j * kLargeWin, cnt = min(wb + kLargeWin, r1) - wb;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        (void)gather_bin(records, myrun, slab_base_l, 2u, 2u * wb, 2u * cnt, smem_u32(&S.stage[s][0][0]), smem_u32(S.mbar + s), lane);
        if (lane == 0) mbar_expect_tx(smem_u32(S.mbar + s), 32u * cnt);
        __syncwarp();
    };
    auto wait_buffer = [&](int b) {              // every tcgen05.mma that reads operand buffer b has completed
        if (b == 0) while (g_waited0 < g_issued0) { mbar_wait(smem_u32(S.gbar + 0), g_waited0 & 1u); ++g_waited0; }
        else        while (g_waited1 < g_issued1) { mbar_wait(smem_u32(S.gbar + 1), g_waited1 & 1u); ++g_waited1; }
    };
    // tensor-memory accumulator d -> second-level sums (a thread touches only its own column of acc2: no conflicts, no synchronisation)
    auto fold = [&](int d) {
        if (warp < 3) {
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                unsigned int v[16];
                tmem_ld16(tlane + (unsigned int)(d * 32 + half * 16), v);
#pragma unroll
                for (int j = 0; j < 16; ++j) S.acc2[half * 16 + j][threadIdx.x] += __uint_as_float(v[j]);
            }
        }
    };
    for (;;) {
        __syncthreads();
        if (warp == 0) {
            // next item, and its super-tile: the last s with large_off[s] <= item, by a 32-way search
            unsigned int it = 0u;
            if (lane == 0) it = atomicAdd(&stats->large_counter, 1u);
            it = __shfl_sync(0xffffffffu, it, 0);
            if (it < total) {
                int lo = 0, n = n_reg;
                while (n > 1) {
                    const int step = (n + 31) / 32;
                    const int t = lo + lane * step;
                    const bool le = t < lo + n && __ldg(large_off + t) <= it;
                    const int k = __popc(__ballot_sync(0xffffffffu, le)) - 1;
                    lo += k * step;
                    n = min(step, n - k * step);
                }
                if (lane == 0) S.sup = lo;
            }
            if (lane == 0) S.item = it;
        }
        __syncthreads();
        const unsigned int item = S.item;
        if (item >= total) break;
        const int sup = S.sup;
        const unsigned int local = item - large_off[sup];
        const bool in_tile = sup >= n_super;                       // region = a tile (wide MEDIUM discs): one block, the tile itself
        const unsigned int chunk = in_tile ? local : local / (unsigned int)nblk;
        const int blk = in_tile ? 0 : (int)(local % (unsigned int)nblk);
        // block origin inside the region and on the screen
        const int qx0 = (blk % bps) * kLargeBlock, qy0 = (blk / bps) * kLargeBlock;
        const int X0 = in_tile ? ((sup - n_super) % fp.ntx) << fp.tshift : ((sup % fp.nsx) << fp.sshift) + qx0;
        const int Y0 = in_tile ? ((sup - n_super) / fp.ntx) << fp.tshift : ((sup / fp.nsx) << fp.sshift) + qy0;
        if (X0 >= fp.W || Y0 >= fp.H) continue;                  // the super-tile hangs over the image edge
        const int qx1 = qx0 + kLargeBlock - 1;
        const unsigned int le = bin_count[2 * fp.n_tiles + sup];              // records of the super-tile's bin
        const unsigned int r0 = chunk * kLargeChunk, r1 = min(r0 + kLargeChunk, le);
        const unsigned int nwin = (r1 - r0 + kLargeWin - 1) / kLargeWin;
        const unsigned int wbase = wcount;
        if (warp == 0) {
            myrun = __ldg(run + (size_t)(2 * fp.n_tiles + sup) * kMaxSlabs + lane);
            for (unsigned int j = 0; j < min(nwin, (unsigned int)kLargeStages); ++j) issue(wbase, j, r0, r1);
        }
        // centres of the block's corner pixels
        const float cxl = __fadd_rn((float)X0, 0.5f), cxh = __fadd_rn((float)(X0 + kLargeBlock - 1), 0.5f);
        const float cyl = __fadd_rn((float)Y0, 0.5f);
        const float fyc = __fadd_rn((float)(Y0 + row), 0.5f);
        // operand rows of this thread: warps 0-2 produce A row (colour = warp, y = lane), warp 3 produces B (x = 8 j + lane / 4)
        const float fyg = __fadd_rn((float)(Y0 + lane), 0.5f), fxg = __fadd_rn((float)(X0 + (lane >> 2)), 0.5f);
        f32x2 fxp[kLargePpt / 2], sub[kLargePpt / 2][3];
#pragma unroll
        for (int j = 0; j < kLargePpt / 2; ++j) {
            fxp[j] = pk2(__fadd_rn((float)(X0 + col0 + 2 * j), 0.5f), __fadd_rn((float)(X0 + col0 + 2 * j + 1), 0.5f));
#pragma unroll
            for (int c = 0; c < 3; ++c) sub[j][c] = 0ull;
        }
        // the per-pixel sums of this thread -> the tiles' 64-bit fixed-point sums (every 1024 records: float32 stays accurate)
        auto flush_sub = [&]() {
            const int X = X0 + col0, Y = Y0 + row;
            const int tx = X >> fp.tshift, ty = Y >> fp.tshift;
            if (tx < fp.ntx && ty < fp.nty) {
                unsigned long long *out = accum + (size_t)(ty * fp.ntx + tx) * (3 * kPix) + (Y & tmask) * T + (X & tmask);
#pragma unroll
                for (int j = 0; j < kLargePpt / 2; ++j)
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        float v0, v1;
                        upk2(sub[j][c], v0, v1);
                        const long long f0 = __float2ll_rn(v0 * sc1 * sc2), f1 = __float2ll_rn(v1 * sc1 * sc2);
                        if (f0 != 0ll) atomicAdd(out + c * kPix + 2 * j, (unsigned long long)f0);
                        if (f1 != 0ll) atomicAdd(out + c * kPix + 2 * j + 1, (unsigned long long)f1);
                    }
            }
#pragma unroll
            for (int j = 0; j < kLargePpt / 2; ++j)
#pragma unroll
                for (int c = 0; c < 3; ++c) sub[j][c] = 0ull;
        };
        int dcur = 0;                            // tensor-memory accumulator of the open span
        unsigned int span = 0u;                  // records in it
        bool dirty0 = false, dirty1 = false;     // accumulator holds sums that are not in acc2 yet
        bool any_sub = false;
        for (unsigned int k = 0; k < nwin; ++k, ++wcount) {
            const unsigned int st = wcount % kLargeStages;
            mbar_wait(smem_u32(S.mbar + st), (wcount / kLargeStages) & 1u);
            const unsigned int wb = r0 + k * kLargeWin, cntw = min(wb + kLargeWin, r1) - wb;
            // ---- test two records per thread against the block, band of 8 rows by band: gmask = bands whose 8 x 32 pixels all lie
            //      inside the clip disc (tensor-core path), pmask = bands the disc's edge crosses (per-pixel path); the others are missed
            float4 ra[2], rb[2];
            unsigned int gmask[2] = {0u, 0u}, pmask[2] = {0u, 0u};
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const unsigned int idx = threadIdx.x + t * kLargeThreads;
                ra[t] = rb[t] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (idx < cntw) {
                    ra[t] = S.stage[st][idx][0]; rb[t] = S.stage[st][idx][1];
                    const unsigned int box = __float_as_uint(rb[t].w);
                    const int bx0 = (int)(box & 255u), by0 = (int)((box >> 8) & 255u);
                    const int bx1 = (int)((box >> 16) & 255u), by1 = (int)(box >> 24);
                    if (bx0 <= qx1 && bx1 >= qx0 && by0 <= qy0 + kLargeBlock - 1 && by1 >= qy0) {
                        // nearest and farthest point of a band's rectangle of pixel centres (margins cover the float32 rounding of the
                        // C1 test: a missed band has no pixel inside, a band on the tensor-core path none outside; there every weight
                        // is at least exp2(c r^2) >= e^-chi^2, so neither factor of the separable weight can vanish)
                        const float ax = cxl - ra[t].x, bx = ra[t].x - cxh;
                        const float nx = fmaxf(fmaxf(ax, bx), 0.0f), gx = fmaxf(-ax, -bx);
                        const bool xin = bx0 <= qx0 && bx1 >= qx1;
#pragma unroll
                        for (int w = 0; w < 4; ++w) {
                            const float yl = cyl + (float)(8 * w), yh = yl + 7.0f;
                            const float ay = yl - ra[t].y, by = ra[t].y - yh;
                            const float ny = fmaxf(fmaxf(ay, by), 0.0f), gy = fmaxf(-ay, -by);
                            const bool hit = fmaf(nx, nx, ny * ny) <= ra[t].w * 1.0001f && by0 <= qy0 + 8 * w + 7 && by1 >= qy0 + 8 * w;
                            const bool in = fmaf(gx, gx, gy * gy) <= ra[t].w * 0.9999f && xin && by0 <= qy0 + 8 * w && by1 >= qy0 + 8 * w + 7;
                            gmask[t] |= (hit && in) ? (1u << w) : 0u;
                            pmask[t] |= (hit && !in) ? (1u << w) : 0u;
                        }
                    }
                }
            }
            const unsigned int mi0 = __ballot_sync(0xffffffffu, gmask[0] != 0u), mi1 = __ballot_sync(0xffffffffu, gmask[1] != 0u);
            const unsigned int mb0 = __ballot_sync(0xffffffffu, pmask[0] != 0u), mb1 = __ballot_sync(0xffffffffu, pmask[1] != 0u);
            if (lane == 0) { S.cnt[warp][0] = __popc(mi0) + __popc(mi1); S.cnt[warp][1] = __popc(mb0) + __popc(mb1); S.ccnt[warp] = 0u; }
            __syncthreads();                 // counts visible; every warp is done with the previous window's lists
            // the stage of the previous window is free now: refill it
            if (k >= 1u && warp == 0 && k - 1u + kLargeStages < nwin) issue(wbase, k - 1u + kLargeStages, r0, r1);
            int ioff = 0, boff = 0, n_in = 0, n_cut = 0;
#pragma unroll
            for (int w = 0; w < kLargeThreads / 32; ++w) {
                const int ci = S.cnt[w][0], cb = S.cnt[w][1];
                ioff += w < warp ? ci : 0; boff += w < warp ? cb : 0;
                n_in += ci; n_cut += cb;
            }
            const unsigned int lt = (1u << lane) - 1u;
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                if (gmask[t]) {
                    const int pos = ioff + (t ? __popc(mi0) : 0) + __popc((t ? mi1 : mi0) & lt);
                    S.gA[pos] = ra[t];
                    S.gB[pos] = make_float4(rb[t].x, rb[t].y, rb[t].z, __uint_as_float(gmask[t]));
                }
                if (pmask[t]) {
                    const int pos = boff + (t ? __popc(mb0) : 0) + __popc((t ? mb1 : mb0) & lt);
                    S.cA[pos] = ra[t];
                    S.cB[pos] = rb[t];
#pragma unroll
                    for (int w = 0; w < kLargeThreads / 32; ++w)         // the bands (warps) that evaluate it: one index list per band
                        if ((pmask[t] >> w) & 1u) S.clist[w][atomicAdd(&S.ccnt[w], 1u)] = (unsigned char)pos;
                }
            }
            if ((int)threadIdx.x < ((kGemmGroup - (n_in & (kGemmGroup - 1))) & (kGemmGroup - 1))) {
                // the tensor-core list is padded to whole groups with records that add nothing (amplitudes 0, no rows; weights exp2(0) = 1)
                S.gA[n_in + threadIdx.x] = make_float4(0.0f, 0.0f, 0.0f, 1.0f);
                S.gB[n_in + threadIdx.x] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            }
            __syncthreads();
            // ---- bands that lie inside their disc: the sum over them is a dense contraction, D[(colour, y)][x] = sum_p A[(colour, y)][p] B[p][x]
            //      with A = a_colour exp2(c dy^2) (0 in the rows of the other bands) and B = exp2(c dx^2): the Gaussian is separable and no pixel
            //      of these rows is clipped.  It runs on the tensor cores as three TF32 products of the operands' high and low parts (hi hi +
            //      hi lo + lo hi; the hardware truncates operands to 10 mantissa bits, so hi = the value itself and lo = value - truncated
            //      value): A goes to tensor memory (every lane writes its own row), B to shared memory, groups of 16 records, two buffers.
            for (int g0 = 0; g0 < n_in; g0 += kGemmGroup, ++ngroups) {
                const int buf = (int)(ngroups & 1u);
                wait_buffer(buf);                                   // the products that read this buffer two groups ago are done
                tc_fence_after();
                if (warp < 3) {
#pragma unroll
                    for (int ks = 0; ks < 2; ++ks) {
                        unsigned int va[16];
#pragma unroll
                        for (int q = 0; q < 8; ++q) {
                            const int idx = g0 + ks * 8 + q;
                            const float4 a = S.gA[idx];
                            const float amp = reinterpret_cast<const float *>(&S.gB[idx])[warp];
                            const unsigned int rows = __float_as_uint(S.gB[idx].w);
                            const float dy = fyg - a.y;
                            float v = amp * ex2_approx(a.z * dy * dy);
                            v = ((rows >> (lane >> 3)) & 1u) ? v : 0.0f;
                            va[q] = __float_as_uint(v);
                            va[8 + q] = __float_as_uint(v - __uint_as_float(__float_as_uint(v) & 0xffffe000u));
                        }
                        tmem_st16(tlane + (unsigned int)(64 + buf * 32 + ks * 16), va);
                    }
                    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
                } else {
#pragma unroll
                    for (int ks = 0; ks < 2; ++ks)
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const int idx = g0 + ks * 8 + 4 * h + (lane & 3);
                            const float4 a = S.gA[idx];
#pragma unroll
                            for (int j = 0; j < 4; ++j) {
                                const float dx = (fxg + (float)(8 * j)) - a.x;
                                const float w = ex2_approx(a.z * dx * dx);
                                S.bop[buf][ks][0][(j * 2 + h) * 32 + lane] = w;
                                S.bop[buf][ks][1][(j * 2 + h) * 32 + lane] = w - __uint_as_float(__float_as_uint(w) & 0xffffe000u);
                            }
                        }
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                }
                tc_fence_before();
                __syncthreads();
                if (threadIdx.x == 0) {
                    tc_fence_after();
                    const unsigned int d = tmem + (unsigned int)(dcur * 32);
#pragma unroll
                    for (int ks = 0; ks < 2; ++ks) {
                        if (g0 + ks * 8 < n_in) {
                            const unsigned int ah = tmem + (unsigned int)(64 + buf * 32 + ks * 16);
                            const unsigned long long bh = umma_desc_kmajor(smem_u32(&S.bop[buf][ks][0][0])), bl = umma_desc_kmajor(smem_u32(&S.bop[buf][ks][1][0]));
                            umma_tf32_ts(d, ah, bh, (span > 0u || ks > 0) ? 1u : 0u);
                            umma_tf32_ts(d, ah, bl, 1u);
                            umma_tf32_ts(d, ah + 8u, bh, 1u);
                        }
                    }
                    umma_commit(smem_u32(S.gbar + buf));
                }
                if (buf == 0) ++g_issued0; else ++g_issued1;
                if (dcur == 0) dirty0 = true; else dirty1 = true;
                span += (unsigned int)min(kGemmGroup, n_in - g0);
                if (span >= (unsigned int)kGemmSpan) {
                    // the tensor cores add every product to the running sum with truncation: spans stay short (bias ~ 1.7e-8 per record),
                    // the other accumulator takes the next span, and what it still holds (complete long ago) is folded first
                    dcur ^= 1; span = 0u;
                    if (dcur == 0 && dirty0) { fold(0); dirty0 = false; }
                    if (dcur == 1 && dirty1) { fold(1); dirty1 = false; }
                }
            }
            // ---- bands the edge of the disc crosses: the C1 inside test of every pixel (bit-exact d2, packed), one ex2 per pixel
            //      inside.  (A row recurrence with a 0 / 1 mask per pixel was measured and dropped: its extra multiplications
            //      cost more FMA-pipe time than the ex2 they save.)
            const unsigned int n_mine = S.ccnt[warp];
            const unsigned char *pl = S.clist[warp];
#pragma unroll 4
            for (unsigned int m = 0; m < n_mine; ++m) {
                const unsigned int idx = pl[m];                      // the same for all lanes of the warp
                const float4 a = S.cA[idx], b = S.cB[idx];
                const float dyf = __fsub_rn(fyc, a.y);
                const float t2 = __fmul_rn(dyf, dyf);
                const f32x2 T2 = pk2(t2, t2), NX = pk2(-a.x, -a.x), C = pk2(a.z, a.z);
                const f32x2 BR = pk2(b.x, b.x), BG = pk2(b.y, b.y), BB = pk2(b.z, b.z);
#pragma unroll
                for (int j = 0; j < kLargePpt / 2; ++j) {
                    const f32x2 dx = fadd2(fxp[j], NX);
                    const f32x2 d2 = ffma2(dx, dx, T2);
                    const f32x2 arg = fmul2(d2, C);
                    float d2a, d2b, aa, ab;
                    upk2(d2, d2a, d2b); upk2(arg, aa, ab);
                    const float wa = d2a <= a.w ? ex2_approx(aa) : 0.0f;
                    const float wb2 = d2b <= a.w ? ex2_approx(ab) : 0.0f;
                    const f32x2 Wp = pk2(wa, wb2);
                    ffma2_acc(sub[j][0], BR, Wp); ffma2_acc(sub[j][1], BG, Wp); ffma2_acc(sub[j][2], BB, Wp);
                }
            }
            any_sub = any_sub || n_cut > 0;
            if (any_sub && ((k & 3u) == 3u || k + 1u == nwin)) { flush_sub(); any_sub = false; }
        }
        // ---- the tensor-core sums of the item -> the tiles' 64-bit fixed-point sums
        if (dirty0 || dirty1) {                  // wait for the last products, fold what the accumulators still hold
            wait_buffer(0); wait_buffer(1);
            tc_fence_after();
            if (dirty0) fold(0);
            if (dirty1) fold(1);
            if (warp < 3) {
                const int Y = Y0 + lane, ty = Y >> fp.tshift;
#pragma unroll
                for (int j = 0; j < 32; ++j) {
                    const int X = X0 + j, tx = X >> fp.tshift;
                    const long long f = __float2ll_rn(S.acc2[j][threadIdx.x] * sc1 * sc2);
                    S.acc2[j][threadIdx.x] = 0.0f;
                    if (f != 0ll && tx < fp.ntx && ty < fp.nty)
                        atomicAdd(accum + (size_t)(ty * fp.ntx + tx) * (3 * kPix) + warp * kPix + (Y & tmask) * T + (X & tmask), (unsigned long long)f);
                }
            }
        }
    }
    // every product has completed (each item waits for its own); give the tensor memory back
    tc_fence_before();
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem), "n"(kLargeTmemCols) : "memory");
}

}  // namespace splotch
