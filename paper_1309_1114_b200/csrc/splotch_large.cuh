// splotch_large.cuh -- A6, the cooperative path for LARGE particles (r(p) > r_0) (sm_100a).
//
// The paper renders large particles on the CPU while the GPU works on the rest and names the
// resulting imbalance as its bottleneck for R_0 > 2 (:324).  Here they stay on the GPU: k_scatter files each LARGE
// particle under every super-tile (up to 256 x 256 px) its box touches, and k_large splits the work into items of
// (chunk of a super-tile's records) x (32 x 32-pixel block of that super-tile) that CTAs take from an atomic counter,
// so a region covered by hundreds of thousands of large discs (camera inside a halo, cfg3) is shared by many CTAs.
//   * the chunk's records stream through shared memory with bulk copies on mbarriers, as in k_splat;
//   * every thread tests two records per window against the block (box, then disc against the block's rectangle of
//     pixel centres) and sorts the survivors into two lists: discs that contain the whole block, and the others;
//   * pixel owners: a thread owns 8 horizontally adjacent pixels and keeps their sums in registers as packed pairs;
//       - block inside the disc: no clip test is needed, and the Gaussian along the row follows the recurrence
//         w(x+2) = w(x) h(x), h(x+2) = h(x) q^8 with h(x) = exp2(c (4 dx + 4)), q^8 = exp2(8 c): four ex2 per 8 pixels
//         instead of eight (round 1 was bound by MUFU.EX2, one per evaluated pixel, profiles/r1_step5_*);
//       - otherwise: the C1 inside test of every pixel (bit-exact d2, packed), one ex2 per pixel;
//   * an item ends with 64-bit fixed-point reductions into the tiles' sums in L2 (exact, commutative), the same sums
//     k_splat feeds; k_compose turns them into the float32 image.
// Blocks are 32 x 32 px whatever the tile side T is (a thread's 8-pixel run never straddles a tile).
#pragma once
#include "splotch_kernels.cuh"
#include "splotch_splat.cuh"

namespace splotch {

constexpr int kLargeThreads = 128;
constexpr int kLargeWin = 256;            // records per bulk copy; every thread tests two of them
constexpr int kLargeStages = 2;
constexpr int kLargeChunk = 4096;         // records per work item
constexpr int kLargeBlock = 32;           // block side in px
constexpr int kLargePpt = 8;              // pixels per thread (one row segment)

__global__ void __launch_bounds__(kLargeThreads)
k_large(const float4 *__restrict__ records, const unsigned int *__restrict__ bin_count, const uint2 *__restrict__ run,
        const unsigned int *__restrict__ large_off, DeviceStats *__restrict__ stats,
        unsigned long long *__restrict__ accum, const __grid_constant__ FrameParams fp)
{
    __shared__ __align__(128) float4 stage[kLargeStages][kLargeWin][2];
    __shared__ float4 sA[kLargeWin], sB[kLargeWin];
    __shared__ unsigned int sC[kLargeWin];                       // cutting discs: 2 bits per warp band (0 cut, 1 inside, 2 outside)
    __shared__ unsigned long long mbar[kLargeStages];
    __shared__ int s_cnt[kLargeThreads / 32][2];
    __shared__ unsigned int s_item;
    __shared__ int s_sup;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (stats->overflow || stats->large_pairs == 0ull) return;          // no LARGE particle in this frame
    const int n_super = fp.n_super;
    const unsigned int total = large_off[n_super];
    if (total == 0u) return;
    if (threadIdx.x == 0) {
        for (int s = 0; s < kLargeStages; ++s) mbar_init(smem_u32(mbar + s), 1u);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const int e = fixed_exponent(stats->amax_bits);
    const float sc1 = pow2i(e / 2), sc2 = pow2i(e - e / 2);
    const int bps = 1 << (fp.sshift - 5);                               // blocks per super-tile side
    const int nblk = bps * bps;
    const int T = fp.T, tmask = T - 1, kPix = T * T;
    // this thread's pixels inside the block: 8 adjacent ones of one row
    const int row = threadIdx.x >> 2, col0 = (threadIdx.x & 3) * kLargePpt;
    unsigned int wcount = 0u;
    const unsigned int slab_base_l = stats->slab_base[lane];
    uint2 myrun = make_uint2(0u, 0u);            // warp 0: lane s holds run s of the item's super-tile bin
    // window j of the current item (records [r0, r1) of the bin, counted over its runs) -> stage (wbase + j) % kLargeStages;
    // called by all lanes of warp 0: every lane copies the part of its run inside the window
    auto issue = [&](unsigned int wbase, unsigned int j, unsigned int r0, unsigned int r1) {
        const unsigned int s = (wbase + j) % kLargeStages;
        const unsigned int wb = r0 + j * kLargeWin, cnt = min(wb + kLargeWin, r1) - wb;
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        (void)gather_bin(records, myrun, slab_base_l, 2u, 2u * wb, 2u * cnt, smem_u32(&stage[s][0][0]), smem_u32(mbar + s), lane);
        if (lane == 0) mbar_expect_tx(smem_u32(mbar + s), 32u * cnt);
        __syncwarp();
    };
    for (;;) {
        __syncthreads();
        if (warp == 0) {
            // next item, and its super-tile: the last s with large_off[s] <= item, by a 32-way search
            unsigned int it = 0u;
            if (lane == 0) it = atomicAdd(&stats->large_counter, 1u);
            it = __shfl_sync(0xffffffffu, it, 0);
            if (it < total) {
                int lo = 0, n = n_super;
                while (n > 1) {
                    const int step = (n + 31) / 32;
                    const int t = lo + lane * step;
                    const bool le = t < lo + n && __ldg(large_off + t) <= it;
                    const int k = __popc(__ballot_sync(0xffffffffu, le)) - 1;
                    lo += k * step;
                    n = min(step, n - k * step);
                }
                if (lane == 0) s_sup = lo;
            }
            if (lane == 0) s_item = it;
        }
        __syncthreads();
        const unsigned int item = s_item;
        if (item >= total) break;
        const int sup = s_sup;
        const unsigned int local = item - large_off[sup];
        const unsigned int chunk = local / (unsigned int)nblk;
        const int blk = (int)(local % (unsigned int)nblk);
        // block origin inside the super-tile and on the screen (record boxes are relative to the super-tile)
        const int qx0 = (blk % bps) * kLargeBlock, qy0 = (blk / bps) * kLargeBlock;
        const int X0 = ((sup % fp.nsx) << fp.sshift) + qx0, Y0 = ((sup / fp.nsx) << fp.sshift) + qy0;
        if (X0 >= fp.W || Y0 >= fp.H) continue;                  // the super-tile hangs over the image edge
        const int qx1 = qx0 + kLargeBlock - 1, qy1 = qy0 + kLargeBlock - 1;
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
        const float cyl = __fadd_rn((float)Y0, 0.5f), cyh = __fadd_rn((float)(Y0 + kLargeBlock - 1), 0.5f);
        const float fyc = __fadd_rn((float)(Y0 + row), 0.5f);
        const float fx0 = __fadd_rn((float)(X0 + col0), 0.5f);
        f32x2 fxp[kLargePpt / 2], acc[kLargePpt / 2][3], sub[kLargePpt / 2][3];
#pragma unroll
        for (int j = 0; j < kLargePpt / 2; ++j) {
            fxp[j] = pk2(__fadd_rn((float)(X0 + col0 + 2 * j), 0.5f), __fadd_rn((float)(X0 + col0 + 2 * j + 1), 0.5f));
#pragma unroll
            for (int c = 0; c < 3; ++c) acc[j][c] = sub[j][c] = 0ull;
        }
        for (unsigned int k = 0; k < nwin; ++k, ++wcount) {
            const unsigned int st = wcount % kLargeStages;
            mbar_wait(smem_u32(mbar + st), (wcount / kLargeStages) & 1u);
            const unsigned int wb = r0 + k * kLargeWin, cntw = min(wb + kLargeWin, r1) - wb;
            // ---- test two records per thread: 0 = miss, 1 = the disc contains the block, 2 = the disc cuts the block
            float4 ra[2], rb[2];
            int kind[2];
            bool safe[2] = {false, false};
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                const unsigned int idx = threadIdx.x + t * kLargeThreads;
                kind[t] = 0;
                ra[t] = rb[t] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (idx < cntw) {
                    ra[t] = stage[st][idx][0]; rb[t] = stage[st][idx][1];
                    const unsigned int box = __float_as_uint(rb[t].w);
                    const int bx0 = (int)(box & 255u), by0 = (int)((box >> 8) & 255u);
                    const int bx1 = (int)((box >> 16) & 255u), by1 = (int)(box >> 24);
                    if (bx0 <= qx1 && bx1 >= qx0 && by0 <= qy1 && by1 >= qy0) {
                        // nearest and farthest point of the block's rectangle of pixel centres (margins cover the
                        // float32 rounding of the C1 test: a skipped block has no pixel inside, a "contained" block none outside)
                        const float ax = cxl - ra[t].x, bx = ra[t].x - cxh, ay = cyl - ra[t].y, by = ra[t].y - cyh;
                        const float nx = fmaxf(fmaxf(ax, bx), 0.0f), ny = fmaxf(fmaxf(ay, by), 0.0f);
                        const float gx = fmaxf(-ax, -bx), gy = fmaxf(-ay, -by);         // farthest: max(|cxl - px|, |cxh - px|)
                        if (fmaf(nx, nx, ny * ny) <= ra[t].w * 1.0001f) {
                            kind[t] = (fmaf(gx, gx, gy * gy) <= ra[t].w * 0.9999f && bx0 <= qx0 && bx1 >= qx1 && by0 <= qy0 && by1 >= qy1) ? 1 : 2;
                            // the recurrence is used only where its factors cannot overflow and its products cannot vanish: the
                            // largest |log2 h| over the block is -c (4 (r + 32) + 8), the weights inside the disc are at least
                            // exp2(c r^2), and a run that lies outside the disc is masked, not evaluated
                            safe[t] = -ra[t].z * (4.0f * sqrtf(ra[t].w) + 136.0f) < 120.0f && -ra[t].z * ra[t].w < 100.0f;
                            if (kind[t] == 1 && !safe[t]) kind[t] = 2;
                        }
                    }
                }
            }
            const unsigned int mi0 = __ballot_sync(0xffffffffu, kind[0] == 1), mi1 = __ballot_sync(0xffffffffu, kind[1] == 1);
            const unsigned int mb0 = __ballot_sync(0xffffffffu, kind[0] == 2), mb1 = __ballot_sync(0xffffffffu, kind[1] == 2);
            if (lane == 0) { s_cnt[warp][0] = __popc(mi0) + __popc(mi1); s_cnt[warp][1] = __popc(mb0) + __popc(mb1); }
            __syncthreads();                 // counts visible; every warp is done with the previous window's lists
            // the stage of the previous window is free now: refill it
            if (k >= 1u && warp == 0 && k - 1u + kLargeStages < nwin) issue(wbase, k - 1u + kLargeStages, r0, r1);
            int ioff = 0, boff = 0, n_in = 0, n_cut = 0;
#pragma unroll
            for (int w = 0; w < kLargeThreads / 32; ++w) {
                const int ci = s_cnt[w][0], cb = s_cnt[w][1];
                ioff += w < warp ? ci : 0; boff += w < warp ? cb : 0;
                n_in += ci; n_cut += cb;
            }
            const unsigned int lt = (1u << lane) - 1u;
#pragma unroll
            for (int t = 0; t < 2; ++t) {
                if (kind[t] == 1) {           // the list of containing discs grows from the front
                    const int pos = ioff + (t ? __popc(mi0) : 0) + __popc((t ? mi1 : mi0) & lt);
                    sA[pos] = ra[t];
                    sB[pos] = make_float4(rb[t].x, rb[t].y, rb[t].z, ex2_approx(8.0f * ra[t].z));      // q^8
                } else if (kind[t] == 2) {    // the list of cutting discs grows from the back
                    const int pos = kLargeWin - 1 - (boff + (t ? __popc(mb0) : 0) + __popc((t ? mb1 : mb0) & lt));
                    sA[pos] = ra[t];
                    sB[pos] = make_float4(rb[t].x, rb[t].y, rb[t].z, safe[t] ? ex2_approx(8.0f * ra[t].z) : -1.0f);
                    // the disc against each warp's band of 8 rows: its edge crosses a block almost as a straight line, so most
                    // bands lie wholly inside (no-test recurrence) or wholly outside (skipped); decided once per record here
                    unsigned int code = 0u;
                    const float ax = cxl - ra[t].x, bx = ra[t].x - cxh;
                    const float nx = fmaxf(fmaxf(ax, bx), 0.0f), gx = fmaxf(-ax, -bx);
#pragma unroll
                    for (int w = 0; w < kLargeThreads / 32; ++w) {
                        const float yl = cyl + (float)(8 * w), yh = yl + 7.0f;
                        const float ay = yl - ra[t].y, by = ra[t].y - yh;
                        const float ny = fmaxf(fmaxf(ay, by), 0.0f), gy = fmaxf(-ay, -by);
                        const bool out = fmaf(nx, nx, ny * ny) > ra[t].w * 1.0001f;
                        const bool in = safe[t] && fmaf(gx, gx, gy * gy) <= ra[t].w * 0.9999f;
                        code |= (out ? 2u : (in ? 1u : 0u)) << (2 * w);
                    }
                    sC[pos] = code;
                }
            }
            __syncthreads();
            // ---- discs that contain the block: recurrence along the row, no clip test
            for (int m = 0; m < n_in; ++m) {
                const float4 a = sA[m], b = sB[m];
                const float dy = fyc - a.y, dx0 = fx0 - a.x;
                const float d20 = fmaf(dx0, dx0, dy * dy);
                const float d21 = d20 + fmaf(2.0f, dx0, 1.0f);
                const float u0 = fmaf(4.0f, dx0, 4.0f);
                f32x2 P = pk2(ex2_approx(a.z * d20), ex2_approx(a.z * d21));
                f32x2 H = pk2(ex2_approx(a.z * u0), ex2_approx(a.z * (u0 + 4.0f)));
                const f32x2 Q = pk2(b.w, b.w), BR = pk2(b.x, b.x), BG = pk2(b.y, b.y), BB = pk2(b.z, b.z);
#pragma unroll
                for (int j = 0; j < kLargePpt / 2; ++j) {
                    sub[j][0] = ffma2(BR, P, sub[j][0]); sub[j][1] = ffma2(BG, P, sub[j][1]); sub[j][2] = ffma2(BB, P, sub[j][2]);
                    if (j + 1 < kLargePpt / 2) P = fmul2(P, H);
                    if (j + 2 < kLargePpt / 2) H = fmul2(H, Q);
                }
            }
            // ---- discs that cut the block: per band of 8 rows (one warp) skipped, no-test recurrence, or the C1 inside test per
            //      pixel (bit-exact d2, packed), one ex2 per pixel.  (The recurrence with a 0 / 1 mask for every pixel was
            //      measured and dropped: its extra multiplications cost more FMA-pipe time than the ex2 they save.)
            for (int m = 0; m < n_cut; ++m) {
                const unsigned int code = (sC[kLargeWin - 1 - m] >> (2 * warp)) & 3u;      // the same for all lanes of the warp
                if (code == 2u) continue;
                const float4 a = sA[kLargeWin - 1 - m], b = sB[kLargeWin - 1 - m];
                if (code == 1u) {
                    const float dy = fyc - a.y, dx0 = fx0 - a.x;
                    const float d20 = fmaf(dx0, dx0, dy * dy);
                    const float d21 = d20 + fmaf(2.0f, dx0, 1.0f);
                    const float u0 = fmaf(4.0f, dx0, 4.0f);
                    f32x2 P = pk2(ex2_approx(a.z * d20), ex2_approx(a.z * d21));
                    f32x2 H = pk2(ex2_approx(a.z * u0), ex2_approx(a.z * (u0 + 4.0f)));
                    const f32x2 Q = pk2(b.w, b.w), BR = pk2(b.x, b.x), BG = pk2(b.y, b.y), BB = pk2(b.z, b.z);
#pragma unroll
                    for (int j = 0; j < kLargePpt / 2; ++j) {
                        sub[j][0] = ffma2(BR, P, sub[j][0]); sub[j][1] = ffma2(BG, P, sub[j][1]); sub[j][2] = ffma2(BB, P, sub[j][2]);
                        if (j + 1 < kLargePpt / 2) P = fmul2(P, H);
                        if (j + 2 < kLargePpt / 2) H = fmul2(H, Q);
                    }
                    continue;
                }
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
                    sub[j][0] = ffma2(BR, Wp, sub[j][0]); sub[j][1] = ffma2(BG, Wp, sub[j][1]); sub[j][2] = ffma2(BB, Wp, sub[j][2]);
                }
            }
            if ((k & 3u) == 3u || k + 1u == nwin) {              // two-level sums: fold the sub-sums every 4 windows
#pragma unroll
                for (int j = 0; j < kLargePpt / 2; ++j)
#pragma unroll
                    for (int c = 0; c < 3; ++c) { acc[j][c] = fadd2(acc[j][c], sub[j][c]); sub[j][c] = 0ull; }
            }
        }
        // ---- the item's sums -> the tiles' 64-bit fixed-point sums
        {
            const int X = X0 + col0, Y = Y0 + row;
            const int tx = X >> fp.tshift, ty = Y >> fp.tshift;
            if (tx < fp.ntx && ty < fp.nty) {
                unsigned long long *out = accum + (size_t)(ty * fp.ntx + tx) * (3 * kPix) + (Y & tmask) * T + (X & tmask);
#pragma unroll
                for (int j = 0; j < kLargePpt / 2; ++j)
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        float v0, v1;
                        upk2(acc[j][c], v0, v1);
                        const long long f0 = __float2ll_rn(v0 * sc1 * sc2), f1 = __float2ll_rn(v1 * sc1 * sc2);
                        if (f0 != 0ll) atomicAdd(out + c * kPix + 2 * j, (unsigned long long)f0);
                        if (f1 != 0ll) atomicAdd(out + c * kPix + 2 * j + 1, (unsigned long long)f1);
                    }
            }
        }
    }
}

}  // namespace splotch
