// splotch_large.cuh -- A6, the cooperative path for LARGE particles (r(p) > r_0), and A8, the epilogue (sm_100a).
//
// The paper renders large particles on the CPU while the GPU works on the rest and names the
// resulting imbalance as its bottleneck for R_0 > 2 (:324).  Here they stay on the GPU: k_scatter files each LARGE
// particle under every 8 x 8-tile super-tile its box touches, and k_large splits the work into (chunk of a super-tile's
// records) x (tile of that super-tile) items that CTAs take from an atomic counter, so a tile covered by hundreds of
// thousands of large discs (camera inside a halo, cfg3) is shared by many CTAs instead of serialising one
// (the first version gave every tile to one CTA: 494 ms for cfg3, 58 % of the issue slots, profiles/r1_step4_*).
//   * the chunk's records stream through shared memory with bulk copies on mbarriers, as in k_splat;
//   * every thread tests one record's box against the tile; survivors are compacted in order (deterministic sums);
//   * pixel owners: a thread owns kPpt horizontally adjacent pixels, every pixel of a large disc is a useful lane;
//   * an item ends with 64-bit fixed-point reductions into the tile's sums in L2 (exact, commutative), the same sums
//     k_splat feeds; k_compose turns them into the float32 image.
#pragma once
#include "splotch_kernels.cuh"
#include "splotch_splat.cuh"

namespace splotch {

constexpr int kLargeThreads = 256;
constexpr int kLargeWin = 256;            // records per bulk copy
constexpr int kLargeStages = 2;
constexpr int kLargeChunk = 4096;         // records per work item
constexpr int kMaxSuper = 1024;           // super-tiles an image can have (the per-CTA histograms of k_count bound it)

template <int T>
__global__ void __launch_bounds__(kLargeThreads)
k_large(const float4 *__restrict__ records, const unsigned int *__restrict__ bin_start, DeviceStats *__restrict__ stats,
        unsigned long long *__restrict__ accum, const __grid_constant__ FrameParams fp)
{
    constexpr int kPix = T * T;
    constexpr int kPpt = (kPix + kLargeThreads - 1) / kLargeThreads;
    constexpr int kTilesPerSuper = 1 << (2 * kSuperShift);
    __shared__ __align__(128) float4 stage[kLargeStages][kLargeWin][2];
    __shared__ float4 sA[kLargeWin], sB[kLargeWin];
    __shared__ unsigned int s_off[kMaxSuper + 1];                 // first item of every super-tile
    __shared__ unsigned int s_part[kLargeThreads / 32];
    __shared__ unsigned long long mbar[kLargeStages];
    __shared__ int s_woff[kLargeThreads / 32];
    __shared__ unsigned int s_item;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (stats->overflow || stats->large_pairs == 0ull) return;          // no LARGE particle in this frame
    // ---- item table: items of super-tile s = ceil(records / kLargeChunk) * 64, exclusive prefix over s
    const int n_super = fp.n_super;
    {
        const int per = (n_super + kLargeThreads - 1) / kLargeThreads;
        const int b0 = min(n_super, (int)threadIdx.x * per), b1 = min(n_super, b0 + per);
        unsigned int sum = 0u;
        for (int s = b0; s < b1; ++s) {
            const unsigned int c = bin_start[fp.n_tiles + s + 1] - bin_start[fp.n_tiles + s];
            sum += (c + kLargeChunk - 1) / kLargeChunk * kTilesPerSuper;
        }
        unsigned int inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_part[warp] = inc;
        __syncthreads();
        unsigned int run = inc - sum;
        for (int w = 0; w < warp; ++w) run += s_part[w];
        for (int s = b0; s < b1; ++s) {
            const unsigned int c = bin_start[fp.n_tiles + s + 1] - bin_start[fp.n_tiles + s];
            s_off[s] = run;
            run += (c + kLargeChunk - 1) / kLargeChunk * kTilesPerSuper;
        }
        if (threadIdx.x == kLargeThreads - 1) s_off[n_super] = run;
        if (threadIdx.x == 0) {
            for (int s = 0; s < kLargeStages; ++s) mbar_init(smem_u32(mbar + s), 1u);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
    }
    const unsigned int total = s_off[n_super];
    if (total == 0u) return;
    const int e = fixed_exponent(stats->amax_bits);
    const float sc1 = pow2i(e / 2), sc2 = pow2i(e - e / 2);
    // this thread's pixels inside the tile: kPpt adjacent ones in one row
    const int p0 = threadIdx.x * kPpt;
    const bool owner = p0 < kPix;
    const int row = owner ? p0 / T : 0, col0 = owner ? p0 % T : 0;
    unsigned int wcount = 0u;
    auto issue = [&](unsigned int wbase, unsigned int j, unsigned int r0, unsigned int r1) {
        const unsigned int s = (wbase + j) % kLargeStages;
        const unsigned int wb = r0 + j * kLargeWin, bytes = 32u * (min(wb + kLargeWin, r1) - wb);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(smem_u32(mbar + s), bytes);
        bulk_copy_g2s(smem_u32(&stage[s][0][0]), records + 2ull * wb, bytes, smem_u32(mbar + s));
    };
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_item = atomicAdd(&stats->large_counter, 1u);
        __syncthreads();
        const unsigned int item = s_item;
        if (item >= total) break;
        // super-tile of the item: the last s with s_off[s] <= item (items of one chunk, 64 tiles, are neighbours:
        // the CTAs that work on them read the same records at about the same time, from L2)
        int lo = 0, hi = n_super;
        while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (s_off[mid] <= item) lo = mid; else hi = mid; }
        const int sup = lo;
        const unsigned int local = item - s_off[sup];
        const unsigned int chunk = local >> (2 * kSuperShift);
        const int tin = (int)(local & (kTilesPerSuper - 1));
        const int tx = ((sup % fp.nsx) << kSuperShift) + (tin & ((1 << kSuperShift) - 1));
        const int ty = ((sup / fp.nsx) << kSuperShift) + (tin >> kSuperShift);
        if (tx >= fp.ntx || ty >= fp.nty) continue;              // the super-tile hangs over the image edge
        const int tile = ty * fp.ntx + tx;
        const int tx0 = tx * T, ty0 = ty * T;
        const unsigned int lb = bin_start[fp.n_tiles + sup], le = bin_start[fp.n_tiles + sup + 1];
        const unsigned int r0 = lb + chunk * kLargeChunk, r1 = min(r0 + kLargeChunk, le);
        const unsigned int nwin = (r1 - r0 + kLargeWin - 1) / kLargeWin;
        const unsigned int wbase = wcount;
        if (threadIdx.x == 0)
            for (unsigned int j = 0; j < min(nwin, (unsigned int)kLargeStages); ++j) issue(wbase, j, r0, r1);
        // the tile inside its super-tile, in pixels (record boxes are relative to the super-tile)
        const int qx0 = (tin & ((1 << kSuperShift) - 1)) * T, qy0 = (tin >> kSuperShift) * T;
        const int qx1 = qx0 + T - 1, qy1 = qy0 + T - 1;
        // centres of the tile's corner pixels
        const float cxl = __fadd_rn((float)tx0, 0.5f), cxh = __fadd_rn((float)(tx0 + T - 1), 0.5f);
        const float cyl = __fadd_rn((float)ty0, 0.5f), cyh = __fadd_rn((float)(ty0 + T - 1), 0.5f);
        float acc[kPpt][3], sub[kPpt][3], fxc[kPpt];
        const float fyc = __fadd_rn((float)(ty0 + row), 0.5f);
#pragma unroll
        for (int k = 0; k < kPpt; ++k) {
            acc[k][0] = acc[k][1] = acc[k][2] = 0.0f;
            sub[k][0] = sub[k][1] = sub[k][2] = 0.0f;
            fxc[k] = __fadd_rn((float)(tx0 + col0 + k), 0.5f);
        }
        for (unsigned int k = 0; k < nwin; ++k, ++wcount) {
            const unsigned int st = wcount % kLargeStages;
            mbar_wait(smem_u32(mbar + st), (wcount / kLargeStages) & 1u);
            const unsigned int wb = r0 + k * kLargeWin, cntw = min(wb + kLargeWin, r1) - wb;
            bool hit = false;
            float4 ra = make_float4(0.f, 0.f, 0.f, 0.f), rb = ra;
            if (threadIdx.x < cntw) {
                ra = stage[st][threadIdx.x][0]; rb = stage[st][threadIdx.x][1];
                const unsigned int box = __float_as_uint(rb.w);
                const int bx0 = (int)(box & 255u), by0 = (int)((box >> 8) & 255u);
                const int bx1 = (int)((box >> 16) & 255u), by1 = (int)(box >> 24);
                hit = bx0 <= qx1 && bx1 >= qx0 && by0 <= qy1 && by1 >= qy0;
                if (hit) {
                    // the disc against the tile: skip it when even the nearest point of the tile's pixel-centre
                    // rectangle is outside (with a margin that covers the float32 rounding of the C1 test)
                    const float nx = fmaxf(fmaxf(cxl - ra.x, ra.x - cxh), 0.0f), ny = fmaxf(fmaxf(cyl - ra.y, ra.y - cyh), 0.0f);
                    hit = fmaf(nx, nx, ny * ny) <= ra.w * 1.0001f;
                }
            }
            const unsigned int bal = __ballot_sync(0xffffffffu, hit);
            if (lane == 0) s_woff[warp] = __popc(bal);
            __syncthreads();                 // counts visible; every warp is done with the previous window's hits
            // the stage of the previous window is free now: refill it
            if (k >= 1u && threadIdx.x == 0 && k - 1u + kLargeStages < nwin) issue(wbase, k - 1u + kLargeStages, r0, r1);
            int woff = 0, cnt = 0;
#pragma unroll
            for (int w = 0; w < kLargeThreads / 32; ++w) { const int c = s_woff[w]; woff += w < warp ? c : 0; cnt += c; }
            if (hit) {
                const int pos = woff + __popc(bal & ((1u << lane) - 1u));
                sA[pos] = ra; sB[pos] = rb;
            }
            __syncthreads();
            if (owner) {
                for (int m = 0; m < cnt; ++m) {
                    const float4 a = sA[m], b = sB[m];
                    const float dyf = __fsub_rn(fyc, a.y);
                    const float t2 = __fmul_rn(dyf, dyf);
#pragma unroll
                    for (int q = 0; q < kPpt; ++q) {
                        const float dxf = __fsub_rn(fxc[q], a.x);
                        const float d2 = __fmaf_rn(dxf, dxf, t2);
                        const float wgt = d2 <= a.w ? ex2_approx(d2 * a.z) : 0.0f;
                        sub[q][0] = fmaf(b.x, wgt, sub[q][0]);
                        sub[q][1] = fmaf(b.y, wgt, sub[q][1]);
                        sub[q][2] = fmaf(b.z, wgt, sub[q][2]);
                    }
                }
            }
            if ((k & 3u) == 3u || k + 1u == nwin) {              // two-level sums: fold the sub-sums every 4 windows
#pragma unroll
                for (int q = 0; q < kPpt; ++q)
#pragma unroll
                    for (int c = 0; c < 3; ++c) { acc[q][c] += sub[q][c]; sub[q][c] = 0.0f; }
            }
        }
        // ---- the item's sums -> the tile's 64-bit fixed-point sums
        if (owner) {
            unsigned long long *out = accum + (size_t)tile * (3 * kPix) + p0;
#pragma unroll
            for (int q = 0; q < kPpt; ++q)
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const long long f = __float2ll_rn(acc[q][c] * sc1 * sc2);
                    if (f != 0ll) atomicAdd(out + c * kPix + q, (unsigned long long)f);
                }
        }
    }
}

}  // namespace splotch
