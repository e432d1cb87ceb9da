// splotch_btile.cuh -- the paper's own medium-particle scheme, kept as an alternative renderer for comparison
// (Table 1 :254-266: t_x = 8, n_p = 16, r_0 = 8 was the best tuning on K20X).
//
//   * a MEDIUM particle belongs to ONE tile, the tile of its centre, i(p) (:172); k_count / k_scatter bin it there;
//   * a CUDA block owns a tile and keeps the "Btile" in shared memory: the t x t body plus a boundary of r_0 pixels on
//     every side, so that every particle of the tile lies entirely inside it (:224; needs r_0 <= t);
//   * the tile's particles are staged n_p at a time "by a single read operation performed simultaneously by the
//     threads of the block" and rendered one after the other, "each with a single parallel operation so that each pixel
//     affected by a particle is processed by a different thread of the block" (:226): thread (i, j) of a (2 r_0 + 1)^2
//     block takes pixel (x0 + i, y0 + j) of the particle's box.  (The paper's block has 4 r_0^2 threads; the pixel box of
//     a disc of radius exactly r_0 centred on a pixel centre is 2 r_0 + 1 wide, hence the + 1.)  A barrier separates
//     consecutive particles: they map threads to pixels differently;
//   * "when all particles of the block are rendered" the body goes to the image and the boundary to "three more copies
//     of the image ... to store corners, rows and columns of the boundary" (:228); a second kernel composes them with
//     "the partial image produced by the small particles".  With r_0 > t / 2 two neighbours' boundaries can meet on a
//     pixel of the same copy, so the boundary is added with float32 atomics (red.global.add.f32);
//   * SMALL particles: the paper reduces a fragment buffer by pixel with Thrust (:179); here k_scatter adds them to the
//     small-particle partial image with float32 atomics -- the same partial image, built without a sort;
//   * LARGE particles (r > r_0): the paper's CPU path (:232-238) is k_large here, as in the default renderer.
// Sums are plain float32 in arrival order, as in the paper: accuracy degrades like sqrt(n) 2^-24 with the number of
// contributions per pixel, where the default renderer's two-level and fixed-point sums do not.
#pragma once
#include "splotch_kernels.cuh"

namespace splotch {

constexpr int kBtilePlanes = 5;          // body, corners, rows, columns, small particles

__device__ __forceinline__ void red_add_f32(float *p, float v)
{
    asm volatile("red.global.add.f32 [%0], %1;" :: "l"(p), "f"(v) : "memory");
}

// dynamic shared memory: Btile 3 x side^2 floats, then n_p records
__global__ void __launch_bounds__(1024)
k_btile(const float4 *__restrict__ records, const uint2 *__restrict__ run, const DeviceStats *__restrict__ stats,
        float *__restrict__ planes, const __grid_constant__ FrameParams fp)
{
    extern __shared__ __align__(16) float bt_smem[];
    const int T = fp.T, r0 = fp.btile_r0, np = fp.btile_np;
    const int side = T + 2 * r0, npix = side * side, B = 2 * r0 + 1;
    float *bt = bt_smem;                                            // [3][side * side]
    float4 *stage = reinterpret_cast<float4 *>(bt_smem + ((3 * npix + 3) & ~3));
    if (stats->overflow) return;
    const int tile = blockIdx.x;
    const int X0 = (tile % fp.ntx) * T - r0, Y0 = (tile / fp.ntx) * T - r0;       // Btile origin on the screen
    for (int i = threadIdx.x; i < 3 * npix; i += blockDim.x) bt[i] = 0.0f;
    const int ti = threadIdx.x % B, tj = threadIdx.x / B;
    const bool worker = (int)threadIdx.x < B * B;
    __syncthreads();
    for (int s = 0; s < kMaxSlabs; ++s) {
        const uint2 rn = run[(size_t)(2 * tile) * kMaxSlabs + s];
        const float4 *src = records + stats->slab_base[s] + rn.x;
        for (unsigned int c0 = 0; c0 < rn.y; c0 += (unsigned int)np) {
            const int m = (int)min((unsigned int)np, rn.y - c0);
            for (int i = threadIdx.x; i < 2 * m; i += blockDim.x) stage[i] = src[2 * (size_t)c0 + i];
            __syncthreads();
            for (int q = 0; q < m; ++q) {
                const float4 A = stage[2 * q], Bv = stage[2 * q + 1];
                const unsigned int box = __float_as_uint(Bv.w);
                const int bx0 = (int)(box & 63u), by0 = (int)((box >> 6) & 63u);
                const int bw1 = (int)((box >> 12) & 63u), bh1 = (int)((box >> 18) & 63u);
                if (worker && ti <= bw1 && tj <= bh1) {
                    const int bx = bx0 + ti, by = by0 + tj;
                    const float dxf = __fsub_rn(__fadd_rn((float)(X0 + bx), 0.5f), A.x);
                    const float dyf = __fsub_rn(__fadd_rn((float)(Y0 + by), 0.5f), A.y);
                    const float d2 = __fmaf_rn(dxf, dxf, __fmul_rn(dyf, dyf));
                    if (d2 <= A.w) {
                        const float w = ex2_approx(d2 * A.z);
                        float *px = bt + by * side + bx;
                        px[0] = fmaf(Bv.x, w, px[0]); px[npix] = fmaf(Bv.y, w, px[npix]); px[2 * npix] = fmaf(Bv.z, w, px[2 * npix]);
                    }
                }
                __syncthreads();
            }
        }
    }
    // ---- body -> image copy 0 (this block only), boundary -> corners / rows / columns copies
    const size_t plane = 3 * (size_t)fp.W * fp.H;
    for (int p = threadIdx.x; p < npix; p += blockDim.x) {
        const int bx = p % side, by = p / side, X = X0 + bx, Y = Y0 + by;
        if (X < 0 || Y < 0 || X >= fp.W || Y >= fp.H) continue;
        const bool in_x = bx >= r0 && bx < r0 + T, in_y = by >= r0 && by < r0 + T;
        const float v0 = bt[p], v1 = bt[npix + p], v2 = bt[2 * npix + p];
        float *o = planes + 3 * ((size_t)Y * fp.W + X);
        if (in_x && in_y) { o[0] = v0; o[1] = v1; o[2] = v2; }
        else if (v0 != 0.0f || v1 != 0.0f || v2 != 0.0f) {
            o += plane * (in_y ? 3 : (in_x ? 2 : 1));                 // beside the body: columns; above / below: rows; else corners
            red_add_f32(o, v0); red_add_f32(o + 1, v1); red_add_f32(o + 2, v2);
        }
    }
}

// image (already holding the LARGE particles' part from k_compose) += body + corners + rows + columns + small; transfer last
__global__ void __launch_bounds__(256)
k_btile_compose(const float *__restrict__ planes, size_t n, int apply_transfer, float *__restrict__ image)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        float v = image[i];
#pragma unroll
        for (int k = 0; k < kBtilePlanes; ++k) v += planes[k * n + i];
        image[i] = apply_transfer ? -expm1f(-v) : v;
    }
}

}  // namespace splotch
