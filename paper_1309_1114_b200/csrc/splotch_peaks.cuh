// splotch_peaks.cuh -- the two ALU rates the splat stages are measured against ("confirm by
// microbenchmark on the box"): FP32 FMA lane-operations per second and MUFU.EX2 results per second, whole GPU.
// Eight independent dependency chains per thread, two 1024-thread CTAs per SM; no memory traffic.
#pragma once
#include <cuda_runtime.h>

namespace splotch {

constexpr int kPeakChains = 8, kPeakIters = 4096, kPeakThreads = 1024;

template <int OP>      // 0: fma.rn.f32, 1: ex2.approx.ftz.f32
__global__ void __launch_bounds__(kPeakThreads, 2)
k_peak(float *__restrict__ out, float seed)
{
    float a[kPeakChains];
#pragma unroll
    for (int k = 0; k < kPeakChains; ++k) a[k] = seed + 0.37f * k + 1e-3f * threadIdx.x;
    for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
        for (int k = 0; k < kPeakChains; ++k) {
            if (OP == 0) a[k] = __fmaf_rn(a[k], 0.9999999f, 0.5f);
            else asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[k]));
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int k = 0; k < kPeakChains; ++k) s += a[k];
    out[(size_t)blockIdx.x * kPeakThreads + threadIdx.x] = s;
}

}  // namespace splotch
