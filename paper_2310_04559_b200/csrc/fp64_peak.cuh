// cc_ladder_fp64_peak: the roofline denominator measured on the device the ladder runs on.
// A register-only DMMA.8x8x4 loop (8 warps per SM, 8 independent accumulator pairs per warp -- the issue pattern that
// saturates the FP64 tensor pipe, profiles/round1_microbench.md) timed with CUDA events and with the SM cycle counter.
#pragma once
#include "ladder_common.cuh"

namespace ccl {

__global__ void __launch_bounds__(256) fp64_peak_kernel(double *sink, int iters, long long *cycles)
{
    double acc[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        acc[i][0] = 1e-300 * threadIdx.x;
        acc[i][1] = 1e-300 * i;
    }
    const double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) dmma_8x8x4(acc[i][0], acc[i][1], a, b);
    }
    const long long t1 = clock64();
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += acc[i][0] + acc[i][1];
    if (s == 12345.678) sink[0] = s;                     // keeps the loop alive, never true in practice
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

}  // namespace ccl
