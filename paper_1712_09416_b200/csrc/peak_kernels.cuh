// peak_kernels.cuh -- measured FP32 issue peaks of the device, the denominators of K5's roofline (DESIGN.md
// "Kernels, bounds"): independent chains of fused multiply-adds (the machine's FP32 peak) and of un-fused
// multiply + add pairs (the ceiling of arithmetic that is defined without contraction, as the tracker's is).
// Not part of the hot path: bench.py calls tpc_measure_fp32_peak once.
#pragma once
#include <cuda_runtime.h>

namespace tpc {

constexpr int kPeakThreads = 256;
constexpr int kPeakChains = 8;       // independent accumulators per thread (hides the 4-cycle FMA latency)
constexpr int kPeakIters = 4096;

template <bool FUSED>
__global__ void __launch_bounds__(kPeakThreads) k_fp32_peak(float* out, float a, float b) {
    float acc[kPeakChains];
#pragma unroll
    for (int k = 0; k < kPeakChains; k++) acc[k] = (float)(threadIdx.x + k);
    for (int it = 0; it < kPeakIters; it++) {
#pragma unroll
        for (int k = 0; k < kPeakChains; k++)
            acc[k] = FUSED ? __fmaf_rn(acc[k], a, b) : __fadd_rn(__fmul_rn(acc[k], a), b);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kPeakChains; k++) s += acc[k];
    if (s == 12345.678f) out[0] = s;   // keeps the chains alive; practically never true
}

// 2 flops per chain step either way (multiply + add)
inline double fp32_peak_flops_per_launch(int blocks) { return 2.0 * kPeakChains * (double)kPeakIters * kPeakThreads * blocks; }

}  // namespace tpc
