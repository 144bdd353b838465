// gp_peak.cuh -- register-resident FP64 throughput microbenchmarks (measurement support, not on
// the hot path).  north_star asks for the FP64 peak of the chip "also measured by a
// microbenchmark and stated": these two kernels issue nothing but independent DMMA.8x8x4
// (mode 0) or DFMA (mode 1) chains from registers on every SM, so their rate is the ceiling any
// FP64 contraction on this chip can reach.  bench.py times them with CUDA events.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gpb {

constexpr int kPeakChains = 16;       // independent accumulator chains per warp (DMMA) / thread (DFMA)
constexpr int kPeakThreads = 256;
constexpr int kPeakCtasPerSm = 4;     // 32 resident warps per SM

__global__ void __launch_bounds__(kPeakThreads) peak_dmma_kernel(double* __restrict__ sink, int iters, double seed) {
    double acc[kPeakChains][2];
    const int lane = threadIdx.x & 31;
    // 4 distinct A and 4 distinct B fragments, used as a 4x4 outer product like the real kernel:
    // issuing every chain from the SAME operand registers measures 29.7 instead of 37.1 TFLOP/s
    double a[4], b[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) { a[i] = seed + 1e-9 * lane + i; b[i] = 1.0 - 1e-9 * lane - i; }
#pragma unroll
    for (int j = 0; j < kPeakChains; ++j) acc[j][0] = acc[j][1] = 0.0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < kPeakChains; ++j)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(acc[j][0]), "+d"(acc[j][1])
                         : "d"(a[j & 3]), "d"(b[(j >> 2) & 3]));
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < kPeakChains; ++j) s += acc[j][0] + acc[j][1];
    if (s == 123.456) sink[0] = s;    // never true: keeps the chains alive without memory traffic
}

__global__ void __launch_bounds__(kPeakThreads) peak_dfma_kernel(double* __restrict__ sink, int iters, double seed) {
    double acc[kPeakChains];
    const double a = seed + 1e-9 * threadIdx.x, b = 1e-12;
#pragma unroll
    for (int j = 0; j < kPeakChains; ++j) acc[j] = (double)j;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < kPeakChains; ++j) acc[j] = fma(acc[j], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < kPeakChains; ++j) s += acc[j];
    if (s == 123.456) sink[0] = s;
}


}  // namespace gpb
