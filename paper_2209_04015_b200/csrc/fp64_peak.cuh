// Register-resident FP64 throughput microbenchmarks: the roofline denominator for K2 (MEASURED_PEAKS.json has no
// FP64 entry; SURVEY.md §8(d) asks the builder to measure it).  mode 0 = DMMA.8x8x4 chains, mode 1 = DFMA chains.
#pragma once
#include "common.cuh"

namespace afqmc {

constexpr int PEAK_NACC = 8;     // independent DMMA accumulators per warp
constexpr int PEAK_NCH = 16;     // independent DFMA chains per thread

__global__ void __launch_bounds__(512) peak_dmma(double *out, int iters, double x, double y) {
    double c0[PEAK_NACC], c1[PEAK_NACC];
#pragma unroll
    for (int i = 0; i < PEAK_NACC; ++i) { c0[i] = i; c1[i] = -i; }
    const double a = x + threadIdx.x * 1e-12, b = y;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < PEAK_NACC; ++i) dmma_m8n8k4(c0[i], c1[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < PEAK_NACC; ++i) s += c0[i] + c1[i];
    if (s == 12345.678) out[0] = s;
}

__global__ void __launch_bounds__(512) peak_dfma(double *out, int iters, double x, double y) {
    double acc[PEAK_NCH];
#pragma unroll
    for (int i = 0; i < PEAK_NCH; ++i) acc[i] = threadIdx.x * 1e-9 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < PEAK_NCH; ++i) acc[i] = fma(acc[i], x, y);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < PEAK_NCH; ++i) s += acc[i];
    if (s == 12345.678) out[0] = s;
}

}  // namespace afqmc
