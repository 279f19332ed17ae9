// probe.cuh -- FP64 FMA throughput probe (roofline denominator for an ALU-bound FP64 path).
// PROBE_CHAINS independent dependent-FMA chains per thread keep the DFMA pipe full.
#pragma once
#include "common.cuh"

constexpr int PROBE_CHAINS = 8;
constexpr int PROBE_UNROLL = 16;

__global__ void __launch_bounds__(256)
k_probe_dfma(double* sink, int iters, double seed)
{
    double acc[PROBE_CHAINS];
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) acc[k] = seed + k + threadIdx.x * 1e-9;
    const double m = 1.0 - 1e-9 * seed, b = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < PROBE_UNROLL; ++u)
#pragma unroll
            for (int k = 0; k < PROBE_CHAINS; ++k) acc[k] = fma(acc[k], m, b);
    }
    double s = 0;
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) s += acc[k];
    if (s == 123.456) sink[threadIdx.x] = s;   // never true; keeps the chains alive
}
