// nep_probe.cuh -- FP32 FMA throughput probe: the measured denominator of the "alu" roofline that
// bench.py reports beside the derived 148 SM x 128 lanes x 2 x clock figure.
// NEP_PROBE_CHAINS independent 3-register FFMA chains per thread, no memory traffic in the loop.
#pragma once
#include <cuda_runtime.h>

#define NEP_PROBE_CHAINS 16

__global__ void __launch_bounds__(256)
k_probe_ffma(int iters, float m, float* __restrict__ sink)
{
    float acc[NEP_PROBE_CHAINS], mul[NEP_PROBE_CHAINS];
#pragma unroll
    for (int c = 0; c < NEP_PROBE_CHAINS; ++c) {
        acc[c] = 1e-3f * (float)(threadIdx.x + c);
        mul[c] = m - 1e-6f * (float)c;
    }
    const float add = 1e-9f * (float)blockIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < NEP_PROBE_CHAINS; ++c) acc[c] = fmaf(acc[c], mul[c], add);
    }
    float s = 0.0f;
#pragma unroll
    for (int c = 0; c < NEP_PROBE_CHAINS; ++c) s += acc[c];
    if (s == 123.456f) sink[threadIdx.x] = s;      // never true: keeps the chains alive
}
