// nep_probe.cuh -- measurement and unit-test probes that are not part of the path.
// k_probe_ffma: FP32 FMA throughput, the measured figure bench.py reports beside the derived
// 148 SM x 128 lanes x 2 x clock peak.  NEP_PROBE_CHAINS independent chains per thread of the
// form a = fma(a, m, a): two distinct register sources per instruction (a three-source FFMA is limited by register
// operand bandwidth, not by the FMA pipe), no memory traffic in the loop.
// k_probe_entry: round trip of the packed list entry (entry_pack / entry_j of nep_kernels.cuh and the slot mask the
// walkers use) for a cheap test of indices j >= 2^23, which the signed-shift form would sign-extend.
#pragma once
#include <cuda_runtime.h>

#define NEP_PROBE_CHAINS 16

__global__ void __launch_bounds__(256)
k_probe_ffma(int iters, float m, float* __restrict__ sink)
{
    float acc[NEP_PROBE_CHAINS];
#pragma unroll
    for (int c = 0; c < NEP_PROBE_CHAINS; ++c) acc[c] = 1e-3f * (float)(threadIdx.x + c + 1) + 1e-9f * (float)blockIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < NEP_PROBE_CHAINS; ++c) acc[c] = fmaf(acc[c], m, acc[c]);      // a (1 + m), m ~ 1e-7: stays finite
    }
    float s = 0.0f;
#pragma unroll
    for (int c = 0; c < NEP_PROBE_CHAINS; ++c) s += acc[c];
    if (s == 123.456f) sink[threadIdx.x] = s;      // never true: keeps the chains alive
}

__global__ void k_probe_entry(int count, const int* __restrict__ j, const int* __restrict__ slot, int* __restrict__ packed,
                              int* __restrict__ j_out, int* __restrict__ slot_out)
{
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= count) return;
    const int e = entry_pack(j[a], slot[a]);
    packed[a] = e;
    j_out[a] = entry_j(e);
    slot_out[a] = e & ((1 << NEP_SLOT_BITS) - 1);
}
