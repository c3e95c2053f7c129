// probe.cuh -- fp64 FMA micro-benchmark: the measured fp64 leg of the roofline (SURVEY.md 8(d):
// "fp64-pipe utilisation against a peak the builder measures"; north_star: "fp64 pipe utilisation
// against the chip's fp64 peak").  No part of the method: a timing probe on the profiling surface.
#pragma once
#include "common.cuh"

namespace cuba {

constexpr int kProbeThreads = 256;
constexpr int kProbeChains = 8;     // independent dependency chains per thread: hides the DFMA latency

// Every thread runs kProbeChains independent chains of `iters` dependent DFMAs (explicit
// __fma_rn: the library is compiled with -fmad=false).  The result is stored so that nothing is
// optimised away; a, b are kernel arguments so that nothing is folded.
__global__ void __launch_bounds__(kProbeThreads)
k_probe_fp64(int iters, double a, double b, double *__restrict__ out)
{
    double v[kProbeChains];
#pragma unroll
    for (int k = 0; k < kProbeChains; ++k) v[k] = (double)(threadIdx.x + k);
#pragma unroll 1
    for (int i = 0; i < iters; i += 4) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int k = 0; k < kProbeChains; ++k) v[k] = __fma_rn(v[k], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < kProbeChains; ++k) s += v[k];
    out[(size_t)blockIdx.x * kProbeThreads + threadIdx.x] = s;
}

}  // namespace cuba
