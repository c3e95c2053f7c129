// observe.cuh -- observables (PAPER.md:66 total energy; Fig. 2 energy density
// per x-slab).  One HBM pass over x, px, py, pz (32 B per particle), warp-shuffle
// reductions, no floating-point atomics: the summation order is fixed, so the result is
// bit-reproducible from run to run.
#pragma once
#include "common.cuh"

namespace cuba {

constexpr int kObsThreads = 256;
constexpr int kObsWarps = kObsThreads / 32;
constexpr int kObsItems = 4;                    // particles per thread per tile: 16 independent loads in flight
constexpr int kObsTile = kObsThreads * kObsItems;
constexpr int kObsMaxSlabs = 1024;

// partial layout per block: [0..3] totals, [4 .. 4+nslab) slab energies
__global__ void __launch_bounds__(kObsThreads, 4)
k_observe_partial(int64_t n, const double *__restrict__ x, const double *__restrict__ px,
                  const double *__restrict__ py, const double *__restrict__ pz, double inv_w,
                  int nslab, double *__restrict__ partial)
{
    extern __shared__ double s_bins[];          // [kObsWarps][nslab]
    __shared__ double s_tot[kObsWarps][4];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    double *bins = s_bins + (size_t)wid * nslab;
    for (int s = lane; s < nslab; s += 32) bins[s] = 0.0;
    __syncwarp();
    double tE = 0.0, tx = 0.0, ty = 0.0, tz = 0.0;
    const int64_t ntiles = (n + kObsTile - 1) / kObsTile;
    for (int64_t tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        double a[kObsItems], b[kObsItems], c[kObsItems], xx[kObsItems];
#pragma unroll
        for (int k = 0; k < kObsItems; ++k) {
            const int64_t i = min(tile * kObsTile + k * kObsThreads + tid, n - 1);
            a[k] = px[i]; b[k] = py[i]; c[k] = pz[i]; xx[k] = x[i];
        }
#pragma unroll
        for (int k = 0; k < kObsItems; ++k) {
            const bool valid = tile * kObsTile + k * kObsThreads + tid < n;
            const double E = valid ? energy(a[k], b[k], c[k]) : 0.0;
            if (valid) { tE += E; tx += a[k]; ty += b[k]; tz += c[k]; }
            const int slab = valid ? min(max(__double2int_rz(xx[k] * inv_w), 0), nslab - 1) : -1;
            // the store is sorted with x slowest, so a warp sees one or two slabs: peel them off
            uint32_t todo = __ballot_sync(0xFFFFFFFFu, valid);
            while (todo) {
                const int leader = __ffs(todo) - 1;
                const int s0 = __shfl_sync(0xFFFFFFFFu, slab, leader);
                const bool mine = valid && slab == s0;
                double v = mine ? E : 0.0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
                if (lane == 0) bins[s0] += v;
                todo &= ~__ballot_sync(0xFFFFFFFFu, mine);
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        tE += __shfl_xor_sync(0xFFFFFFFFu, tE, o);
        tx += __shfl_xor_sync(0xFFFFFFFFu, tx, o);
        ty += __shfl_xor_sync(0xFFFFFFFFu, ty, o);
        tz += __shfl_xor_sync(0xFFFFFFFFu, tz, o);
    }
    if (lane == 0) { s_tot[wid][0] = tE; s_tot[wid][1] = tx; s_tot[wid][2] = ty; s_tot[wid][3] = tz; }
    __syncthreads();
    double *out = partial + (size_t)blockIdx.x * (4 + nslab);
    if (tid < 4) {
        double s = 0.0;
        for (int w = 0; w < kObsWarps; ++w) s += s_tot[w][tid];
        out[tid] = s;
    }
    for (int s = tid; s < nslab; s += kObsThreads) {
        double v = 0.0;
        for (int w = 0; w < kObsWarps; ++w) v += s_bins[(size_t)w * nslab + s];
        out[4 + s] = v;
    }
}

// result[0..3] totals, result[4..] = slab energy / (r_test * V_slab).  One warp per output: lane l
// adds the partials of blocks l, l+32, ... in that order, then a fixed shuffle tree: the order of
// the summation does not depend on scheduling.
__global__ void __launch_bounds__(256)
k_observe_final(int nblocks, int nslab, const double *__restrict__ partial, double vol,
                double *__restrict__ result)
{
    const int e = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (e >= 4 + nslab) return;
    double s = 0.0;
    for (int b = lane; b < nblocks; b += 32) s += partial[(size_t)b * (4 + nslab) + e];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    if (lane == 0) result[e] = (e < 4) ? s : s / vol;
}

}  // namespace cuba
