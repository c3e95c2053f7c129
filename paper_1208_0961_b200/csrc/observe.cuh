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
constexpr int kLrfComp = 5;                     // T00, T0x, Txx, Tyy, Tzz
constexpr int kLrfMaxSlabs = 256;               // kObsWarps * 5 * 256 doubles = 80 KB of shared memory

// Every thread keeps running sums for two adjacent slabs, base and base + 1, with base uniform
// over the warp.  The store is cell-sorted with x slowest and a CTA walks a contiguous range of
// tiles, so consecutive particles lie in one layer of cells -- which spans one or two slabs when
// nslab <= 2 nx (x is random inside a cell, so the two alternate from particle to particle).  Only
// when some lane meets a slab outside {base, base + 1} does the warp reduce its sums (shuffle
// trees) into its shared-memory bins and move the base.  When that happens depends on the data
// only, never on scheduling: the result is bit-reproducible from run to run.  (More than two
// slabs per cell layer still work, with a flush per change.)
template <int NC>
__device__ __forceinline__ void warp_flush(double (&acc0)[NC], double (&acc1)[NC], int base, double *bins, int nslab, int lane)
{
    if (base < 0) return;
#pragma unroll
    for (int q = 0; q < NC; ++q) {
        double r0 = acc0[q], r1 = acc1[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            r0 += __shfl_xor_sync(0xFFFFFFFFu, r0, o);
            r1 += __shfl_xor_sync(0xFFFFFFFFu, r1, o);
        }
        if (lane == 0) {
            bins[q * nslab + base] += r0;
            if (base + 1 < nslab) bins[q * nslab + base + 1] += r1;
        }
        acc0[q] = 0.0; acc1[q] = 0.0;
    }
}

// LRF = false: energy density per slab (NC = 1) + totals (sum E, sum p); partial layout per
//       block: [0..3] totals, [4 .. 4+nslab) slab energies.
// LRF = true:  T00, T0x, Txx, Tyy, Tzz per slab (A22): per particle
//       w = 1/E and the contributions E, px, (px*px)*w, (py*py)*w, (pz*pz)*w; partial layout
//       per block: [comp][nslab].
// One HBM pass over x, px, py, pz (32 B per particle).
// WIDE (more than two slabs per layer of cells, nslab > 2 nx): the running sums live in shared memory
//       instead of registers -- every lane owns a private column of `window` consecutive slabs
//       [base, base + window) per component (index (s * NC + q) * 32 + lane: no bank conflicts, no
//       atomics, the order of a lane's additions is the order of its particles), reduced over the
//       lanes (shuffle trees) into the warp's bins when a particle falls outside the window.  Data-
//       dependent only, like the register path: bit-reproducible.  Rows that span more than `window`
//       slabs are peeled slab by slab as before.
constexpr int kObsWindowMax = 32, kLrfWindowMax = 9;

template <int NC>
__device__ __forceinline__ void window_flush(double *wb, int window, int base, double *bins, int nslab, int lane)
{
    if (base < 0) return;
    for (int s = 0; s < window && base + s < nslab; ++s) {
#pragma unroll
        for (int q = 0; q < NC; ++q) {
            double r = wb[(s * NC + q) * 32 + lane];
            wb[(s * NC + q) * 32 + lane] = 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xFFFFFFFFu, r, o);
            if (lane == 0) bins[q * nslab + base + s] += r;
        }
    }
}

template <bool LRF, bool WIDE>
__global__ void __launch_bounds__(kObsThreads, WIDE ? 1 : (LRF ? 3 : 4))
k_observe_partial(int64_t n, const double *__restrict__ x, const double *__restrict__ px,
                  const double *__restrict__ py, const double *__restrict__ pz, double inv_w,
                  int nslab, int window, double *__restrict__ partial)
{
    constexpr int NC = LRF ? kLrfComp : 1;
    extern __shared__ double s_bins[];          // [kObsWarps][NC][nslab], WIDE: then [kObsWarps][window][NC][32]
    __shared__ double s_tot[kObsWarps][4];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    double *bins = s_bins + (size_t)wid * NC * nslab;
    for (int s = lane; s < NC * nslab; s += 32) bins[s] = 0.0;
    double *wb = s_bins + (size_t)kObsWarps * NC * nslab + (size_t)wid * window * NC * 32;
    if (WIDE)
        for (int s = 0; s < window * NC; ++s) wb[s * 32 + lane] = 0.0;
    __syncwarp();
    double tE = 0.0, tx = 0.0, ty = 0.0, tz = 0.0;
    double acc0[NC], acc1[NC];
#pragma unroll
    for (int q = 0; q < NC; ++q) { acc0[q] = 0.0; acc1[q] = 0.0; }
    int base = -1;                              // warp-uniform
    const int64_t ntiles = (n + kObsTile - 1) / kObsTile;
    const int64_t per = (ntiles + gridDim.x - 1) / gridDim.x;     // contiguous range of tiles per CTA
    const int64_t t0 = blockIdx.x * per, t1 = min(ntiles, t0 + per);
    for (int64_t tile = t0; tile < t1; ++tile) {
        double a[kObsItems], b[kObsItems], c[kObsItems], xx[kObsItems];
#pragma unroll
        for (int k = 0; k < kObsItems; ++k) {
            const int64_t i = min(tile * kObsTile + k * kObsThreads + tid, n - 1);
            a[k] = px[i]; b[k] = py[i]; c[k] = pz[i]; xx[k] = x[i];
        }
#pragma unroll
        for (int k = 0; k < kObsItems; ++k) {
            const bool valid = tile * kObsTile + k * kObsThreads + tid < n;
            double v[NC];
#pragma unroll
            for (int q = 0; q < NC; ++q) v[q] = 0.0;
            if (valid) {
                const double E = energy(a[k], b[k], c[k]);
                v[0] = E;
                if (LRF) {
                    const double w = 1.0 / E;
                    v[1 % NC] = a[k];
                    v[2 % NC] = (a[k] * a[k]) * w;
                    v[3 % NC] = (b[k] * b[k]) * w;
                    v[4 % NC] = (c[k] * c[k]) * w;
                } else {
                    tE += E; tx += a[k]; ty += b[k]; tz += c[k];
                }
            }
            const int slab = valid ? min(max(__double2int_rz(xx[k] * inv_w), 0), nslab - 1) : -1;
            bool keep = true;
            const int span = WIDE ? window : 2;           // slabs the running sums cover: [base, base + span)
            if (__any_sync(0xFFFFFFFFu, valid && (base < 0 || slab < base || slab >= base + span))) {
                if (WIDE) window_flush<NC>(wb, window, base, bins, nslab, lane);
                else warp_flush<NC>(acc0, acc1, base, bins, nslab, lane);
                int m = valid ? slab : 0x7FFFFFFF;              // new base: the smallest slab present
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) m = min(m, __shfl_xor_sync(0xFFFFFFFFu, m, o));
                base = m;
                if (__any_sync(0xFFFFFFFFu, valid && slab >= base + span)) {
                    // more slabs among these 32 particles than the running sums cover: peel them off one
                    // slab at a time straight into the bins; nothing is carried over
                    uint32_t todo = __ballot_sync(0xFFFFFFFFu, valid);
                    while (todo) {
                        const int leader = __ffs(todo) - 1;
                        const int s0 = __shfl_sync(0xFFFFFFFFu, slab, leader);
                        const bool mine = valid && slab == s0;
#pragma unroll
                        for (int q = 0; q < NC; ++q) {
                            double r = mine ? v[q] : 0.0;
#pragma unroll
                            for (int o = 16; o > 0; o >>= 1) r += __shfl_xor_sync(0xFFFFFFFFu, r, o);
                            if (lane == 0) bins[q * nslab + s0] += r;
                        }
                        todo &= ~__ballot_sync(0xFFFFFFFFu, mine);
                    }
                    base = -1;
                    keep = false;
                }
            }
            if (keep && valid) {
                if (WIDE) {
                    double *col = wb + (size_t)(slab - base) * NC * 32 + lane;
#pragma unroll
                    for (int q = 0; q < NC; ++q) col[q * 32] += v[q];
                } else if (slab == base) {
#pragma unroll
                    for (int q = 0; q < NC; ++q) acc0[q] += v[q];
                } else {
#pragma unroll
                    for (int q = 0; q < NC; ++q) acc1[q] += v[q];
                }
            }
        }
    }
    if (WIDE) window_flush<NC>(wb, window, base, bins, nslab, lane);
    else warp_flush<NC>(acc0, acc1, base, bins, nslab, lane);
    if (!LRF) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            tE += __shfl_xor_sync(0xFFFFFFFFu, tE, o);
            tx += __shfl_xor_sync(0xFFFFFFFFu, tx, o);
            ty += __shfl_xor_sync(0xFFFFFFFFu, ty, o);
            tz += __shfl_xor_sync(0xFFFFFFFFu, tz, o);
        }
        if (lane == 0) { s_tot[wid][0] = tE; s_tot[wid][1] = tx; s_tot[wid][2] = ty; s_tot[wid][3] = tz; }
    }
    __syncthreads();
    const int head = LRF ? 0 : 4;
    double *out = partial + (size_t)blockIdx.x * (head + NC * nslab);
    if (!LRF && tid < 4) {
        double s = 0.0;
        for (int w = 0; w < kObsWarps; ++w) s += s_tot[w][tid];
        out[tid] = s;
    }
    for (int s = tid; s < NC * nslab; s += kObsThreads) {
        double v = 0.0;
        for (int w = 0; w < kObsWarps; ++w) v += s_bins[(size_t)w * NC * nslab + s];
        out[head + s] = v;
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

// result: T[5][nslab] then lrf[4][nslab] = e, v, P_L, P_T (Landau matching for a flow along x).
// One warp per slab; lanes sum the block partials in a fixed order.
__global__ void __launch_bounds__(256)
k_observe_lrf_final(int nblocks, int nslab, const double *__restrict__ partial, double vol,
                    double *__restrict__ result)
{
    const int j = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (j >= nslab) return;
    double T[kLrfComp];
#pragma unroll
    for (int q = 0; q < kLrfComp; ++q) {
        double s = 0.0;
        for (int b = lane; b < nblocks; b += 32) s += partial[((size_t)b * kLrfComp + q) * nslab + j];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
        T[q] = s / vol;
    }
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < kLrfComp; ++q) result[q * nslab + j] = T[q];
        const double tr = T[0] + T[2];
        double disc = tr * tr - 4.0 * (T[1] * T[1]);
        if (!(disc > 0.0)) disc = 0.0;
        const double e = 0.5 * ((T[0] - T[2]) + sqrt(disc));
        const double den = e + T[2];
        double *lrf = result + (size_t)kLrfComp * nslab;
        lrf[0 * nslab + j] = e;
        lrf[1 * nslab + j] = (den > 0.0) ? T[1] / den : 0.0;
        lrf[2 * nslab + j] = (e - T[0]) + T[2];
        lrf[3 * nslab + j] = 0.5 * (T[3] + T[4]);
    }
}

}  // namespace cuba
