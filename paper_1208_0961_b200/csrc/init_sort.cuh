// init_sort.cuh -- cuba_init's device work: validation, persistent ids, and the general
// stable sort that bins an arbitrary (unsorted) initial store by cell (S3 + S4, A19).
// Runs once per context, so it favours simplicity: a classical stable LSD radix sort on
// (cell key, original index) pairs, 8 bits per pass, then one gather of the seven arrays.
#pragma once
#include "common.cuh"

namespace cuba {

constexpr int kRsThreads = 256;
constexpr int kRsItems = 8;
constexpr int kRsTile = kRsThreads * kRsItems;   // each warp owns a contiguous 256-element strip

// validate (PAPER.md:44 box; massless particle needs |p| > 0), key = cell, val = index
__global__ void __launch_bounds__(256)
k_init_keys(Geom g, int64_t n, Soa in, uint32_t *__restrict__ keys, uint32_t *__restrict__ vals,
            uint32_t *__restrict__ flags)
{
    // positions only: the momenta are validated where they are first read (k_gather_perm), so that a caller
    // who uploads them on a second stream can overlap that copy with the sort of the keys (cuba_run_host)
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    const double x = in.x[i], y = in.y[i], z = in.z[i];
    const bool ok = (x >= 0.0 && x <= g.L[0] && y >= 0.0 && y <= g.L[1] && z >= 0.0 && z <= g.L[2]);
    if (!ok) atomicOr(flags, kFlagState);
    keys[i] = ok ? cell_linear(g, axis_index(x, g.inv_d[0], g.nc[0]), axis_index(y, g.inv_d[1], g.nc[1]),
                               axis_index(z, g.inv_d[2], g.nc[2])) : 0u;
    vals[i] = (uint32_t)i;
}

// H[digit * nblocks + block] = number of keys of this block with that digit
__global__ void __launch_bounds__(kRsThreads)
k_rs_hist(const uint32_t *__restrict__ keys, int64_t n, int shift, uint32_t nblocks, uint32_t *__restrict__ H)
{
    __shared__ uint32_t s_h[256];
    s_h[threadIdx.x] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * kRsTile;
    for (int j = 0; j < kRsItems; ++j) {
        const int64_t i = base + j * kRsThreads + threadIdx.x;
        if (i < n) atomicAdd(&s_h[(keys[i] >> shift) & 255u], 1u);
    }
    __syncthreads();
    H[(size_t)threadIdx.x * nblocks + blockIdx.x] = s_h[threadIdx.x];
}

// Exclusive scan of the digit-major histogram table H (256 * nblocks entries, millions for tens
// of millions of particles) in three launches: per-chunk sums, a one-CTA scan of those sums
// (k_scan_blocks), and a per-chunk scan on top of its offset.
constexpr int kScanThreads = 1024;
constexpr int kScanItems = 4;
constexpr int kScanChunk = kScanThreads * kScanItems;

__global__ void __launch_bounds__(kScanThreads)
k_chunk_sums(const uint32_t *__restrict__ H, int64_t total, uint32_t *__restrict__ sums)
{
    __shared__ uint32_t s_warp[32];
    const int64_t base = (int64_t)blockIdx.x * kScanChunk + (int64_t)threadIdx.x * kScanItems;
    uint32_t v = 0;
#pragma unroll
    for (int q = 0; q < kScanItems; ++q) v += (base + q < total) ? H[base + q] : 0u;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    if ((threadIdx.x & 31) == 0) s_warp[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        uint32_t w = s_warp[threadIdx.x];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xFFFFFFFFu, w, o);
        if (threadIdx.x == 0) sums[blockIdx.x] = w;
    }
}

__global__ void __launch_bounds__(kScanThreads)
k_chunk_scan(uint32_t *__restrict__ H, int64_t total, const uint32_t *__restrict__ chunk_prefix)
{
    __shared__ uint32_t s_warp[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t base = (int64_t)blockIdx.x * kScanChunk + (int64_t)threadIdx.x * kScanItems;
    uint32_t v[kScanItems], sum = 0;
#pragma unroll
    for (int q = 0; q < kScanItems; ++q) { v[q] = (base + q < total) ? H[base + q] : 0u; sum += v[q]; }
    uint32_t inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_warp[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        const uint32_t w = s_warp[lane];
        uint32_t winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, winc, o);
            if (lane >= o) winc += t;
        }
        s_warp[lane] = winc - w;
    }
    __syncthreads();
    uint32_t run = chunk_prefix[blockIdx.x] + s_warp[wid] + inc - sum;
#pragma unroll
    for (int q = 0; q < kScanItems; ++q) {
        if (base + q < total) H[base + q] = run;
        run += v[q];
    }
}

// stable scatter: order inside a block is (warp, row, lane) = ascending input index
__global__ void __launch_bounds__(kRsThreads)
k_rs_scatter(const uint32_t *__restrict__ keys, const uint32_t *__restrict__ vals,
             uint32_t *__restrict__ keys_out, uint32_t *__restrict__ vals_out, int64_t n, int shift,
             uint32_t nblocks, const uint32_t *__restrict__ H)
{
    __shared__ uint32_t s_w[kRsThreads / 32][256];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (int q = tid; q < (kRsThreads / 32) * 256; q += kRsThreads) (&s_w[0][0])[q] = 0;
    __syncthreads();
    const int64_t strip = (int64_t)blockIdx.x * kRsTile + (int64_t)wid * (32 * kRsItems);
    uint32_t k[kRsItems], v[kRsItems];
#pragma unroll
    for (int r = 0; r < kRsItems; ++r) {
        const int64_t i = strip + r * 32 + lane;
        const bool valid = i < n;
        k[r] = valid ? keys[i] : 0u;
        v[r] = valid ? vals[i] : 0u;
        const uint32_t active = __ballot_sync(0xFFFFFFFFu, valid);
        if (valid) {
            const uint32_t dg = (k[r] >> shift) & 255u;
            const uint32_t peers = __match_any_sync(active, dg);
            if ((peers & lanemask_lt()) == 0) s_w[wid][dg] += __popc(peers);
        }
        __syncwarp();
    }
    __syncthreads();
    {   // per digit: exclusive prefix over the warps, on top of the block's global offset
        uint32_t run = H[(size_t)tid * nblocks + blockIdx.x];
        for (int w = 0; w < kRsThreads / 32; ++w) { const uint32_t c = s_w[w][tid]; s_w[w][tid] = run; run += c; }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kRsItems; ++r) {
        const int64_t i = strip + r * 32 + lane;
        const bool valid = i < n;
        const uint32_t active = __ballot_sync(0xFFFFFFFFu, valid);
        if (valid) {
            const uint32_t dg = (k[r] >> shift) & 255u;
            const uint32_t peers = __match_any_sync(active, dg);
            const uint32_t pos = s_w[wid][dg] + __popc(peers & lanemask_lt());
            keys_out[pos] = k[r];
            vals_out[pos] = v[r];
            __syncwarp(active);
            if ((peers & lanemask_lt()) == 0) s_w[wid][dg] += __popc(peers);
        }
        __syncwarp();
    }
}

// out[k] = in[perm[k]] for the six fp64 arrays; pid[k] = perm[k] (ids are the original indices)
__global__ void __launch_bounds__(256)
k_gather_perm(int64_t n, const uint32_t *__restrict__ perm, Soa in, Soa out, uint32_t *__restrict__ flags)
{
    const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (k >= n) return;
    const uint32_t s = perm[k];
    out.x[k] = in.x[s]; out.y[k] = in.y[s]; out.z[k] = in.z[s];
    const double px = in.px[s], py = in.py[s], pz = in.pz[s];
    const double E = energy(px, py, pz);
    if (!(E > 0.0) || !isfinite(E)) atomicOr(flags, kFlagState);       // finite momenta, |p| > 0 (A21)
    out.px[k] = px; out.py[k] = py; out.pz[k] = pz;
    out.pid[k] = s;
}

// x-slab decomposition: the particles of a slab carry their index in the whole problem
__global__ void __launch_bounds__(256)
k_map_pid(int64_t n, uint32_t *__restrict__ pid, const uint32_t *__restrict__ pid_global)
{
    const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (k < n) pid[k] = pid_global[pid[k]];
}

// cell_start from the sorted keys: slot k opens every cell in (key[k-1], key[k]]
__global__ void __launch_bounds__(256)
k_starts_from_sorted(int64_t n, uint32_t ncells, const uint32_t *__restrict__ keys, uint32_t *__restrict__ cell_start)
{
    const int64_t k = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (k >= n) return;
    const uint32_t c = keys[k];
    const uint32_t first = (k == 0) ? 0u : keys[k - 1] + 1u;
    if (k == 0 || keys[k - 1] != c)
        for (uint32_t q = first; q <= c; ++q) cell_start[q] = (uint32_t)k;
    if (k == n - 1)
        for (uint32_t q = c + 1; q <= ncells; ++q) cell_start[q] = (uint32_t)n;
}

}  // namespace cuba
