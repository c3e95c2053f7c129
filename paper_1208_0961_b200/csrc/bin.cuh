// bin.cuh -- S1-S4: streaming, wall reflection, cell index and the stable counting sort.
//
// B200-first design:
// the store is always cell-sorted (A19) and dt < cell edge, so a particle of
// old cell c can only land in one of the 27 cells around c.  A counting sort keyed by
// (old cell, direction d in 0..26) is therefore sparse:
//   K_A  k_stream_hist   per particle: S1-S3, d; cnt[d][c_old] += 1   (order-free u32 adds).  In the
//                        steady state this pass and K_carry do not run: the collision kernel of
//                        the previous step has written cnt and carry (collide.cuh, fused histogram)
//   K_B  k_gather        per new cell: the <= 27 (source cell, d) counts that feed it, taken
//                        in ascending source-cell order = ascending previous array index,
//                        turned into exclusive offsets in place; their sum is the new count
//   K_S/K_F              exclusive scan of the new counts -> cell_start
//   K_carry              per tile: particles of the tile's first cell that sit in earlier tiles
//   K_D  k_dest_base     off[d][c_old] += cell_start[c_new(c_old, d)] (one gather per particle later)
//   K_C  k_scatter       per particle again: S1-S3 recomputed, stable rank inside its
//                        (c_old, d) group from warp votes, dest = cell_start[c_new] +
//                        off[d][c_old] + rank.  No atomics touch the order: the placement is
//                        the stable counting sort of north_star (3), deterministic by construction.
// HBM traffic per particle-step: K_A reads 48 B (when it runs), K_C reads 52 B and writes 52 B.
#pragma once
#include "common.cuh"

namespace cuba {

struct Moved {
    double x, y, z, px, py, pz;
    uint32_t c_old, c_new;
    int d;   // direction code, -1 when the particle crossed more than one cell (error)
};

__device__ __forceinline__ Moved move_particle(const Geom &g, double dt, double x, double y,
                                               double z, double px, double py, double pz)
{
    Moved m;
    const int ix0 = axis_index(x, g.inv_d[0], g.nc[0]);
    const int iy0 = axis_index(y, g.inv_d[1], g.nc[1]);
    const int iz0 = axis_index(z, g.inv_d[2], g.nc[2]);
    m.c_old = cell_linear(g, ix0, iy0, iz0);
    stream_reflect(g, dt, x, y, z, px, py, pz);
    const int ix1 = axis_index(x, g.inv_d[0], g.nc[0]);
    const int iy1 = axis_index(y, g.inv_d[1], g.nc[1]);
    const int iz1 = axis_index(z, g.inv_d[2], g.nc[2]);
    m.c_new = cell_linear(g, ix1, iy1, iz1);
    const int dx = ix1 - ix0 + 1, dy = iy1 - iy0 + 1, dz = iz1 - iz0 + 1;
    m.d = ((unsigned)dx <= 2u && (unsigned)dy <= 2u && (unsigned)dz <= 2u) ? (dx * 9 + dy * 3 + dz) : -1;
    m.x = x; m.y = y; m.z = z; m.px = px; m.py = py; m.pz = pz;
    return m;
}

// ---- tile staging shared by K_A and K_C -----------------------------------------------------
// Persistent CTAs walk the tiles blockIdx.x, blockIdx.x + gridDim.x, ...  Each tile's arrays
// are contiguous 4 KB (fp64) / 2 KB (pid) chunks, fetched with cp.async.bulk (TMA bulk copy)
// into one of two shared-memory stages and signalled on an mbarrier, so a whole tile of the
// next iteration is in flight while the current one is computed -- no registers are tied up
// by loads, which is what bounded the first version (ncu: long-scoreboard stalls at 24-36 %
// occupancy, profiles/r01_*).  The last, partial tile is loaded with plain loads.
template <int NARR>   // 6: x,y,z,px,py,pz   7: + pid
struct alignas(128) TileStage {
    double v[6][kTile];
    uint32_t pid[NARR == 7 ? kTile : 1];
};

template <int NARR>
__device__ __forceinline__ void stage_issue(TileStage<NARR> &st, uint64_t *bar, const Soa &in, int64_t n, int64_t tile)
{
    const int64_t base = tile * kTile;
    if (base + kTile <= n) {                      // full tile: one elected thread issues the bulk copies
        if (threadIdx.x == 0) {
            mbar_expect_tx(bar, 6 * kTile * 8 + (NARR == 7 ? kTile * 4 : 0));
            bulk_g2s(st.v[0], in.x + base, kTile * 8, bar);
            bulk_g2s(st.v[1], in.y + base, kTile * 8, bar);
            bulk_g2s(st.v[2], in.z + base, kTile * 8, bar);
            bulk_g2s(st.v[3], in.px + base, kTile * 8, bar);
            bulk_g2s(st.v[4], in.py + base, kTile * 8, bar);
            bulk_g2s(st.v[5], in.pz + base, kTile * 8, bar);
            if (NARR == 7) bulk_g2s(st.pid, in.pid + base, kTile * 4, bar);
        }
    } else {                                      // ragged tail: plain loads by everybody
        for (int li = threadIdx.x; li < kTile; li += kTileThreads) {
            const int64_t i = base + li;
            if (i < n) {
                st.v[0][li] = in.x[i]; st.v[1][li] = in.y[i]; st.v[2][li] = in.z[i];
                st.v[3][li] = in.px[i]; st.v[4][li] = in.py[i]; st.v[5][li] = in.pz[i];
                if (NARR == 7) st.pid[li] = in.pid[i];
            }
        }
    }
}

template <int NARR>
__device__ __forceinline__ void stage_wait(uint64_t *bar, uint32_t parity, int64_t n, int64_t tile)
{
    if (tile * kTile + kTile <= n) mbar_wait(bar, parity);
    else __syncthreads();
}

// ---- K_A ------------------------------------------------------------------------------
__global__ void __launch_bounds__(kTileThreads, 4)
k_stream_hist(Geom g, double dt, int64_t n, int64_t ntiles, Soa in, uint32_t *__restrict__ cnt,
              uint32_t *__restrict__ tile_rec, uint32_t *__restrict__ flags)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    TileStage<6> *stage = reinterpret_cast<TileStage<6> *>(smem_raw);
    __shared__ __align__(8) uint64_t s_bar[2];
    __shared__ uint32_t s_tail[kDirs];
    __shared__ uint32_t s_cf, s_cl;
    const int tid = threadIdx.x;
    if (tid == 0) { mbar_init(&s_bar[0], 1); mbar_init(&s_bar[1], 1); mbar_fence_init(); }
    __syncthreads();
    int64_t tile = blockIdx.x;
    if (tile < ntiles) stage_issue<6>(stage[0], &s_bar[0], in, n, tile);
    for (int it = 0; tile < ntiles; ++it, tile += gridDim.x) {
        const int b = it & 1;
        const int64_t next = tile + gridDim.x;
        if (next < ntiles) stage_issue<6>(stage[b ^ 1], &s_bar[b ^ 1], in, n, next);
        if (tid < kDirs) s_tail[tid] = 0;
        stage_wait<6>(&s_bar[b], (uint32_t)((it >> 1) & 1), n, tile);
        const TileStage<6> &st = stage[b];
        const int64_t base = tile * kTile;
        const int64_t last = min(n, base + kTile) - 1;
        uint32_t c_old[kTileItems];
        int d[kTileItems];
#pragma unroll
        for (int j = 0; j < kTileItems; ++j) {
            const int li = j * kTileThreads + tid;
            const int64_t i = base + li;
            const bool valid = i < n;
            c_old[j] = 0; d[j] = -1;
            const uint32_t active = __ballot_sync(0xFFFFFFFFu, valid);
            if (valid) {
                Moved m = move_particle(g, dt, st.v[0][li], st.v[1][li], st.v[2][li], st.v[3][li], st.v[4][li], st.v[5][li]);
                c_old[j] = m.c_old; d[j] = m.d;
                if (m.d < 0) atomicOr(flags, kFlagMoved);
                const uint32_t key = (uint32_t)max(m.d, 0) * g.ncells + m.c_old;
                const uint32_t peers = __match_any_sync(active, key);
                if ((peers & lanemask_lt()) == 0) atomicAdd(&cnt[key], (uint32_t)__popc(peers));
                if (i == base) s_cf = m.c_old;
                if (i == last) s_cl = m.c_old;
            }
        }
        __syncthreads();
        const uint32_t cl = s_cl;
        // tail record: how many particles of the tile's LAST cell, per direction (feeds K_carry)
#pragma unroll
        for (int j = 0; j < kTileItems; ++j) {
            const int64_t i = base + j * kTileThreads + tid;
            const bool mine = (i < n) && c_old[j] == cl;
            const uint32_t active = __ballot_sync(0xFFFFFFFFu, mine);
            if (mine) {
                const int dd = max(d[j], 0);
                const uint32_t peers = __match_any_sync(active, dd);
                if ((peers & lanemask_lt()) == 0) atomicAdd(&s_tail[dd], (uint32_t)__popc(peers));
            }
        }
        __syncthreads();
        uint32_t *rec = tile_rec + (size_t)tile * kTileRec;
        if (tid < kDirs) rec[tid] = s_tail[tid];
        if (tid == 27) rec[27] = s_cf;
        if (tid == 28) rec[28] = s_cl;
        __syncthreads();   // stage b and s_tail are free again
    }
}

// ---- K_B ------------------------------------------------------------------------------
// A block owns 256 NEW cells (the unit of the block-sum scan); each of its 32 warps takes 8 of
// them, lane q < 27 the q-th source.  Sources in ascending linear index (x slowest) == ascending
// previous array position, which is what makes the placement stable (A8).  The 8 gathers of a
// lane are issued together; a warp scan turns the counts into exclusive offsets.
constexpr int kGatherThreads = 1024;
constexpr int kGatherCellsPerWarp = 256 / (kGatherThreads / 32);

__global__ void __launch_bounds__(kGatherThreads)
k_gather(Geom g, uint32_t *__restrict__ cnt, uint32_t *__restrict__ count_new,
         uint32_t *__restrict__ block_sum)
{
    __shared__ uint32_t s_warp[kGatherThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int ox = lane / 9 - 1, oy = (lane / 3) % 3 - 1, oz = lane % 3 - 1;   // source = new cell + o
    const int dcode = (1 - ox) * 9 + (1 - oy) * 3 + (1 - oz);                  // the source moved by -o
    uint32_t v[kGatherCellsPerWarp];
    size_t e[kGatherCellsPerWarp];
    bool ok[kGatherCellsPerWarp];
#pragma unroll
    for (int k = 0; k < kGatherCellsPerWarp; ++k) {
        const uint32_t c = blockIdx.x * 256u + wid * kGatherCellsPerWarp + k;
        const int sz = (int)(c % (uint32_t)g.nc[2]) + oz;
        const int sy = (int)((c / (uint32_t)g.nc[2]) % (uint32_t)g.nc[1]) + oy;
        const int sx = (int)(c / ((uint32_t)g.nc[2] * (uint32_t)g.nc[1])) + ox;
        ok[k] = lane < kDirs && c < g.ncells && sx >= 0 && sx < g.nc[0] && sy >= 0 && sy < g.nc[1] && sz >= 0 && sz < g.nc[2];
        e[k] = ok[k] ? (size_t)dcode * g.ncells + cell_linear(g, sx, sy, sz) : 0;
        v[k] = ok[k] ? cnt[e[k]] : 0u;
    }
    uint32_t wsum = 0;
#pragma unroll
    for (int k = 0; k < kGatherCellsPerWarp; ++k) {
        const uint32_t c = blockIdx.x * 256u + wid * kGatherCellsPerWarp + k;
        uint32_t inc = v[k];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
            if (lane >= o) inc += t;
        }
        if (ok[k]) cnt[e[k]] = inc - v[k];
        const uint32_t total = __shfl_sync(0xFFFFFFFFu, inc, 31);
        if (lane == 0 && c < g.ncells) count_new[c] = total;
        wsum += total;
    }
    if (lane == 0) s_warp[wid] = wsum;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < kGatherThreads / 32; ++w) t += s_warp[w];
        block_sum[blockIdx.x] = t;
    }
}

// ---- K_S: exclusive scan of the per-block sums (one CTA), also resets the per-step
// work counters of the collision kernels ------------------------------------------------
__global__ void __launch_bounds__(1024)
k_scan_blocks(uint32_t *__restrict__ block_sum, int nblocks, uint32_t *__restrict__ zero_me, int nzero)
{
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_carry;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid < nzero) zero_me[tid] = 0;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (int b0 = 0; b0 < nblocks; b0 += 1024) {
        const int i = b0 + tid;
        const uint32_t v = (i < nblocks) ? block_sum[i] : 0u;
        uint32_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_warp[wid] = inc;
        __syncthreads();
        if (wid == 0) {
            uint32_t w = s_warp[lane], winc = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, winc, o);
                if (lane >= o) winc += t;
            }
            s_warp[lane] = winc - w;   // exclusive over warps
        }
        __syncthreads();
        const uint32_t carry = s_carry;
        if (i < nblocks) block_sum[i] = carry + s_warp[wid] + inc - v;
        __syncthreads();
        if (tid == 1023) s_carry = carry + s_warp[wid] + inc;
        __syncthreads();
    }
}

// ---- K_F: cell_start = block prefix + local exclusive scan; cells with n >= 2 are appended
// to the work list of their size class for the collision kernels -------------------------
constexpr int kNumClasses = 8;   // 7 shared-memory classes + the global-memory overflow class

struct ClassTable {
    uint32_t max_n[kNumClasses];   // inclusive upper bound of each class (last = UINT32_MAX)
    uint32_t c_lo, c_hi;           // cells [c_lo, c_hi) are collided (x-slab decomposition: the owned layers; else all)
};

__global__ void __launch_bounds__(256)
k_cell_start(uint32_t ncells, const uint32_t *__restrict__ count_new,
             const uint32_t *__restrict__ block_prefix, uint32_t *__restrict__ cell_start,
             ClassTable ct, uint32_t *__restrict__ class_count, uint4 *__restrict__ class_list,
             unsigned long long *__restrict__ max_occ, uint32_t *__restrict__ step_max)
{
    __shared__ uint32_t s_warp[8];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const uint32_t c = blockIdx.x * 256u + tid;
    const uint32_t v = (c < ncells) ? count_new[c] : 0u;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
        if (lane >= o) inc += t;
    }
    if (lane == 31) s_warp[wid] = inc;
    __syncthreads();
    uint32_t wpre = 0;
    for (int w = 0; w < wid; ++w) wpre += s_warp[w];
    const uint32_t start = block_prefix[blockIdx.x] + wpre + inc - v;
    if (c < ncells) {
        cell_start[c] = start;
        if (c == ncells - 1) cell_start[ncells] = start + v;
    }
    // size class (warp-aggregated append; the list order does not affect any result).  Cells with
    // a single particle have no pair but take part in the fused histogram of the next step.
    int k = -1;
    if (v >= 1 && c >= ct.c_lo && c < ct.c_hi) {
        k = 0;
        while (v > ct.max_n[k]) ++k;
    }
    const uint32_t peers = __match_any_sync(0xFFFFFFFFu, k);
    if (k >= 0) {
        const int leader = __ffs(peers) - 1;
        uint32_t pos = 0;
        if (lane == leader) pos = atomicAdd(&class_count[k], (uint32_t)__popc(peers));
        pos = __shfl_sync(peers, pos, leader) + __popc(peers & lanemask_lt());
        class_list[(size_t)k * ncells + pos] = make_uint4(c, start, v, 0u);   // {cell, first slot, population}: no dependent loads in the consumer
    }
    uint32_t vmax = v;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vmax = max(vmax, __shfl_xor_sync(0xFFFFFFFFu, vmax, o));
    if (lane == 0 && vmax > 0) {
        atomicMax(max_occ, (unsigned long long)vmax);   // since cuba_init (cuba_counters)
        atomicMax(step_max, vmax);                      // of this binning (cleared per step; feeds the variable time step)
    }
}

// ---- K_D: dest_base[d][c_old] = cell_start[c_new(c_old, d)] + off[d][c_old], in place ------
// One thread per (direction, old cell): the scatter then needs a single table gather per
// particle, which it can issue as soon as the direction is known.
__global__ void __launch_bounds__(256)
k_dest_base(Geom g, uint32_t *__restrict__ off, const uint32_t *__restrict__ cell_start)
{
    const uint32_t c = blockIdx.x * 256u + threadIdx.x;
    const int d = blockIdx.y;
    if (c >= g.ncells) return;
    const int iz = (int)(c % (uint32_t)g.nc[2]) + d % 3 - 1;
    const int iy = (int)((c / (uint32_t)g.nc[2]) % (uint32_t)g.nc[1]) + (d / 3) % 3 - 1;
    const int ix = (int)(c / ((uint32_t)g.nc[2] * (uint32_t)g.nc[1])) + d / 9 - 1;
    if (ix < 0 || ix >= g.nc[0] || iy < 0 || iy >= g.nc[1] || iz < 0 || iz >= g.nc[2]) return;   // no particle goes there
    off[(size_t)d * g.ncells + c] += cell_start[cell_linear(g, ix, iy, iz)];
}

// ---- K_carry ---------------------------------------------------------------------------
// carry[b][d] = number of particles with (cell = first cell of tile b, direction d) that sit in
// tiles before b.  One warp per tile (lane = d).  A tile starts a walk for its last cell
// unless it lies in the middle of that cell's run; the walk is linear in the run length.
__global__ void __launch_bounds__(256)
k_carry(int ntiles, const uint32_t *__restrict__ tile_rec, uint32_t *__restrict__ carry)
{
    const int lane = threadIdx.x & 31;
    const int b = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (b >= ntiles || lane >= kDirs) return;
    const uint32_t *rec = tile_rec + (size_t)b * kTileRec;
    const uint32_t cf = rec[27], cl = rec[28];
    const bool has_carry = b > 0 && tile_rec[(size_t)(b - 1) * kTileRec + 28] == cf;
    if (!has_carry) carry[(size_t)b * kTileRec + lane] = 0;
    const bool middle = has_carry && cf == cl;
    if (middle) return;
    uint32_t acc = rec[lane];
    for (int bb = b + 1; bb < ntiles; ++bb) {
        const uint32_t *r2 = tile_rec + (size_t)bb * kTileRec;
        if (r2[27] != cl) break;
        carry[(size_t)bb * kTileRec + lane] = acc;
        if (r2[28] != cl) break;
        acc += r2[lane];
    }
}

// ---- K_C ------------------------------------------------------------------------------
// Rows are the 32 consecutive particles one warp handles for one item; row r = j*8 + warp,
// local index li = r*32 + lane = j*256 + tid.  prefix_d(li) = number of particles before li
// in the tile that moved in direction d.  Stable rank inside (c_old, d) =
// prefix_d(li) - prefix_d(first particle of c_old in the tile) [+ carry if that is li 0].
#ifndef CUBA_SCAT_MB   // resident CTAs per SM asked for the scatter (build-time tunable; 4 needs <= 64 registers)
#define CUBA_SCAT_MB 3
#endif
template <bool WITH_CELL_OF_PID>
__global__ void __launch_bounds__(kTileThreads, CUBA_SCAT_MB)
k_scatter(Geom g, double dt, int64_t n, int64_t ntiles, Soa in, Soa out, const uint32_t *__restrict__ dest_base,
          const uint32_t *__restrict__ carry, uint32_t *__restrict__ cell_of_pid)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    TileStage<7> *stage = reinterpret_cast<TileStage<7> *>(smem_raw);
    __shared__ __align__(8) uint64_t s_bar[2];
    __shared__ uint32_t s_rowlast[kTileRows];   // old cell of the last particle of every row (its successor is lane 0 of the next row)
    __shared__ uint32_t s_ball[kTileRows][kDirs];
    __shared__ uint32_t s_pref[kTileRows][kDirs];
    __shared__ uint32_t s_head[kTileRows];
    __shared__ int s_lasthead[kTileRows];
    __shared__ uint32_t s_carry[32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) { mbar_init(&s_bar[0], 1); mbar_init(&s_bar[1], 1); mbar_fence_init(); }
    __syncthreads();
    int64_t tile = blockIdx.x;
    if (tile < ntiles) stage_issue<7>(stage[0], &s_bar[0], in, n, tile);
    for (int it = 0; tile < ntiles; ++it, tile += gridDim.x) {
        const int b = it & 1;
        const int64_t next = tile + gridDim.x;
        if (next < ntiles) stage_issue<7>(stage[b ^ 1], &s_bar[b ^ 1], in, n, next);
        stage_wait<7>(&s_bar[b], (uint32_t)((it >> 1) & 1), n, tile);
        const TileStage<7> &st = stage[b];
        const int64_t base = tile * kTile;

        Moved m[kTileItems];
        uint32_t dbase[kTileItems];   // cell_start[c_new] + off[d][c_old]: gathered now, used after the ranking
        if (tid < kDirs) s_carry[tid] = carry[(size_t)tile * kTileRec + tid];
        for (int e = tid; e < kTileRows * kDirs; e += kTileThreads) (&s_ball[0][0])[e] = 0;
#pragma unroll
        for (int j = 0; j < kTileItems; ++j) {
            const int li = j * kTileThreads + tid;
            m[j].d = -1; m[j].c_old = 0xFFFFFFFFu;
            if (base + li < n)
                m[j] = move_particle(g, dt, st.v[0][li], st.v[1][li], st.v[2][li], st.v[3][li], st.v[4][li], st.v[5][li]);
            if (lane == 31) s_rowlast[j * (kTileThreads / 32) + wid] = m[j].c_old;
            dbase[j] = (m[j].d >= 0) ? dest_base[(size_t)m[j].d * g.ncells + m[j].c_old] : 0u;
        }
        __syncthreads();
#pragma unroll
        for (int j = 0; j < kTileItems; ++j) {
            const int r = j * (kTileThreads / 32) + wid;
            const int li = j * kTileThreads + tid;
            const bool valid = (base + li) < n;
            const int dd = m[j].d;
            // one bit mask per direction present in the row (absent directions stay zero)
            const uint32_t peers = __match_any_sync(0xFFFFFFFFu, dd);
            if (dd >= 0 && (peers & lanemask_lt()) == 0) s_ball[r][dd] = peers;
            // the predecessor's old cell: the lane below, for lane 0 the last lane of the previous row (2 KB of
            // shared memory less than a per-particle table: four CTAs fit an SM with it)
            uint32_t prev = __shfl_up_sync(0xFFFFFFFFu, m[j].c_old, 1);
            if (lane == 0) prev = r > 0 ? s_rowlast[r - 1] : 0xFFFFFFFFu;
            const bool head = valid && (li == 0 || prev != m[j].c_old);
            const uint32_t hb = __ballot_sync(0xFFFFFFFFu, head);
            if (lane == 0) s_head[r] = hb;
        }
        __syncthreads();
        if (tid < kDirs) {
            uint32_t run = 0;
#pragma unroll
            for (int r = 0; r < kTileRows; ++r) {
                s_pref[r][tid] = run;
                run += __popc(s_ball[r][tid]);
            }
        } else if (tid == 32) {
            int lh = -1;
#pragma unroll
            for (int r = 0; r < kTileRows; ++r) {
                s_lasthead[r] = lh;
                const uint32_t hb = s_head[r];
                if (hb) lh = r * 32 + 31 - __clz(hb);
            }
        }
        __syncthreads();
#pragma unroll
        for (int j = 0; j < kTileItems; ++j) {
            const int li = j * kTileThreads + tid;
            if ((base + li) >= n) continue;
            const int dd = m[j].d;
            if (dd < 0) continue;   // flagged by K_A; the particle is dropped from the placement
            const int r = j * (kTileThreads / 32) + wid;
            const uint32_t pre_i = s_pref[r][dd] + __popc(s_ball[r][dd] & lanemask_lt());
            const uint32_t hm = s_head[r] & lanemask_le();
            const int sli = hm ? (r * 32 + 31 - __clz(hm)) : s_lasthead[r];
            const int rs = sli >> 5, ls = sli & 31;
            const uint32_t pre_s = s_pref[rs][dd] + __popc(s_ball[rs][dd] & ((1u << ls) - 1u));
            uint32_t rank = pre_i - pre_s;
            if (sli == 0) rank += s_carry[dd];
            const uint32_t dest = dbase[j] + rank;
            const uint32_t id = st.pid[li];
            // (measured, no effect: L2 evict-last / evict-first cache hints on the movers' / stayers' stores)
            out.x[dest] = m[j].x; out.y[dest] = m[j].y; out.z[dest] = m[j].z;
            out.px[dest] = m[j].px; out.py[dest] = m[j].py; out.pz[dest] = m[j].pz;
            out.pid[dest] = id;
            if (WITH_CELL_OF_PID) cell_of_pid[id] = m[j].c_new;
        }
        __syncthreads();   // stage b and the ballot tables are free again
    }
}

}  // namespace cuba
