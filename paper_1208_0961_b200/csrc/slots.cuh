// slots.cuh -- the whole step (S1-S5) as ONE kernel per step on a slotted particle store.
//
// The compact store of bin.cuh needs a global prefix sum between the collisions of step t and the
// placement of step t+1 (cell_start of the new binning), hence a separate placement pass over the
// whole store (k_scatter: 104 B per particle) and, because that pass is HBM bound while the collision
// kernels are bound by instruction issue and latency, two passes that cannot use the machine together.
// Here every cell owns a fixed region of SLOTS particle slots, divided into 27 INBOX SEGMENTS, one per
// source cell (the cell itself, code 13, and its 26 neighbours), in two parity copies:
//
//   segment s = (sx, sy, sz) of cell c holds, in stable order, the particles that came from cell
//   c + (sx-1, sy-1, sz-1) in the last step; cnt[c][s] says how many.
//
// One CTA per cell (the size classes of collide.cuh):
//   assemble   the cell from its 27 segments taken in ascending s = ascending source-cell index --
//              which IS the order of the stable counting sort (A8): within a segment the particles sit
//              in the order of their previous array index, because the source wrote them at their
//              stable rank;
//   collide    all R rounds on chip (run_sweeps of collide.cuh, unchanged);
//   stream     S1-S3 exactly (the arithmetic of move_particle), direction d of every particle;
//   rank       stably inside each of the 27 directions from one match.any per row of 32 particles
//              and a prefix over the rows -- no atomics touch the order;
//   write      the particle at rank r of direction d goes to slot r of segment 26-d of the
//              destination cell's OTHER parity copy; the 27 counts follow.
// No histogram, no scan, no cell_start, no placement pass: the step reads 52 B and writes 52 B per
// particle (the compulsory floor of SURVEY.md 8(d)).  Segment capacities are sized from the fullest
// cell and dt / cell edge with a wide margin; an overflow (or a cell beyond the largest shared-memory
// class) raises a flag and the host replays the affected steps on the compact path from the state it
// kept (cuba_api.cu), so the result never depends on the capacities.
// k_slot_unpack / k_slot_pack convert between the compact store (what every other entry point and
// cuba_get_particles use: the oracle's array order) and the slotted one.
#pragma once
#include "collide.cuh"

namespace cuba {

constexpr uint32_t kFlagSlots = 16u;   // a segment or a cell outgrew the slotted layout: replay on the compact path

struct SlotGeom {
    uint32_t slots;              // slots per cell
    uint32_t seg_off[kDirs + 1]; // first slot of segment s inside the cell's region; seg_off[27] = slots
};

struct SlotStore {
    double *x, *y, *z, *px, *py, *pz;   // [ncells * slots]
    uint32_t *pid;
    uint32_t *cnt;                      // [ncells][27]
};

struct SlotParams {
    SlotGeom sg;
    SlotStore in, out;          // this step reads `in`, writes `out`
    double dt;
};

// neighbour of cell (i0,i1,i2) in direction code d, or -1 outside the box
__device__ __forceinline__ int slot_neighbour(const Geom &g, int i0, int i1, int i2, int d)
{
    const int j0 = i0 + d / 9 - 1, j1 = i1 + (d / 3) % 3 - 1, j2 = i2 + d % 3 - 1;
    if (j0 < 0 || j0 >= g.nc[0] || j1 < 0 || j1 >= g.nc[1] || j2 < 0 || j2 >= g.nc[2]) return -1;
    return (int)cell_linear(g, j0, j1, j2);
}

// ---- per step: populations, size classes; empty cells send nothing ---------------------------------
__global__ void __launch_bounds__(256)
k_slot_classify(Geom g, const uint32_t *__restrict__ cnt_in, uint32_t *__restrict__ cnt_out, ClassTable ct,
                uint32_t *__restrict__ class_count, uint4 *__restrict__ class_list,
                unsigned long long *__restrict__ max_occ, uint32_t *__restrict__ step_max, uint32_t *__restrict__ flags,
                const uint32_t *__restrict__ cell_start)   // non-null in the first pass: the cells are taken from the compact store
{
    const int lane = threadIdx.x & 31;
    const uint32_t c = blockIdx.x * 256u + threadIdx.x;
    uint32_t v = 0;
    if (c < g.ncells) {
#pragma unroll
        for (int s = 0; s < kDirs; ++s) v += cnt_in[(size_t)c * kDirs + s];
        if (v == 0) {      // nobody works on an empty cell: its outgoing counts are written here
            const int i2 = (int)(c % (uint32_t)g.nc[2]);
            const int i1 = (int)((c / (uint32_t)g.nc[2]) % (uint32_t)g.nc[1]);
            const int i0 = (int)(c / ((uint32_t)g.nc[2] * (uint32_t)g.nc[1]));
            for (int d = 0; d < kDirs; ++d) {
                const int nb = slot_neighbour(g, i0, i1, i2, d);
                if (nb >= 0) cnt_out[(size_t)nb * kDirs + (kDirs - 1 - d)] = 0;
            }
        }
    }
    int k = -1;
    if (v >= 1) {
        k = 0;
        while (v > ct.max_n[k]) ++k;
        if (k == kNumClasses - 1) { atomicOr(flags, kFlagSlots); k = -1; }   // beyond the shared-memory classes
    }
    const uint32_t peers = __match_any_sync(0xFFFFFFFFu, k);
    if (k >= 0) {
        const int leader = __ffs(peers) - 1;
        uint32_t pos = 0;
        if (lane == leader) pos = atomicAdd(&class_count[k], (uint32_t)__popc(peers));
        pos = __shfl_sync(peers, pos, leader) + __popc(peers & lanemask_lt());
        class_list[(size_t)k * g.ncells + pos] = make_uint4(c, cell_start ? cell_start[c] : 0u, v, 0u);
    }
    uint32_t vmax = v;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vmax = max(vmax, __shfl_xor_sync(0xFFFFFFFFu, vmax, o));
    if (lane == 0 && vmax > 0) {
        atomicMax(max_occ, (unsigned long long)vmax);
        atomicMax(step_max, vmax);
    }
}

// ---- per-cell tables of the step kernel (static shared memory) -------------------------------------
struct SlotCell {
    uint32_t seg_start[kDirs + 1];   // exclusive prefix of the 27 segment populations (assembly order)
    uint32_t src_base[kDirs];        // first slot of segment s of this cell in the `in` copy
    uint32_t dst_base[kDirs];        // direction d: first slot of segment 26-d of the destination cell in `out`
    uint32_t dst_cap[kDirs];         // its capacity (0: no such neighbour)
    uint32_t dst_cnt[kDirs];         // index of its count in out.cnt (0xFFFFFFFF: no such neighbour)
    uint32_t total[kDirs];           // particles of this cell leaving in direction d
};

// slot index (in the `in` copy) of the particle at assembly position j
__device__ __forceinline__ uint32_t slot_source(const SlotCell *t, uint32_t j)
{
    uint32_t s = kDirStay;
    if (j < t->seg_start[kDirStay] || j >= t->seg_start[kDirStay + 1]) {
        s = 0;
#pragma unroll
        for (uint32_t step = 16; step; step >>= 1)
            if (s + step < (uint32_t)kDirs && t->seg_start[s + step] <= j) s += step;
    }
    return t->src_base[s] + (j - t->seg_start[s]);
}

// Tail scratch in the dynamic shared memory (all dead by then): the duplicate counters' space holds the
// row masks [rows][27], the lists' space their prefixes (16 bit), the orders' space the direction codes.
template <int CAP, int LCAP>
struct SlotTail {
    using S = CellSmem<CAP, LCAP>;
    static __device__ __forceinline__ uint32_t *ball() { return S::cnt(); }                                      // [rows][27] <= CAP words
    static __device__ __forceinline__ uint16_t *pref() { return reinterpret_cast<uint16_t *>(S::lkey(0)); }      // [rows][27] 16 bit <= 12 LCAP bytes... checked below
    static __device__ __forceinline__ uint16_t *dir() { return S::ord(0); }                                      // [CAP]
};

// What a pass does.  A call of n steps is n + 1 passes: the first one takes the cells from the compact store and
// only streams (the compact state is the state after the collisions of the previous step); the middle ones
// collide and stream; the last one collides and writes the compact store (its cell_start is known beforehand:
// collisions move nobody).
enum SlotMode { kSlotMiddle = 0, kSlotFirst = 1, kSlotLast = 2 };

template <int THREADS, int ITEMS, int G, int CAP, int LCAP, int MODE>
__device__ __forceinline__ void step_cell_slots(const CollideParams &P, const SlotParams &Q, uint32_t c, uint32_t lo, uint32_t n,
                                                uint32_t *s_warp, CtaStats *stats, SlotCell *tab, ThreadStats &acc,
                                                uint32_t c_next, uint32_t lo_next, uint32_t n_next)
{
    using S = CellSmem<CAP, LCAP>;
    using T = SlotTail<CAP, LCAP>;
    constexpr int W = THREADS / 32, ROWS = ITEMS * W;
    static_assert(ROWS * kDirs <= CAP, "row masks fit the duplicate counters' space");
    static_assert(ROWS * kDirs * 2 <= 24 * LCAP, "row prefixes fit the lists' space");
    constexpr bool COLLIDE = MODE != kSlotFirst, STREAM = MODE != kSlotLast, FROM_SLOTS = MODE != kSlotFirst;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const uint32_t tcur = P.t;
    int R = 0;
    if (COLLIDE) {
        const double base = P.base;
        const double cn = (n & 1u) ? (double)n : (double)(n - 1u);
        const double pmax = (2.0 * cn) * base;
        if (!(pmax <= 64.0)) { if (tid == 0) atomicOr(P.flags, kFlagRounds); R = 64; }
        else R = (pmax <= 1.0) ? 1 : (int)ceil(pmax);
        if (n < 2u) R = 0;
        for (int e = tid; e < 2 * kChains; e += THREADS) (&stats->head[0][0])[e] = kNil;
        if (tid == 0) {
            stats->nlist[0] = 0; stats->nlist[1] = 0;
            const double scale = (cn * base) / (double)R;
            stats->scale = scale; stats->hscale = 0.5 * scale;
        }
    }
    // ---- per-cell tables (warp 0) --------------------------------------------------------------------
    if (tid < 32) {
        const int i2 = (int)(c % (uint32_t)P.g.nc[2]);
        const int i1 = (int)((c / (uint32_t)P.g.nc[2]) % (uint32_t)P.g.nc[1]);
        const int i0 = (int)(c / ((uint32_t)P.g.nc[2] * (uint32_t)P.g.nc[1]));
        if (STREAM) hist_cell_setup(P.g, c, &stats->h, tid);
        if (FROM_SLOTS) {
            const uint32_t v = lane < kDirs ? Q.in.cnt[(size_t)c * kDirs + lane] : 0u;
            uint32_t inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
                if (lane >= o) inc += t;
            }
            if (lane <= kDirs) tab->seg_start[lane] = inc - v;       // lane 27: the total
            if (lane < kDirs) tab->src_base[lane] = c * Q.sg.slots + Q.sg.seg_off[lane];
        }
        if (STREAM && lane < kDirs) {
            const int nb = slot_neighbour(P.g, i0, i1, i2, lane);
            const int seg = kDirs - 1 - lane;
            tab->dst_base[lane] = nb >= 0 ? (uint32_t)nb * Q.sg.slots + Q.sg.seg_off[seg] : 0u;
            tab->dst_cap[lane] = nb >= 0 ? Q.sg.seg_off[seg + 1] - Q.sg.seg_off[seg] : 0u;
            tab->dst_cnt[lane] = nb >= 0 ? (uint32_t)nb * kDirs + (uint32_t)seg : 0xFFFFFFFFu;
        }
    }
    __syncthreads();
    const uint32_t last = n - 1u;
    double *sE = S::E();
    // ---- assemble: momenta and pids (from the 27 segments in order); clear the sort structures ---------
#pragma unroll
    for (int g = 0; g < ITEMS / G; ++g) {
        if ((uint32_t)(g * G * THREADS) >= n) break;
        double a[G], b[G], cc[G];
        uint32_t id[G];
#pragma unroll
        for (int i = 0; i < G; ++i) {
            const uint32_t jc = min((uint32_t)(tid + (g * G + i) * THREADS), last);
            const uint32_t src = FROM_SLOTS ? slot_source(tab, jc) : lo + jc;
            a[i] = Q.in.px[src]; b[i] = Q.in.py[src]; cc[i] = Q.in.pz[src]; id[i] = Q.in.pid[src];
        }
#pragma unroll
        for (int i = 0; i < G; ++i) {
            const uint32_t j = tid + (g * G + i) * THREADS;
            if (j < n) {
                S::pxy()[j] = make_double2(a[i], b[i]); S::pz()[j] = cc[i]; S::pid()[j] = id[i];
                if (COLLIDE) { *reinterpret_cast<uint2 *>(S::bm() + 2 * j) = make_uint2(0u, 0u); S::cnt()[j] = 0; }
                else sE[j] = energy(a[i], b[i], cc[i]);
            }
        }
    }
    __syncthreads();
    // the CTA's next cell goes to L2 while this one is processed (its own segment holds most of it)
    if (n_next) {
        const uint32_t b0 = FROM_SLOTS ? c_next * Q.sg.slots + Q.sg.seg_off[kDirStay] : lo_next;
        for (uint32_t l = tid * 16u; l < n_next + 16u; l += THREADS * 16u) {
            const uint32_t e = b0 + min(l, n_next - 1u);
            prefetch_l2(Q.in.px + e); prefetch_l2(Q.in.py + e); prefetch_l2(Q.in.pz + e);
            prefetch_l2(Q.in.x + e); prefetch_l2(Q.in.y + e); prefetch_l2(Q.in.z + e);
            if ((l & 16u) == 0) prefetch_l2(Q.in.pid + e);
        }
    }
    if (COLLIDE) {
        const uint32_t warp_hits = run_sweeps<THREADS, ITEMS, G, CAP, LCAP, false>(P, c, n, R, tcur, STREAM, s_warp, stats);
        if (STREAM && R == 0 && tid == 0) {     // a lone particle: no pair phase has computed its energy
            const double2 xy = S::pxy()[0];
            sE[0] = energy(xy.x, xy.y, S::pz()[0]);
        }
        __syncthreads();
        acc.hits += warp_hits;
        acc.pairs += (unsigned long long)R * (n >> 1);
        acc.rounds += (unsigned long long)R;
    }
    constexpr int HB = (ITEMS % 2 == 0) ? 2 : 1;
    if (!STREAM) {
        // ---- last pass: the cell goes to its place in the compact store, positions unchanged -----------
#pragma unroll 1
        for (int g = 0; g < ITEMS / HB; ++g) {
            if ((uint32_t)(g * HB * THREADS) >= n) break;
            double xx[HB], yy[HB], zz[HB];
#pragma unroll
            for (int i = 0; i < HB; ++i) {
                const uint32_t src = slot_source(tab, min((uint32_t)(tid + (g * HB + i) * THREADS), last));
                xx[i] = Q.in.x[src]; yy[i] = Q.in.y[src]; zz[i] = Q.in.z[src];
            }
#pragma unroll
            for (int i = 0; i < HB; ++i) {
                const uint32_t j = tid + (g * HB + i) * THREADS;
                if (j < n) {
                    const double2 xy = S::pxy()[j];
                    const uint32_t dst = lo + j;
                    Q.out.x[dst] = xx[i]; Q.out.y[dst] = yy[i]; Q.out.z[dst] = zz[i];
                    Q.out.px[dst] = xy.x; Q.out.py[dst] = xy.y; Q.out.pz[dst] = S::pz()[j];
                    Q.out.pid[dst] = S::pid()[j];
                }
            }
        }
        return;
    }

    // ---- tail, pass 1: direction of every particle; one mask per row of 32 and direction --------------
    for (int e = tid; e < ROWS * kDirs; e += THREADS) T::ball()[e] = 0;
    __syncthreads();
    const HistCell &hc = stats->h;
#pragma unroll 1
    for (int g = 0; g < ITEMS / HB; ++g) {
        if ((uint32_t)(g * HB * THREADS) >= n) break;
        double xx[HB], yy[HB], zz[HB];
#pragma unroll
        for (int i = 0; i < HB; ++i) {
            const uint32_t jc = min((uint32_t)(tid + (g * HB + i) * THREADS), last);
            const uint32_t src = FROM_SLOTS ? slot_source(tab, jc) : lo + jc;
            xx[i] = Q.in.x[src]; yy[i] = Q.in.y[src]; zz[i] = Q.in.z[src];
        }
#pragma unroll
        for (int i = 0; i < HB; ++i) {
            const int it = g * HB + i;
            const uint32_t j = tid + it * THREADS, jj = min(j, last);
            const double2 xy = S::pxy()[jj];
            int d = next_direction_guarded(P.g, Q.dt, hc, xx[i], yy[i], zz[i], xy.x, xy.y, S::pz()[jj], sE[jj]);
            if (j >= n) d = 31;                                   // not a particle
            else if (d < 0) { atomicOr(P.flags, kFlagMoved); d = 30; }   // dropped from the placement, as in k_scatter
            const uint32_t peers = __match_any_sync(0xFFFFFFFFu, d);
            if (d < kDirs && (peers & lanemask_lt()) == 0) T::ball()[(it * W + wid) * kDirs + d] = peers;
            if (j < n) T::dir()[j] = (uint16_t)d;
        }
    }
    __syncthreads();
    // ---- prefix of the row masks per direction (27 threads walk the rows) ------------------------------
    if (tid < kDirs) {
        uint32_t run = 0;
#pragma unroll 4
        for (int r = 0; r < ROWS; ++r) {
            T::pref()[r * kDirs + tid] = (uint16_t)run;
            run += __popc(T::ball()[r * kDirs + tid]);
        }
        tab->total[tid] = run;
        if (tab->dst_cnt[tid] != 0xFFFFFFFFu) Q.out.cnt[tab->dst_cnt[tid]] = min(run, tab->dst_cap[tid]);
        if (run > tab->dst_cap[tid]) atomicOr(P.flags, kFlagSlots);          // capacity: the host redoes the run on the compact path
    }
    __syncthreads();
    // ---- tail, pass 2: S1-S2 exactly, stable rank, write into the destination's inbox -------------------
#pragma unroll 1
    for (int g = 0; g < ITEMS / HB; ++g) {
        if ((uint32_t)(g * HB * THREADS) >= n) break;
        double xx[HB], yy[HB], zz[HB];
#pragma unroll
        for (int i = 0; i < HB; ++i) {
            const uint32_t jc = min((uint32_t)(tid + (g * HB + i) * THREADS), last);
            const uint32_t src = FROM_SLOTS ? slot_source(tab, jc) : lo + jc;
            xx[i] = Q.in.x[src]; yy[i] = Q.in.y[src]; zz[i] = Q.in.z[src];
        }
#pragma unroll
        for (int i = 0; i < HB; ++i) {
            const int it = g * HB + i;
            const uint32_t j = tid + it * THREADS;
            if (j < n) {
                const double2 xy = S::pxy()[j];
                double x = xx[i], y = yy[i], z = zz[i], px = xy.x, py = xy.y, pz = S::pz()[j];
                const double w = Q.dt / sE[j];                    // PAPER.md:34 Eq. 2 with c = 1; E = |p| as in S1
                x = x + px * w;
                y = y + py * w;
                z = z + pz * w;
                reflect_axis(x, px, P.g.L[0]);
                reflect_axis(y, py, P.g.L[1]);
                reflect_axis(z, pz, P.g.L[2]);
                const uint32_t d = T::dir()[j];
                if (d < (uint32_t)kDirs) {
                    const uint32_t row = (uint32_t)(it * W + wid) * kDirs + d;
                    const uint32_t rank = T::pref()[row] + __popc(T::ball()[row] & lanemask_lt());
                    if (rank < tab->dst_cap[d]) {
                        const uint32_t dst = tab->dst_base[d] + rank;
                        Q.out.x[dst] = x; Q.out.y[dst] = y; Q.out.z[dst] = z;
                        Q.out.px[dst] = px; Q.out.py[dst] = py; Q.out.pz[dst] = pz;
                        Q.out.pid[dst] = S::pid()[j];
                    }
                }
            }
        }
    }
}

template <int THREADS, int ITEMS, int CAP, int MIN_BLOCKS, int MODE>
__global__ void __launch_bounds__(THREADS, MIN_BLOCKS)
k_slot_step(CollideParams P, SlotParams Q)
{
    static_assert(CAP <= THREADS * ITEMS && CAP < 8192 && CAP % 32 == 0, "class capacity");
    constexpr int G = (ITEMS == 6) ? CUBA_G6 : ((ITEMS % 2 == 0) ? 2 : ITEMS);
    constexpr int LCAP = collide_list_cap(CAP);
    __shared__ uint32_t s_warp[32];
    __shared__ CtaStats s_stats;
    __shared__ SlotCell s_tab;
    const uint32_t nlist = *P.list_count;
    if (threadIdx.x == 0) s_stats.near = 0;
    ThreadStats acc{0ull, 0ull, 0u};
    __shared__ uint32_t s_item[2];
    if (threadIdx.x == 0) s_item[0] = atomicAdd(P.work, 1u);
    __syncthreads();
    uint32_t item = s_item[0];
    uint4 cur = make_uint4(0u, 0u, 0u, 0u);
    if (item < nlist) cur = P.list[item];
    for (int it = 0; item < nlist; ++it) {
        if (threadIdx.x == 0) s_item[(it + 1) & 1] = atomicAdd(P.work, 1u);
        __syncthreads();
        item = s_item[(it + 1) & 1];
        uint4 nxt = make_uint4(0u, 0u, 0u, 0u);
        if (item < nlist) nxt = P.list[item];
        step_cell_slots<THREADS, ITEMS, G, CAP, LCAP, MODE>(P, Q, cur.x, cur.y, cur.z, s_warp, &s_stats, &s_tab, acc, nxt.x, nxt.y, nxt.z);
        __syncthreads();
        cur = nxt;
    }
    if ((threadIdx.x & 31) == 0 && acc.hits) atomicAdd(&P.counters[1], (unsigned long long)acc.hits);
    if (threadIdx.x == 0) {
        if (acc.pairs) atomicAdd(&P.counters[0], acc.pairs);
        if (acc.rounds) atomicAdd(&P.counters[2], acc.rounds);
        if (s_stats.near) atomicAdd(&P.counters[3], (unsigned long long)s_stats.near);
    }
}

// ---- compact -> slotted, counts only: every cell's particles are its own segment (13); the first pass of a
// run takes them from the compact store -----------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_slot_init_counts(uint32_t ncells, const uint32_t *__restrict__ cell_start, SlotGeom sg, uint32_t *__restrict__ cnt)
{
    const uint32_t e = blockIdx.x * 256u + threadIdx.x;
    if (e >= ncells * (uint32_t)kDirs) return;
    const uint32_t c = e / (uint32_t)kDirs, s = e - c * (uint32_t)kDirs;
    cnt[e] = s == kDirStay ? cell_start[c + 1] - cell_start[c] : 0u;
}

// ---- slotted -> compact -------------------------------------------------------------------------------
// population of every cell and the per-block sums for the scan (k_scan_blocks, k_cell_start of bin.cuh)
__global__ void __launch_bounds__(256)
k_slot_count(uint32_t ncells, const uint32_t *__restrict__ cnt, uint32_t *__restrict__ count_new,
             uint32_t *__restrict__ block_sum)
{
    __shared__ uint32_t s_warp[8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const uint32_t c = blockIdx.x * 256u + threadIdx.x;
    uint32_t v = 0;
    if (c < ncells) {
#pragma unroll
        for (int s = 0; s < kDirs; ++s) v += cnt[(size_t)c * kDirs + s];
        count_new[c] = v;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    if (lane == 0) s_warp[wid] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t t = 0;
        for (int w = 0; w < 8; ++w) t += s_warp[w];
        block_sum[blockIdx.x] = t;
    }
}

}  // namespace cuba
