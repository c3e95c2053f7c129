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
    int i0[3];                       // cell coordinates (x slowest)
};

// The tables of cell c, by one warp.  v: lane s < 27 holds the population of inbox segment s of the cell
// (loaded by the caller, possibly long before: the tables of a CTA's NEXT cell are built while the
// current one is processed, so that nobody waits for that load).
template <bool FROM_SLOTS, bool STREAM>
__device__ __forceinline__ void slot_tables(const Geom &g, const SlotGeom &sg, uint32_t c, uint32_t v, SlotCell *tab)
{
    const int lane = threadIdx.x & 31;
    const int i2 = (int)(c % (uint32_t)g.nc[2]);
    const int i1 = (int)((c / (uint32_t)g.nc[2]) % (uint32_t)g.nc[1]);
    const int i0 = (int)(c / ((uint32_t)g.nc[2] * (uint32_t)g.nc[1]));
    if (lane == 0) { tab->i0[0] = i0; tab->i0[1] = i1; tab->i0[2] = i2; }
    if (FROM_SLOTS) {
        uint32_t inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane <= kDirs) tab->seg_start[lane] = inc - v;       // lane 27: the total
        if (lane < kDirs) tab->src_base[lane] = c * sg.slots + sg.seg_off[lane];
    }
    if (STREAM && lane < kDirs) {
        const int nb = slot_neighbour(g, i0, i1, i2, lane);
        const int seg = kDirs - 1 - lane;
        tab->dst_base[lane] = nb >= 0 ? (uint32_t)nb * sg.slots + sg.seg_off[seg] : 0u;
        tab->dst_cap[lane] = nb >= 0 ? sg.seg_off[seg + 1] - sg.seg_off[seg] : 0u;
        tab->dst_cnt[lane] = nb >= 0 ? (uint32_t)nb * kDirs + (uint32_t)seg : 0xFFFFFFFFu;
    }
}

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
// row masks [rows][27], the lists' space their prefixes (16 bit).
template <int CAP, int LCAP>
struct SlotTail {
    using S = CellSmem<CAP, LCAP>;
    static __device__ __forceinline__ uint32_t *ball() { return S::cnt(); }                                      // [rows][27] <= CAP words
    static __device__ __forceinline__ uint16_t *pref() { return reinterpret_cast<uint16_t *>(S::lkey(0)); }      // [rows][27] 16 bit <= 12 LCAP bytes... checked below
};

// What a pass does.  A call of n steps is n + 1 passes: the first one takes the cells from the compact store and
// only streams (the compact state is the state after the collisions of the previous step); the middle ones
// collide and stream; the last one collides and writes the compact store (its cell_start is known beforehand:
// collisions move nobody).
enum SlotMode { kSlotMiddle = 0, kSlotFirst = 1, kSlotLast = 2 };

template <int THREADS, int ITEMS, int G, int CAP, int LCAP, int MODE>
__device__ __forceinline__ void step_cell_slots(const CollideParams &P, const SlotParams &Q, uint32_t c, uint32_t lo, uint32_t n,
                                                uint32_t *s_warp, CtaStats *stats, SlotCell *tab, SlotCell *tab_next, bool tab_ready,
                                                uint32_t *s_vnext, uint32_t c_next, uint32_t lo_next, uint32_t n_next)
{
    using S = CellSmem<CAP, LCAP>;
    using T = SlotTail<CAP, LCAP>;
    constexpr int W = THREADS / 32, ROWS = ITEMS * W;
    static_assert(ROWS * kDirs <= CAP, "row masks fit the duplicate counters' space");
    static_assert(ROWS * kDirs * 2 <= 24 * LCAP, "row prefixes fit the lists' space");
    static_assert(ITEMS <= 6, "direction codes of a thread's items are packed 5 bits each");
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
    // ---- per-cell tables (warp 0): this cell's only for the first cell of a CTA; the inbox counts of the NEXT
    // cell are fetched now and turned into its tables after the rounds, so that nobody waits for the load --
    // (an asynchronous copy into shared memory: no register is held across the rounds)
    if (tid < 32) {
        if (!tab_ready) {
            const uint32_t v = (FROM_SLOTS && lane < kDirs) ? Q.in.cnt[(size_t)c * kDirs + lane] : 0u;
            slot_tables<FROM_SLOTS, STREAM>(P.g, Q.sg, c, v, tab);
        }
        if (FROM_SLOTS && n_next && lane < kDirs)
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(s_vnext + lane)), "l"(Q.in.cnt + (size_t)c_next * kDirs + lane) : "memory");
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    __syncthreads();
    const uint32_t last = n - 1u;
    double *sE = S::E();
    // items it of this warp with a particle in them: (tid & ~31) + it * THREADS < n
    const int nit = (int)min((uint32_t)ITEMS, (n + (uint32_t)THREADS - 1u - min(n, (uint32_t)(tid & ~31))) / (uint32_t)THREADS);
    // ---- assemble: momenta and pids (from the 27 segments in order); clear the sort structures ---------
#pragma unroll
    for (int g = 0; g < ITEMS / G; ++g) {
        if (g * G >= nit) break;       // warp-uniform; inside a group the padding is loaded (clamped) and dropped
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
#ifdef CUBA_PHASE_CLOCKS
        long long g_last = 0;
        run_sweeps<THREADS, ITEMS, G, CAP, LCAP, false>(P, c, n, R, tcur, STREAM, s_warp, stats, g_last);
#else
        run_sweeps<THREADS, ITEMS, G, CAP, LCAP, false>(P, c, n, R, tcur, STREAM, s_warp, stats);
#endif
        if (STREAM && R == 0 && tid == 0) {     // a lone particle: no pair phase has computed its energy
            const double2 xy = S::pxy()[0];
            sE[0] = energy(xy.x, xy.y, S::pz()[0]);
        }
        if (tid == 0) { stats->pairs += (unsigned long long)R * (n >> 1); stats->rounds += (unsigned long long)R; }
    }
    if (tid < 32 && n_next) {
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncwarp();
        slot_tables<FROM_SLOTS, STREAM>(P.g, Q.sg, c_next, (FROM_SLOTS && lane < kDirs) ? s_vnext[lane] : 0u, tab_next);
    }
    if (!STREAM) {
        __syncthreads();
        // ---- last pass: the cell goes to its place in the compact store, positions unchanged -----------
        constexpr int HB = (ITEMS % 2 == 0) ? 2 : 1;
#pragma unroll 1
        for (int g = 0; g < ITEMS / HB; ++g) {
            if (g * HB >= nit) break;
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

    // ---- tail, pass 1: S1-S3 exactly (the arithmetic of move_particle); one mask per row of 32 particles and
    // direction.  The positions of the next item are in flight while an item is moved; the new x goes into the
    // particle's (now dead) energy slot, the new y and z stay in registers across the prefix. ----
    double Y[ITEMS], Z[ITEMS];
    double xa = 0.0, ya = 0.0, za = 0.0;
    if (nit > 0) {
        const uint32_t jc = min((uint32_t)tid, last);
        const uint32_t src = FROM_SLOTS ? slot_source(tab, jc) : lo + jc;
        xa = Q.in.x[src]; ya = Q.in.y[src]; za = Q.in.z[src];
    }
    for (int e = tid; e < ROWS * kDirs; e += THREADS) T::ball()[e] = 0;    // the dirty lists were last read before the last pair phase
    __syncthreads();     // the rounds are over (energies final), the masks are clear
    const int ix0 = tab->i0[0], iy0 = tab->i0[1], iz0 = tab->i0[2];
    uint32_t dpk = 0;
#pragma unroll
    for (int it = 0; it < ITEMS; ++it) {
        if (it < nit) {
            double xn = 0.0, yn = 0.0, zn = 0.0;
            if (it + 1 < nit) {
                const uint32_t jc = min((uint32_t)(tid + (it + 1) * THREADS), last);
                const uint32_t src = FROM_SLOTS ? slot_source(tab, jc) : lo + jc;
                xn = Q.in.x[src]; yn = Q.in.y[src]; zn = Q.in.z[src];
            }
            const uint32_t j = tid + it * THREADS, jj = min(j, last);
            const double2 xy = S::pxy()[jj];
            const double pz0 = S::pz()[jj];
            double px = xy.x, py = xy.y, pz = pz0;
            const double w = Q.dt / sE[jj];                   // PAPER.md:34 Eq. 2 with c = 1; E = |p| as in S1
            double x = xa + px * w;
            double y = ya + py * w;
            double z = za + pz * w;
            reflect_axis(x, px, P.g.L[0]);
            reflect_axis(y, py, P.g.L[1]);
            reflect_axis(z, pz, P.g.L[2]);
            const int dx = axis_index(x, P.g.inv_d[0], P.g.nc[0]) - ix0 + 1;
            const int dy = axis_index(y, P.g.inv_d[1], P.g.nc[1]) - iy0 + 1;
            const int dz = axis_index(z, P.g.inv_d[2], P.g.nc[2]) - iz0 + 1;
            int d = ((unsigned)dx <= 2u && (unsigned)dy <= 2u && (unsigned)dz <= 2u) ? (dx * 9 + dy * 3 + dz) : -1;
            if (j >= n) d = 31;                                   // not a particle
            else if (d < 0) { atomicOr(P.flags, kFlagMoved); d = 30; }   // dropped from the placement, as in k_scatter
            const uint32_t peers = __match_any_sync(0xFFFFFFFFu, d);
            if (d < kDirs && (peers & lanemask_lt()) == 0) T::ball()[(it * W + wid) * kDirs + d] = peers;
            if (j < n) {
                sE[j] = x;                                        // only this thread reads the slot again
                if (px != xy.x || py != xy.y || pz != pz0) {      // reflected off a wall: rare
                    S::pxy()[j] = make_double2(px, py); S::pz()[j] = pz;
                }
            }
            Y[it] = y; Z[it] = z;
            dpk |= (uint32_t)d << (5 * it);
            xa = xn; ya = yn; za = zn;
        }
    }
    __syncthreads();
    // ---- exclusive prefix of the row masks per direction: 27 directions x 8 chunks of rows, 8 adjacent lanes each ----
    {
        constexpr int RCH = (ROWS + 7) / 8;
#pragma unroll 1
        for (int e0 = 0; e0 < kDirs * 8; e0 += THREADS) {
            const int e = e0 + tid;
            const bool valid = e < kDirs * 8;
            const int d = min(e >> 3, kDirs - 1), q = e & 7;
            uint32_t v[RCH], sum = 0;
#pragma unroll
            for (int r = 0; r < RCH; ++r) {
                const int row = q * RCH + r;
                v[r] = row < ROWS ? (uint32_t)__popc(T::ball()[row * kDirs + d]) : 0u;
                sum += v[r];
            }
            uint32_t inc = sum;
#pragma unroll
            for (int o = 1; o < 8; o <<= 1) {
                const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o, 8);
                if (q >= o) inc += t;
            }
            uint32_t run = inc - sum;
            if (valid) {
#pragma unroll
                for (int r = 0; r < RCH; ++r) {
                    const int row = q * RCH + r;
                    if (row < ROWS) T::pref()[row * kDirs + d] = (uint16_t)run;
                    run += v[r];
                }
                if (q == 7) {                 // inc: all particles of the cell that leave in direction d
                    const uint32_t cap = tab->dst_cap[d], at = tab->dst_cnt[d];
                    if (at != 0xFFFFFFFFu) Q.out.cnt[at] = min(inc, cap);
                    if (inc > cap) atomicOr(P.flags, kFlagSlots);          // capacity: the host redoes the run on the compact path
                }
            }
        }
    }
    __syncthreads();
    // ---- tail, pass 2: stable rank, write into the destination's inbox ------------------------------------
#pragma unroll
    for (int it = 0; it < ITEMS; ++it) {
        if (it < nit) {
            const uint32_t j = tid + it * THREADS;
            const uint32_t d = (dpk >> (5 * it)) & 31u;
            if (j < n && d < (uint32_t)kDirs) {
                const uint32_t row = (uint32_t)(it * W + wid) * kDirs + d;
                const uint32_t rank = T::pref()[row] + __popc(T::ball()[row] & lanemask_lt());
                if (rank < tab->dst_cap[d]) {
                    const uint32_t dst = tab->dst_base[d] + rank;
                    const double2 xy = S::pxy()[j];
                    Q.out.x[dst] = sE[j]; Q.out.y[dst] = Y[it]; Q.out.z[dst] = Z[it];
                    Q.out.px[dst] = xy.x; Q.out.py[dst] = xy.y; Q.out.pz[dst] = S::pz()[j];
                    Q.out.pid[dst] = S::pid()[j];
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
    __shared__ SlotCell s_tab[2];
    const uint32_t nlist = *P.list_count;
    __shared__ uint32_t s_vnext[32];
    if (threadIdx.x == 0) { s_stats.near = 0; s_stats.hits = 0; s_stats.pairs = 0; s_stats.rounds = 0; }
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
        step_cell_slots<THREADS, ITEMS, G, CAP, LCAP, MODE>(P, Q, cur.x, cur.y, cur.z, s_warp, &s_stats, &s_tab[it & 1], &s_tab[(it + 1) & 1], it > 0,
                                                            s_vnext, nxt.x, nxt.y, nxt.z);
        __syncthreads();
        cur = nxt;
    }
    if (threadIdx.x == 0) {       // the loop ends with a block barrier
        if (s_stats.hits) atomicAdd(&P.counters[1], (unsigned long long)s_stats.hits);
        if (s_stats.pairs) atomicAdd(&P.counters[0], s_stats.pairs);
        if (s_stats.rounds) atomicAdd(&P.counters[2], s_stats.rounds);
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
