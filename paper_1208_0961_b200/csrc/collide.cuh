// collide.cuh -- S5: per-cell Philox-keyed shuffle, pairing, Eq. 3 decision and the fused
// boost / isotropic scatter / boost-back.
//
// One CTA per cell (persistent CTAs pull cells of their size class from a work list).
// The cell's momenta, cached energies and pids are staged in shared memory once; all R(n)
// rounds run on chip; momenta are written back once.  HBM traffic: 28 B read + 24 B written
// per particle.
//
// The shuffle is "sort by (Philox word, pid)" (A7).  Keys are uniform 32-bit
// numbers, so the sort is a one-pass bucket sort: n buckets, bucket = floor(key * n / 2^32)
// (monotone in the key), a scan of the bucket counts, then each element ranks itself inside
// its bucket (expected occupancy 1) by comparing (key, pid) -- the result depends on the
// keys only, never on the order in which threads arrived.
#pragma once
#include "common.cuh"

namespace cuba {

struct CollideParams {
    uint64_t seed;
    uint32_t t;           // global step index
    double base;          // sigma*dt/(r_test*V_cell): Eq. 3 without v_rel
    const uint32_t *cell_start;
    const uint32_t *list; // cells of this size class
    const uint32_t *list_count;
    uint32_t *work;       // dynamic work counter of this class
    double *px, *py, *pz;
    const uint32_t *pid;
    unsigned long long *counters; // [0] pairs [1] collisions [2] rounds [3] near-threshold [4] overflow cells
    uint32_t *flags;
    // overflow class only: global scratch, 4 u32 per particle of the cell
    uint32_t *arena;
    // trace (TRACE instantiation only)
    const unsigned long long *trace_off;  // per cell: first pair record
    uint32_t *tr_cell, *tr_round, *tr_pa, *tr_pb;
    double *tr_P, *tr_u;
    uint8_t *tr_dec;
};

// 53-bit uniform in [0,1)
__device__ __forceinline__ double u53(uint32_t w0, uint32_t w1)
{
    return ((double)(w0 >> 5) * 67108864.0 + (double)(w1 >> 6)) * (1.0 / 9007199254740992.0);
}

// Marsaglia disc rejection (A11): words (x,y) of call m>>1 for even attempts, (z,w) for odd.
__device__ __forceinline__ void draw_direction(uint64_t seed, uint32_t pid, uint32_t t, uint32_t rho,
                                               double &nx, double &ny, double &nz)
{
    for (uint32_t call = 0; call < 65536u; ++call) {
        const U4 w = draw(seed, pid, t, rho, kTagDir, call);
#pragma unroll
        for (int half = 0; half < 2; ++half) {
            const uint32_t wa = half ? w.z : w.x, wb = half ? w.w : w.y;
            const double a = ((double)wa + 0.5) * (1.0 / 2147483648.0) - 1.0;
            const double b = ((double)wb + 0.5) * (1.0 / 2147483648.0) - 1.0;
            const double q = a * a + b * b;
            if (q < 1.0) {
                const double h = sqrt(1.0 - q);
                nx = (2.0 * a) * h; ny = (2.0 * b) * h; nz = 1.0 - 2.0 * q;
                return;
            }
        }
    }
    nx = 0.0; ny = 0.0; nz = 1.0;
}

template <int THREADS>
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t *s_warp, uint32_t &total)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
        if (lane >= o) inc += t;
    }
    if (THREADS == 32) {
        total = __shfl_sync(0xFFFFFFFFu, inc, 31);
        return inc - v;
    }
    if (lane == 31) s_warp[wid] = inc;
    __syncthreads();
    uint32_t wpre = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) {
        const uint32_t s = s_warp[w];
        if (w < wid) wpre += s;
        tot += s;
    }
    __syncthreads();   // s_warp may be reused by the caller
    total = tot;
    return wpre + inc - v;
}

// THREADS threads work on one cell of n particles whose scratch arrays are given (shared
// memory for the size classes, global memory for the overflow class).
template <int THREADS, bool TRACE, typename IdxT>
__device__ __forceinline__ void collide_cell(const CollideParams &P, uint32_t c, uint32_t lo, uint32_t n,
                                             double *sp0, double *sp1, double *sp2, double *sE,
                                             uint32_t *spid, uint32_t *skey, uint32_t *sbkt,
                                             IdxT *sord, IdxT *stmp, uint32_t *s_warp,
                                             unsigned long long &n_pairs, unsigned long long &n_coll,
                                             unsigned long long &n_near)
{
    const int tid = threadIdx.x;
    // rounds and scale (A5, A6): identical integer/fp64 results on every thread
    const double cn = (n & 1u) ? (double)n : (double)(n - 1u);
    const double pmax = (2.0 * cn) * P.base;
    int R;
    if (!(pmax <= 64.0)) { if (tid == 0) atomicOr(P.flags, kFlagRounds); R = 64; }
    else R = (pmax <= 1.0) ? 1 : (int)ceil(pmax);
    const double scale = (cn * P.base) / (double)R;
    const uint32_t npairs = n >> 1;

    for (uint32_t j = tid; j < n; j += THREADS) {
        const double a = P.px[lo + j], b = P.py[lo + j], cc = P.pz[lo + j];
        sp0[j] = a; sp1[j] = b; sp2[j] = cc;
        sE[j] = energy(a, b, cc);
        spid[j] = P.pid[lo + j];
    }
    for (uint32_t j = tid; j <= n; j += THREADS) sbkt[j] = 0;
    __syncthreads();

    for (int rho = 0; rho < R; ++rho) {
        // (a) keys and bucket counts; the arrival slot only serves to park the element
        for (uint32_t j = tid; j < n; j += THREADS) {
            const uint32_t k = draw(P.seed, spid[j], P.t, (uint32_t)rho, kTagShuf, 0).x;
            skey[j] = k;
            sord[j] = (IdxT)atomicAdd(&sbkt[__umulhi(k, n)], 1u);
        }
        __syncthreads();
        // (b) exclusive scan of the n bucket counts, contiguous chunk per thread
        {
            const uint32_t chunk = (n + THREADS - 1) / THREADS;
            const uint32_t b0 = min(n, tid * chunk), b1 = min(n, b0 + chunk);
            uint32_t s = 0;
            for (uint32_t b = b0; b < b1; ++b) s += sbkt[b];
            uint32_t total;
            uint32_t run = block_exclusive_scan<THREADS>(s, s_warp, total);
            for (uint32_t b = b0; b < b1; ++b) { const uint32_t v = sbkt[b]; sbkt[b] = run; run += v; }
            if (tid == 0) sbkt[n] = n;
        }
        __syncthreads();
        // (c) park element j at its arrival slot inside its bucket
        for (uint32_t j = tid; j < n; j += THREADS)
            stmp[sbkt[__umulhi(skey[j], n)] + (uint32_t)sord[j]] = (IdxT)j;
        __syncthreads();
        // (d) final rank = bucket start + number of bucket mates with a smaller (key, pid)
        for (uint32_t j = tid; j < n; j += THREADS) {
            const uint32_t k = skey[j], id = spid[j];
            const uint32_t b = __umulhi(k, n);
            const uint32_t beg = sbkt[b], end = sbkt[b + 1];
            uint32_t rank = beg;
            for (uint32_t q = beg; q < end; ++q) {
                const uint32_t jj = (uint32_t)stmp[q];
                const uint32_t k2 = skey[jj];
                rank += (k2 < k || (k2 == k && spid[jj] < id)) ? 1u : 0u;
            }
            sord[rank] = (IdxT)j;   // slots in sord are dead after (c)
        }
        __syncthreads();
        // (e) pair order[2k] with order[2k+1]; Eq. 3; scatter.  Each particle is in one pair.
        for (uint32_t k = tid; k < npairs; k += THREADS) {
            const uint32_t a = (uint32_t)sord[2 * k], b = (uint32_t)sord[2 * k + 1];
            const double pax = sp0[a], pay = sp1[a], paz = sp2[a], Ea = sE[a];
            const double pbx = sp0[b], pby = sp1[b], pbz = sp2[b], Eb = sE[b];
            const double ee = Ea * Eb;
            const double dx = Eb * pax - Ea * pbx;
            const double dy = Eb * pay - Ea * pby;
            const double dz = Eb * paz - Ea * pbz;
            const double s = ((dx * dx + dy * dy) + dz * dz) / ee;   // (p_a+p_b)^2, A9
            const double vrel = 0.5 * (s / ee);                       // s/(2 E_a E_b)
            const double prob = vrel * scale;                         // Eq. 3 * cn/R
            const uint32_t ida = spid[a];
            const U4 w = draw(P.seed, ida, P.t, (uint32_t)rho, kTagDec, 0);
            const double u = u53(w.x, w.y);
            const bool hit = u < prob;
            n_pairs += 1;
            if (fabs(u - prob) <= 1e-12) n_near += 1;
            if (TRACE) {
                const unsigned long long e = P.trace_off[c] + (unsigned long long)rho * npairs + k;
                P.tr_cell[e] = c; P.tr_round[e] = (uint32_t)rho; P.tr_pa[e] = ida; P.tr_pb[e] = spid[b];
                P.tr_P[e] = prob; P.tr_u[e] = u; P.tr_dec[e] = hit ? 1 : 0;
            }
            if (hit) {
                double nx, ny, nz;
                draw_direction(P.seed, ida, P.t, (uint32_t)rho, nx, ny, nz);
                const double rs = sqrt(s);
                const double Pvx = pax + pbx, Pvy = pay + pby, Pvz = paz + pbz;
                const double Et = Ea + Eb;
                const double Pn = (Pvx * nx + Pvy * ny) + Pvz * nz;
                const double al = Pn / (Et + rs);
                const double f1 = 1.0 + al, f2 = 1.0 - al;
                const double qax = 0.5 * (rs * nx + Pvx * f1);
                const double qay = 0.5 * (rs * ny + Pvy * f1);
                const double qaz = 0.5 * (rs * nz + Pvz * f1);
                const double qbx = 0.5 * (Pvx * f2 - rs * nx);
                const double qby = 0.5 * (Pvy * f2 - rs * ny);
                const double qbz = 0.5 * (Pvz * f2 - rs * nz);
                sp0[a] = qax; sp1[a] = qay; sp2[a] = qaz; sE[a] = energy(qax, qay, qaz);
                sp0[b] = qbx; sp1[b] = qby; sp2[b] = qbz; sE[b] = energy(qbx, qby, qbz);
                n_coll += 1;
            }
        }
        for (uint32_t j = tid; j <= n; j += THREADS) sbkt[j] = 0;
        __syncthreads();
    }
    for (uint32_t j = tid; j < n; j += THREADS) {
        P.px[lo + j] = sp0[j]; P.py[lo + j] = sp1[j]; P.pz[lo + j] = sp2[j];
    }
    if (tid == 0) atomicAdd(&P.counters[2], (unsigned long long)R);
}

template <int THREADS>
__device__ __forceinline__ void flush_counters(const CollideParams &P, unsigned long long n_pairs,
                                               unsigned long long n_coll, unsigned long long n_near)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        n_pairs += __shfl_xor_sync(0xFFFFFFFFu, n_pairs, o);
        n_coll += __shfl_xor_sync(0xFFFFFFFFu, n_coll, o);
        n_near += __shfl_xor_sync(0xFFFFFFFFu, n_near, o);
    }
    if ((threadIdx.x & 31) == 0) {
        if (n_pairs) atomicAdd(&P.counters[0], n_pairs);
        if (n_coll) atomicAdd(&P.counters[1], n_coll);
        if (n_near) atomicAdd(&P.counters[3], n_near);
    }
}

// Shared-memory classes: CAP particles at most, 48 B of shared memory per particle.
template <int THREADS, int CAP, int MIN_BLOCKS, bool TRACE>
__global__ void __launch_bounds__(THREADS, MIN_BLOCKS)
k_collide(CollideParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *sp0 = reinterpret_cast<double *>(smem_raw);
    double *sp1 = sp0 + CAP, *sp2 = sp1 + CAP, *sE = sp2 + CAP;
    uint32_t *spid = reinterpret_cast<uint32_t *>(sE + CAP);
    uint32_t *skey = spid + CAP;
    uint32_t *sbkt = skey + CAP;                 // CAP + 2 entries
    uint16_t *sord = reinterpret_cast<uint16_t *>(sbkt + CAP + 2);
    uint16_t *stmp = sord + CAP;
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_item;

    const uint32_t nlist = *P.list_count;
    unsigned long long n_pairs = 0, n_coll = 0, n_near = 0;
    for (;;) {
        if (threadIdx.x == 0) s_item = atomicAdd(P.work, 1u);
        __syncthreads();
        const uint32_t item = s_item;
        if (item >= nlist) break;
        const uint32_t c = P.list[item];
        const uint32_t lo = P.cell_start[c], n = P.cell_start[c + 1] - lo;
        collide_cell<THREADS, TRACE, uint16_t>(P, c, lo, n, sp0, sp1, sp2, sE, spid, skey, sbkt, sord,
                                               stmp, s_warp, n_pairs, n_coll, n_near);
        __syncthreads();
    }
    flush_counters<THREADS>(P, n_pairs, n_coll, n_near);
}

constexpr size_t collide_smem_bytes(int cap) { return (size_t)cap * 48 + 16; }

// Overflow class: cells larger than the biggest shared-memory class.  Same routine, scratch
// in global memory (momenta are updated in place in the particle store; the cached energy
// and the four u32 work arrays live in the arena, bump-allocated per cell).
template <bool TRACE>
__global__ void __launch_bounds__(1024)
k_collide_overflow(CollideParams P, unsigned long long *arena_cursor, double *arena_E)
{
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_item;
    __shared__ unsigned long long s_base;
    const uint32_t nlist = *P.list_count;
    unsigned long long n_pairs = 0, n_coll = 0, n_near = 0;
    for (;;) {
        if (threadIdx.x == 0) s_item = atomicAdd(P.work, 1u);
        __syncthreads();
        const uint32_t item = s_item;
        if (item >= nlist) break;
        const uint32_t c = P.list[item];
        const uint32_t lo = P.cell_start[c], n = P.cell_start[c + 1] - lo;
        if (threadIdx.x == 0) {
            s_base = atomicAdd(arena_cursor, (unsigned long long)n + 2ull);
            atomicAdd(&P.counters[4], 1ull);
        }
        __syncthreads();
        const unsigned long long b = s_base;
        uint32_t *a32 = P.arena + 4ull * b;
        uint32_t *skey = a32, *sbkt = a32 + (n + 2), *sord = a32 + 2ull * (n + 2), *stmp = a32 + 3ull * (n + 2);
        // momenta in place: the "staging" copy is the particle store itself
        collide_cell<1024, TRACE, uint32_t>(P, c, lo, n, P.px + lo, P.py + lo, P.pz + lo, arena_E + b,
                                            const_cast<uint32_t *>(P.pid) + lo, skey, sbkt, sord, stmp,
                                            s_warp, n_pairs, n_coll, n_near);
        __syncthreads();
    }
    flush_counters<1024>(P, n_pairs, n_coll, n_near);
}

}  // namespace cuba
