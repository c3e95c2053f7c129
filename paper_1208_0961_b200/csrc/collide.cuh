// collide.cuh -- S5: per-cell Philox-keyed shuffle, pairing, Eq. 3 decision and the fused
// boost / isotropic scatter / boost-back.
//
// One CTA per cell (persistent CTAs pull cells of their size class from a work list).
// The cell's momenta, cached energies and pids are staged in shared memory once; all R(n)
// rounds run on chip; momenta are written back once.  HBM traffic: 28 B read + 24 B written
// per particle, + 24 B read (x, y, z) when the kernel also prepares the counting-sort
// histogram of the next step ("fused histogram" below).  Template switches: TRACE (parity
// records per pair) and LOCAL (per-cell cross section for constant eta/s, A24).
//
// The shuffle is "sort by (Philox word, pid)" (A7).  Keys are uniform 32-bit
// numbers, so the sort is a one-pass bucket sort: n buckets, bucket = floor(key * n / 2^32)
// (monotone in the key), a scan of the bucket counts, then each element ranks itself inside
// its bucket (expected occupancy 1) by comparing (key, pid) -- the result depends on the
// keys only, never on the order in which threads arrived.
#pragma once
#include "common.cuh"

namespace cuba {

#ifndef CUBA_FORCE_SLOW_PATHS   // test builds set this to 1: every element / pair takes the rare paths
#define CUBA_FORCE_SLOW_PATHS 0
#endif

// Phase clocks (diagnostic builds only, -DCUBA_PHASE_CLOCKS): thread 0 of every CTA of the 256-thread class adds
// the cycles between consecutive marks to a per-phase total; mark k closes phase k (its barrier wait included).
#ifdef CUBA_PHASE_CLOCKS
__device__ unsigned long long g_phase[16];
__device__ __forceinline__ void phase_mark(long long &last, int k)
{
    if (threadIdx.x == 0 && blockDim.x == 256) {
        const long long t = clock64();
        atomicAdd(&g_phase[k], (unsigned long long)(t - last));
        last = t;
    }
}
#define CUBA_MARK(k) phase_mark(g_last, k)
#else
#define CUBA_MARK(k)
#endif

struct CollideParams {
    uint64_t seed;
    uint32_t rk[20];      // Philox round keys: rk[2r] = seed_lo + r*0x9E3779B9, rk[2r+1] = seed_hi + r*0xBB67AE85
    uint32_t t;           // global step index
    const uint32_t *t_dev; // GRAPH instantiations: the step index lives in device memory (a replayed graph cannot carry it)
    double base;          // sigma*dt/(r_test*V_cell): Eq. 3 without v_rel
    const uint32_t *cell_start;
    const uint4 *list;    // cells of this size class: {cell, first slot, population, -}
    const uint32_t *list_count;
    uint32_t *work;       // dynamic work counter of this class (overflow kernel)
    double *px, *py, *pz;
    const uint32_t *pid;
    unsigned long long *counters; // [0] pairs [1] collisions [2] rounds [3] near-threshold [4] overflow cells
    uint32_t *flags;
    // overflow class only: global scratch, 4 u32 per particle of the cell
    uint32_t *arena;
    // local cross section for constant eta/s (etas > 0, A24): Eq. 3 without
    // v_rel is computed per cell from the cell's population and energy sum instead of `base`
    double etas, dt;
    // fused histogram of the NEXT step (next_dt > 0): the cell's CTA holds the final momenta on
    // chip, and the old cell of every particle is the cell itself, so S1-S3 of step t+1 are done
    // here and the (cell, direction) counts and the per-tile carries are written directly --
    // the separate k_stream_hist / k_carry pass (48 B per particle) disappears.
    double next_dt;
    Geom g;
    const double *x, *y, *z;
    uint32_t *cnt;        // [27][ncells], cleared beforehand (empty cells stay zero)
    uint32_t *carry;      // [ntiles][kTileRec]
    // trace (TRACE instantiation only)
    const unsigned long long *trace_off;  // per cell: first pair record
    uint32_t *tr_cell, *tr_round, *tr_pa, *tr_pb;
    double *tr_P, *tr_u;
    uint8_t *tr_dec;
};

// Local cross section (A24): base_cell = ((0.1 S) dt) / ((hbarc (n n)) etas) with S the cell's
// energy sum, DEFINED as the exact fixed-point sum (sum_i rint(E_i 2^40)) 2^-40 so that it does not
// depend on the order in which threads add it up.
constexpr double kHbarC = 0.197327;          // GeV fm (BASELINE.json:configs[0])
constexpr double kFix40 = 1099511627776.0;   // 2^40

__device__ __forceinline__ long long energy_fixed(double E) { return __double2ll_rn(E * kFix40); }

__device__ __forceinline__ double local_base(long long acc, uint32_t n, double dt, double etas)
{
    const double S = (double)acc * (1.0 / kFix40);
    const double nn = (double)n * (double)n;
    return ((0.1 * S) * dt) / ((kHbarC * nn) * etas);
}

// Sum of one 64-bit integer per thread over the CTA (integer addition: any order gives the same
// bits).  Call before a barrier, read with block_sum_ll_read after it.
template <int THREADS>
__device__ __forceinline__ void block_sum_ll_post(long long v, long long *s_slots)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    if ((threadIdx.x & 31) == 0) s_slots[threadIdx.x >> 5] = v;
}

template <int THREADS>
__device__ __forceinline__ long long block_sum_ll_read(const long long *s_slots)
{
    long long t = 0;
#pragma unroll
    for (int w = 0; w < THREADS / 32; ++w) t += s_slots[w];
    return t;
}

// 53-bit uniform in [0,1)
__device__ __forceinline__ double u53(uint32_t w0, uint32_t w1)
{
    return ((double)(w0 >> 5) * 67108864.0 + (double)(w1 >> 6)) * (1.0 / 9007199254740992.0);
}

// draw() with the key schedule taken from the kernel parameters (constant bank operands):
// the same function of (seed, id, t, rho, tag, sub), without 18 key additions per call.
__device__ __forceinline__ U4 drawk(const CollideParams &P, uint32_t t, uint32_t id, uint32_t rho, uint32_t tag, uint32_t sub)
{
    uint32_t c0 = id, c1 = t, c2 = rho, c3 = (tag << 16) | sub;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ P.rk[2 * r], n2 = hi0 ^ c3 ^ P.rk[2 * r + 1];
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    return U4{c0, c1, c2, c3};
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

// Shuffle key of round rho (A7): word rho mod 4 of the call for rounds 4*floor(rho/4)..+3.
__device__ __forceinline__ uint32_t shuf_word(const U4 &w, int rho)
{
    const int q = rho & 3;
    return q == 0 ? w.x : (q == 1 ? w.y : (q == 2 ? w.z : w.w));
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

// Generic routine (overflow class): THREADS threads work on one cell of n particles of any
// size, scratch arrays in global memory, n buckets of 32-bit counters, run-time loops.
template <int THREADS, bool TRACE, typename IdxT>
__device__ __forceinline__ void collide_cell(const CollideParams &P, uint32_t c, uint32_t lo, uint32_t n,
                                             double *sp0, double *sp1, double *sp2, double *sE,
                                             uint32_t *spid, uint32_t *skey, uint32_t *sbkt,
                                             IdxT *sord, IdxT *stmp, uint32_t *s_warp, long long *s_esum,
                                             unsigned long long &n_pairs, unsigned long long &n_coll,
                                             unsigned long long &n_near)
{
    const int tid = threadIdx.x;
    const uint32_t npairs = n >> 1;
    const uint32_t tcur = P.t_dev ? *P.t_dev : P.t;
    long long esum = 0;
    for (uint32_t j = tid; j < n; j += THREADS) {
        const double a = P.px[lo + j], b = P.py[lo + j], cc = P.pz[lo + j];
        sp0[j] = a; sp1[j] = b; sp2[j] = cc;
        const double e = energy(a, b, cc);
        sE[j] = e;
        esum += energy_fixed(e);
        spid[j] = P.pid[lo + j];
    }
    for (uint32_t j = tid; j <= n; j += THREADS) sbkt[j] = 0;
    block_sum_ll_post<THREADS>(esum, s_esum);
    __syncthreads();
    // rounds and scale (A5, A6): identical integer/fp64 results on every thread
    const double base = (P.etas > 0.0) ? local_base(block_sum_ll_read<THREADS>(s_esum), n, P.dt, P.etas) : P.base;
    const double cn = (n & 1u) ? (double)n : (double)(n - 1u);
    const double pmax = (2.0 * cn) * base;
    int R;
    if (!(pmax <= 64.0)) { if (tid == 0) atomicOr(P.flags, kFlagRounds); R = 64; }
    else R = (pmax <= 1.0) ? 1 : (int)ceil(pmax);
    if (n < 2u) R = 0;
    const double scale = (cn * base) / (double)R;

    for (int rho = 0; rho < R; ++rho) {
        // (a) keys and bucket counts; the arrival slot only serves to park the element
        for (uint32_t j = tid; j < n; j += THREADS) {
            const uint32_t k = shuf_word(draw(P.seed, spid[j], tcur, (uint32_t)rho >> 2, kTagShuf, 0), rho);
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
            const U4 w = draw(P.seed, ida, tcur, (uint32_t)rho, kTagDec, 0);
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
                draw_direction(P.seed, ida, tcur, (uint32_t)rho, nx, ny, nz);
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

__device__ __forceinline__ void prefetch_l2(const void *p)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// ---- fused histogram of the next step ---------------------------------------------------
// Direction code of a particle of cell (ix0,iy0,iz0) after S1-S3 with time step dt: the same
// arithmetic as move_particle() in bin.cuh (k_stream_hist / k_scatter), so the counts written
// here equal those k_stream_hist would produce from the written-back store.
__device__ __forceinline__ int next_direction(const Geom &g, double dt, int ix0, int iy0, int iz0,
                                              double x, double y, double z, double px, double py, double pz, double E)
{
    const double w = dt / E;                         // PAPER.md:34 Eq. 2 with c = 1
    x = x + px * w;
    y = y + py * w;
    z = z + pz * w;
    reflect_axis(x, px, g.L[0]);
    reflect_axis(y, py, g.L[1]);
    reflect_axis(z, pz, g.L[2]);
    const int dx = axis_index(x, g.inv_d[0], g.nc[0]) - ix0 + 1;
    const int dy = axis_index(y, g.inv_d[1], g.nc[1]) - iy0 + 1;
    const int dz = axis_index(z, g.inv_d[2], g.nc[2]) - iz0 + 1;
    return ((unsigned)dx <= 2u && (unsigned)dy <= 2u && (unsigned)dz <= 2u) ? (dx * 9 + dy * 3 + dz) : -1;
}

// Per-cell constants of the fused histogram, written when the cell is set up.
struct HistCell {
    int i0[3];            // cell coordinates (x slowest)
    double i0d[3];        // the same as doubles
    uint32_t map[kDirs];  // raw direction code (floor of the estimated position, per axis 0/1/2) -> direction code:
                          // a component that leaves through a wall face becomes 1 (elastic reflection back
                          // into the cell, A12; dt < cell edge keeps the mirror image inside it)
};

__device__ __forceinline__ void hist_cell_setup(const Geom &g, uint32_t c, HistCell *h, int tid)
{
    const int i2 = (int)(c % (uint32_t)g.nc[2]);
    const int i1 = (int)((c / (uint32_t)g.nc[2]) % (uint32_t)g.nc[1]);
    const int i0 = (int)(c / ((uint32_t)g.nc[2] * (uint32_t)g.nc[1]));
    if (tid == 0) {
        h->i0[0] = i0; h->i0[1] = i1; h->i0[2] = i2;
        h->i0d[0] = (double)i0; h->i0d[1] = (double)i1; h->i0d[2] = (double)i2;
    }
    if (tid < kDirs) {
        int dx = tid / 9, dy = (tid / 3) % 3, dz = tid % 3;
        if ((dx == 0 && i0 == 0) || (dx == 2 && i0 == g.nc[0] - 1)) dx = 1;
        if ((dy == 0 && i1 == 0) || (dy == 2 && i1 == g.nc[1] - 1)) dy = 1;
        if ((dz == 0 && i2 == 0) || (dz == 2 && i2 == g.nc[2] - 1)) dz = 1;
        h->map[tid] = (uint32_t)(dx * 9 + dy * 3 + dz);
    }
}

__device__ __forceinline__ double rcp_approx(double a)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));   // ~20 good bits from the upper word
    return r;
}

// Guarded estimate of the direction code.  t = position after the move in units of the cell edge,
// relative to the cell's lower face (the cell is [0,1); dt < cell edge means -1 < t < 2), computed
// without the fp64 division (hardware reciprocal + one Newton step, explicit FMAs: good to ~1e-9).
// Adding 1.5*2^32 leaves round(t*2^20) in the low word of the sum (two's complement) and a fixed high
// word: the integer part of (t+1) is the raw component 0/1/2 and the 20 fraction bits say how close
// the particle is to a face.  Within kHistBand/2^20 = 1.2e-4 cell edges of a face -- or for anything
// unexpected (NaN, a high word that is not the constant's) -- the caller redoes the particle with the
// exact operation order of S1-S3; the scatter always uses the exact arithmetic.
constexpr double kHistMagic = 6442450944.0;        // 1.5 * 2^32
constexpr int kHistMagicHi = 0x41F80000;           // its high word; 0x41F7FFFF just below
constexpr uint32_t kHistOne = 1u << 20;
constexpr uint32_t kHistBand = 128u;

__device__ __forceinline__ int next_direction_guarded(const Geom &g, double dt, const HistCell &h,
                                                      double x, double y, double z, double px, double py, double pz, double E)
{
    double r = rcp_approx(E);
    r = __fma_rn(r, __fma_rn(-E, r, 1.0), r);
    const double w = dt * r;
    const double yx = __dadd_rn(__fma_rn(__fma_rn(px, w, x), g.inv_d[0], -h.i0d[0]), kHistMagic);
    const double yy = __dadd_rn(__fma_rn(__fma_rn(py, w, y), g.inv_d[1], -h.i0d[1]), kHistMagic);
    const double yz = __dadd_rn(__fma_rn(__fma_rn(pz, w, z), g.inv_d[2], -h.i0d[2]), kHistMagic);
    const uint32_t ux = (uint32_t)__double2loint(yx) + kHistOne;     // (t + 1) * 2^20 for -1 <= t < 2
    const uint32_t uy = (uint32_t)__double2loint(yy) + kHistOne;
    const uint32_t uz = (uint32_t)__double2loint(yz) + kHistOne;
    const uint32_t hi = ((uint32_t)__double2hiint(yx) - (uint32_t)(kHistMagicHi - 1)) |
                        ((uint32_t)__double2hiint(yy) - (uint32_t)(kHistMagicHi - 1)) |
                        ((uint32_t)__double2hiint(yz) - (uint32_t)(kHistMagicHi - 1));
    const uint32_t gx = (ux & (kHistOne - 1u)) - kHistBand, gy = (uy & (kHistOne - 1u)) - kHistBand,
                   gz = (uz & (kHistOne - 1u)) - kHistBand;
    const bool safe = hi <= 1u && max(ux, max(uy, uz)) < 3u * kHistOne && max(gx, max(gy, gz)) < kHistOne - 2u * kHistBand;
    if (CUBA_FORCE_SLOW_PATHS || !safe) return next_direction(g, dt, h.i0[0], h.i0[1], h.i0[2], x, y, z, px, py, pz, E);
    return (int)h.map[(ux >> 20) * 9u + (uy >> 20) * 3u + (uz >> 20)];
}

// Tile segments of a cell: the flat passes work on tiles of kTile consecutive slots; segment k of
// the cell [lo, lo+n) is its intersection with tile (lo / kTile) + k.  s_seg[k][d] counts the
// cell's particles of segment k that move in direction d.  From it:
//   cnt[d][c]              = sum over all segments                      (what K_A accumulates)
//   carry[tile T0+k][d]    = sum over segments before k, k >= 1         (what k_carry derives)
//   carry[tile T0][d]      = 0 if the cell starts exactly at the tile start
// Every tile start lies in exactly one non-empty cell, so every carry row is written once.
// Only the particles that leave the cell are counted one by one; the count of the direction "stays"
// (code 13) of a segment is its size minus the others (hist_fill_stay, between two barriers).
constexpr uint32_t kDirStay = 13u;

template <int THREADS>
__device__ __forceinline__ void hist_fill_stay(uint32_t lo, uint32_t n, uint32_t *s_seg)
{
    const uint32_t T0 = lo / kTile, nseg = (lo + n - 1u) / kTile - T0 + 1u;
    if (threadIdx.x < nseg) {
        const uint32_t k = threadIdx.x;
        const uint32_t a = max(lo, (T0 + k) * (uint32_t)kTile), b = min(lo + n, (T0 + k + 1u) * (uint32_t)kTile);
        uint32_t others = 0;
#pragma unroll
        for (uint32_t d = 0; d < (uint32_t)kDirs; ++d) others += (d == kDirStay) ? 0u : s_seg[k * kDirs + d];
        s_seg[k * kDirs + kDirStay] = (b - a) - others;
    }
}

template <int THREADS>
__device__ __forceinline__ void hist_publish(const CollideParams &P, uint32_t c, uint32_t lo, uint32_t n,
                                             const uint32_t *s_seg)
{
    const uint32_t T0 = lo / kTile, nseg = (lo + n - 1u) / kTile - T0 + 1u;
    for (uint32_t e = threadIdx.x; e < nseg * kDirs; e += THREADS) {
        const uint32_t k = e / kDirs, d = e - k * kDirs;
        uint32_t before = 0;
        for (uint32_t q = 0; q < k; ++q) before += s_seg[q * kDirs + d];
        if (k > 0 || lo % kTile == 0) P.carry[(size_t)(T0 + k) * kTileRec + d] = before;
        if (k == nseg - 1u) P.cnt[(size_t)d * P.g.ncells + c] = before + s_seg[k * kDirs + d];
    }
}

// ---- shared-memory classes ------------------------------------------------------------
// Same results as the generic routine above, organised for instruction count and issue efficiency on
// sm_100a.  The momentum-independent part of TWO consecutive rounds (the two shuffles) is done in one
// sweep, then the two rounds' pair phases follow:
//
//   rank by bitmap.  The keys are uniform 32-bit numbers, so a cell of n particles gets a bitmap of
//     M = 32 n bits (n words): bit b = floor(key * M / 2^32), monotone in the key.  Phase A: one
//     atomicOr per element and round; an element that finds its bit already set adds one to the
//     word's duplicate counter.  Phase B: an exclusive scan over the words of popc(word) +
//     duplicates, both rounds packed into one 32-bit scan.  Phase C: rank = prefix of the word +
//     popc(bits below mine) -- two loads and a popc, no parked keys, no comparisons.  The ~5 % of the
//     elements whose word holds a duplicate ("dirty" words) put (key, word, index) on a short list
//     at the end of phase C (every thread lists its own, one per loop trip: a branch taken once per
//     item and round would be executed by almost every warp for one or two lanes) and rank themselves
//     inside the word by scanning that list, with the pid deciding
//     between equal 32-bit keys (A7); if the list overflows (never with uniform keys; forced in the
//     slow-paths test build) a brute-force count over recomputed keys takes over.  The result depends
//     on keys and pids only, never on the order in which threads arrived.
//   pair phases.  Energies are not staged: the first pair phase of a sweep computes E = |p| of both
//     partners for its Eq. 3 decision anyway and leaves them in shared memory -- in the space of the
//     two bitmaps, which are dead by then -- for the second round, the scatters and the fused
//     histogram.  The decision compares u*(EaEb)^2 with |d|^2*scale/2 (no division); only a decision
//     inside a 4e-9 band around the threshold is redone with the exact operation order of the
//     oracle, so the decisions (and the near-threshold counter, A16) are the oracle's bit for bit.
//     Hits are compacted per warp and a warp scatters its own hits right away (pairs are disjoint).
//
// Shared memory: 44 B per particle (p_x,p_y as one 16-byte element, p_z, pid, two bitmaps | E,
// packed duplicate counters | prefixes, two 16-bit orders).  Block barriers per sweep of two rounds: 7;
// per cell otherwise: staging, end of the rounds, fused histogram (2), end of the cell (which also publishes the
// claim of the cell after next).

// 53-bit uniform from two Philox words, same value as u53(): both halves are exact integers
// below 2^27 placed in the mantissa of 2^52, so every operation below is exact.
__device__ __forceinline__ double u53_bits(uint32_t w0, uint32_t w1)
{
    const double hi = __hiloint2double(0x43300000, (int)(w0 >> 5)) - 4503599627370496.0;
    const double lo = __hiloint2double(0x43300000, (int)(w1 >> 6)) - 4503599627370496.0;
    return (hi * 67108864.0 + lo) * (1.0 / 9007199254740992.0);
}

// Marsaglia disc rejection (A11) with the key schedule from the parameters.  Both attempts of the
// first call are evaluated without a branch (95 % of the draws end there) so that a warp stays
// converged; later calls are a rare loop.
__device__ __forceinline__ void disc_point(uint32_t wa, uint32_t wb, double &a, double &b, double &q)
{
    a = ((double)wa + 0.5) * (1.0 / 2147483648.0) - 1.0;
    b = ((double)wb + 0.5) * (1.0 / 2147483648.0) - 1.0;
    q = a * a + b * b;
}

__device__ __forceinline__ void draw_direction_k(const CollideParams &P, uint32_t t, uint32_t pid, uint32_t rho,
                                                 double &nx, double &ny, double &nz)
{
    const U4 w0 = drawk(P, t, pid, rho, kTagDir, 0);
    double a, b, q, a2, b2, q2;
    disc_point(w0.x, w0.y, a, b, q);
    disc_point(w0.z, w0.w, a2, b2, q2);
    bool ok = q < 1.0;
    if (!ok) { a = a2; b = b2; q = q2; ok = q2 < 1.0; }
    if (!ok) {
        for (uint32_t call = 1; call < 65536u && !ok; ++call) {
            const U4 w = drawk(P, t, pid, rho, kTagDir, call);
            disc_point(w.x, w.y, a, b, q);
            ok = q < 1.0;
            if (!ok) { disc_point(w.z, w.w, a, b, q); ok = q < 1.0; }
        }
        if (!ok) { nx = 0.0; ny = 0.0; nz = 1.0; return; }
    }
    const double h = sqrt(1.0 - q);
    nx = (2.0 * a) * h; ny = (2.0 * b) * h; nz = 1.0 - 2.0 * q;
}

// Boost to the CM frame, isotropic direction, boost back (closed form A10).
__device__ __forceinline__ void pair_scatter(const CollideParams &P, uint32_t t, uint32_t ida, uint32_t rho, double s,
                                             double pax, double pay, double paz, double Ea,
                                             double pbx, double pby, double pbz, double Eb,
                                             double q[6])
{
    double nx, ny, nz;
    draw_direction_k(P, t, ida, rho, nx, ny, nz);
    const double rs = sqrt(s);
    const double Pvx = pax + pbx, Pvy = pay + pby, Pvz = paz + pbz;
    const double Et = Ea + Eb;
    const double Pn = (Pvx * nx + Pvy * ny) + Pvz * nz;
    const double al = Pn / (Et + rs);
    const double f1 = 1.0 + al, f2 = 1.0 - al;
    q[0] = 0.5 * (rs * nx + Pvx * f1);
    q[1] = 0.5 * (rs * ny + Pvy * f1);
    q[2] = 0.5 * (rs * nz + Pvz * f1);
    q[3] = 0.5 * (Pvx * f2 - rs * nx);
    q[4] = 0.5 * (Pvy * f2 - rs * ny);
    q[5] = 0.5 * (Pvz * f2 - rs * nz);
}

// Exclusive block scan with one barrier; s_warp is next written a sweep (several barriers) later.
template <int THREADS>
__device__ __forceinline__ uint32_t block_exclusive_scan_1b(uint32_t v, uint32_t *s_warp)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, inc, o);
        if (lane >= o) inc += t;
    }
    if (THREADS == 32) return inc - v;
    if (lane == 31) s_warp[wid] = inc;
    __syncthreads();
    uint32_t w = (lane < THREADS / 32) ? s_warp[lane] : 0u;
    uint32_t winc = w;
#pragma unroll
    for (int o = 1; o < THREADS / 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, winc, o);
        if (lane >= o) winc += t;
    }
    return __shfl_sync(0xFFFFFFFFu, winc - w, wid) + inc - v;
}

// Last resort of the ranking inside a dirty word (the list of dirty elements overflowed): count
// the cell's elements of the same word with a smaller (key, pid), keys recomputed.
// (Scalars only: a reference to the kernel parameters would force a copy of them onto the stack.)
__device__ __noinline__ uint32_t brute_rank(uint64_t seed, uint32_t t, const uint32_t *spid, uint32_t n,
                                            uint32_t M, uint32_t word, uint32_t k, uint32_t id, int rho)
{
    uint32_t cnt = 0;
    for (uint32_t i = 0; i < n; ++i) {
        const uint32_t id2 = spid[i];
        const uint32_t k2 = shuf_word(draw(seed, id2, t, (uint32_t)rho >> 2, kTagShuf, 0), rho);
        if ((__umulhi(k2, M) >> 5) == word && (k2 < k || (k2 == k && id2 < id))) cnt += 1u;
    }
    return cnt;
}

// Rare path of the Eq. 3 decision: the exact operation order of the oracle.
// Returns bit 0: hit, bit 1: |u - P| <= 1e-12 (A16).
__device__ __noinline__ uint32_t exact_decision(double dd, double ee, double u, double scale)
{
    const double s = dd / ee;                 // (p_a+p_b)^2, A9
    const double vrel = 0.5 * (s / ee);       // s/(2 E_a E_b)
    const double prob = vrel * scale;         // Eq. 3 * cn/R
    return (u < prob ? 1u : 0u) | (fabs(u - prob) <= 1e-12 ? 2u : 0u);
}

constexpr int kChains = 64;
constexpr uint32_t kNil = 0xFFFFu;

// Per-CTA state in static shared memory: constants of the current cell that are only needed at a
// few places (kept out of registers across the register-hungry phases) and small counters.
struct CtaStats {
    double scale, hscale;     // Eq. 3 factor cn*base/R of the current cell, and half of it
    uint32_t lo;              // first slot of the current cell
    uint32_t near;            // near-threshold decisions of this CTA (A16; rare)
    uint32_t hits;            // collisions of this CTA since the last flush (lane 0 of every warp adds after a pair phase)
    unsigned long long pairs, rounds;   // pair evaluations and rounds of this CTA (thread 0 adds per cell)
    uint32_t nlist[2];        // entries on the two dirty-element lists of the current sweep
    uint32_t head[2][kChains]; // first entry of the chain of the words with (word mod kChains) equal, per list
    HistCell h;               // fused histogram: constants of the current cell
};

// Shared-memory arrays of one CTA: fixed offsets into the dynamic shared memory, so that every
// access is a shared-memory instruction with an immediate offset (no pointer registers).
extern __shared__ __align__(128) unsigned char cuba_smem[];

template <int CAP, int LCAP>
struct CellSmem {
    // (p_x, p_y) [CAP]
    static __device__ __forceinline__ double2 *pxy() { return reinterpret_cast<double2 *>(cuba_smem); }
    // p_z [CAP]
    static __device__ __forceinline__ double *pz() { return reinterpret_cast<double *>(cuba_smem + 16 * CAP); }
    // [2 CAP] bitmap of round A, bitmap of round B; as doubles: E[CAP] from the first pair phase on
    static __device__ __forceinline__ uint32_t *bm() { return reinterpret_cast<uint32_t *>(cuba_smem + 24 * CAP); }
    static __device__ __forceinline__ double *E() { return reinterpret_cast<double *>(cuba_smem + 24 * CAP); }
    static __device__ __forceinline__ uint32_t *pid() { return reinterpret_cast<uint32_t *>(cuba_smem + 32 * CAP); }
    // [CAP] per word: duplicates of round A | round B << 16; after the scan (prefix << 1 | dirty), packed alike
    static __device__ __forceinline__ uint32_t *cnt() { return reinterpret_cast<uint32_t *>(cuba_smem + 36 * CAP); }
    // [CAP] each: the order of round A / B
    static __device__ __forceinline__ uint16_t *ord(int slot) { return reinterpret_cast<uint16_t *>(cuba_smem + 40 * CAP) + slot * CAP; }
    // [LCAP] each, per round: dirty elements: key; word << 13 | index; prefix of the word | next entry of the chain << 16
    static __device__ __forceinline__ uint32_t *lkey(int slot) { return reinterpret_cast<uint32_t *>(cuba_smem + 44 * CAP) + 3 * LCAP * slot; }
    static __device__ __forceinline__ uint32_t *lwj(int slot) { return lkey(slot) + LCAP; }
    static __device__ __forceinline__ uint32_t *lpn(int slot) { return lkey(slot) + 2 * LCAP; }
    // [warps][PITEMS * 32] this warp's colliding pairs
    static __device__ __forceinline__ uint16_t *hits() { return reinterpret_cast<uint16_t *>(cuba_smem + 44 * CAP + 24 * LCAP); }
};

__host__ __device__ constexpr int collide_list_cap(int cap) { return cap / 8 > 64 ? cap / 8 : 64; }
__host__ __device__ constexpr size_t collide_smem_bytes(int cap, int threads, int items)
{
    return (size_t)cap * 44 + 2 * (size_t)collide_list_cap(cap) * 12 + (size_t)threads * ((items + 1) / 2) * 2 + 64;
}

// One pair phase (one round): Eq. 3 decision for the pairs order[2k], order[2k+1], then this warp's
// hits are scattered.  first: the energies are computed here and left in sE (see above).  The pairs
// are dealt to the warps in rows of 32, round-robin (the hits, and with them the scatter work, are
// then spread evenly: a warp rarely has more than 32); a warp skips the rows beyond the last pair.
// (Measured and rejected: the decisions of a warp's three rows interleaved through register arrays,
// hot class 0.788 -> 0.804 ms.)
template <typename S, int THREADS, int PITEMS, bool TRACE>
__device__ __forceinline__ void pair_phase(const CollideParams &P, uint32_t c, uint32_t n, uint32_t tcur, int rho,
                                            int slot, bool first, bool keepE, CtaStats *stats)
{
    const uint16_t *sord = S::ord(slot);
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const uint32_t npairs = n >> 1;
    constexpr int W = THREADS / 32;
    double *sE = S::E();
    uint16_t *shit = S::hits() + wid * (PITEMS * 32);
    if (first && tid == 0 && (n & 1u)) {          // the particle left over by the pairing: nobody else computes its energy
        const uint32_t i = sord[n - 1u];
        const double2 xy = S::pxy()[i];
        sE[i] = energy(xy.x, xy.y, S::pz()[i]);
    }
    uint32_t nh = 0;
    {
        const double scale = *reinterpret_cast<volatile double *>(&stats->scale);
        const double hscale = *reinterpret_cast<volatile double *>(&stats->hscale);
        // row r = it * W + wid holds the pairs [32 r, 32 r + 32); rows that start beyond the last pair are skipped
        // by the whole warp (no Philox, no loads for padding)
#pragma unroll
        for (int it = 0; it < PITEMS; ++it) {
            const uint32_t row0 = (uint32_t)(it * W + wid) * 32u;
            if (row0 >= npairs) break;
            const uint32_t k = row0 + lane;
            const uint32_t kc = min(k, npairs - 1u);
            const uint32_t ab = *reinterpret_cast<const uint32_t *>(sord + 2 * kc);
            const uint32_t a = ab & 0xFFFFu, b = ab >> 16;
            const double2 pa = S::pxy()[a], pb = S::pxy()[b];
            const double paz = S::pz()[a], pbz = S::pz()[b];
            const uint32_t ida = S::pid()[a];
            double Ea, Eb;
            if (first) {
                Ea = energy(pa.x, pa.y, paz); Eb = energy(pb.x, pb.y, pbz);
                if (k < npairs) { sE[a] = Ea; sE[b] = Eb; }
            } else {
                Ea = sE[a]; Eb = sE[b];
            }
            const double dx = Eb * pa.x - Ea * pb.x;
            const double dy = Eb * pa.y - Ea * pb.y;
            const double dz = Eb * paz - Ea * pbz;
            const double ee = Ea * Eb;
            const double dd = (dx * dx + dy * dy) + dz * dz;
            const U4 w = drawk(P, tcur, ida, (uint32_t)rho, kTagDec, 0);
            const double u = u53_bits(w.x, w.y);
            bool hit;
            if (TRACE) {
                const double s = dd / ee;                 // (p_a+p_b)^2, A9
                const double vrel = 0.5 * (s / ee);       // s/(2 E_a E_b)
                const double prob = vrel * scale;         // Eq. 3 * cn/R
                hit = u < prob;
                if (k < npairs) {
                    if (fabs(u - prob) <= 1e-12) atomicAdd(&stats->near, 1u);
                    const unsigned long long e = P.trace_off[c] + (unsigned long long)rho * npairs + k;
                    P.tr_cell[e] = c; P.tr_round[e] = (uint32_t)rho; P.tr_pa[e] = ida; P.tr_pb[e] = S::pid()[b];
                    P.tr_P[e] = prob; P.tr_u[e] = u; P.tr_dec[e] = hit ? 1 : 0;
                }
            } else {
                // sign(u - P) from u*(EaEb)^2 - |d|^2*scale/2; the exact form only inside a band
                // far wider than the rounding error (it also catches NaN, inf and underflow)
                const double ee2 = ee * ee;
                const double diff = u * ee2 - dd * hscale;
                hit = diff < 0.0;
                if (CUBA_FORCE_SLOW_PATHS || !(fabs(diff) > 4e-9 * ee2) || !(ee2 > 1e-280)) {
                    const uint32_t r = exact_decision(dd, ee, u, scale);
                    hit = (r & 1u) != 0;
                    if ((r & 2u) && k < npairs) atomicAdd(&stats->near, 1u);
                }
            }
            hit = hit && k < npairs;
            const uint32_t hm = __ballot_sync(0xFFFFFFFFu, hit);
            if (hit) shit[nh + __popc(hm & lanemask_lt())] = (uint16_t)k;
            nh += __popc(hm);
        }
    }
    __syncwarp();
    // scatter this warp's colliding pairs, densely
    for (uint32_t h = lane; h < nh; h += 32) {
        const uint32_t k = shit[h];
        const uint32_t ab = *reinterpret_cast<const uint32_t *>(sord + 2 * k);
        const uint32_t a = ab & 0xFFFFu, b = ab >> 16;
        const double2 pa = S::pxy()[a], pb = S::pxy()[b];
        const double paz = S::pz()[a], pbz = S::pz()[b];
        const double Ea = sE[a], Eb = sE[b];
        const double ee = Ea * Eb;
        const double dx = Eb * pa.x - Ea * pb.x;
        const double dy = Eb * pa.y - Ea * pb.y;
        const double dz = Eb * paz - Ea * pbz;
        const double s = ((dx * dx + dy * dy) + dz * dz) / ee;
        double q[6];
        pair_scatter(P, tcur, S::pid()[a], (uint32_t)rho, s, pa.x, pa.y, paz, Ea, pb.x, pb.y, pbz, Eb, q);
        S::pxy()[a] = make_double2(q[0], q[1]); S::pz()[a] = q[2];
        S::pxy()[b] = make_double2(q[3], q[4]); S::pz()[b] = q[5];
        if (keepE) { sE[a] = energy(q[0], q[1], q[2]); sE[b] = energy(q[3], q[4], q[5]); }
    }
    if (lane == 0 && nh) atomicAdd(&stats->hits, nh);
    __syncwarp();   // the hit list is rewritten in the next pair phase
}

// Phase C1 for one element and one of the two rounds of a sweep (slot 0 / 1): the rank of an element of
// a clean word; an element of a dirty word goes onto the round's list, chained by word mod kChains.
// Clean part, straight-line: rank of the element if its word holds no duplicate, stored right away; returns true
// for an element of a dirty word, which rank_listed handles.
template <typename S, int SLOT>
__device__ __forceinline__ bool rank_clean(uint32_t k, uint32_t j, bool valid, uint32_t n, uint32_t M)
{
    const uint32_t b = __umulhi(k, M), word = b >> 5, below = (1u << (b & 31u)) - 1u;
    const uint32_t cw = S::cnt()[word];
    const uint32_t pw = SLOT ? (cw >> 16) : (cw & 0xFFFFu);
    const uint32_t rank = (pw >> 1) + __popc((S::bm() + SLOT * n)[word] & below);
    const bool dirty = CUBA_FORCE_SLOW_PATHS || (pw & 1u);
    if (valid && !dirty) S::ord(SLOT)[rank] = (uint16_t)j;
    return valid && dirty;
}

// An element of a dirty word goes onto the round's list, chained by word mod kChains (phase C2 ranks it).
// slot is a run-time value here: the few listed elements of a thread are handled one after the other.
template <typename S, int LCAP>
__device__ __forceinline__ void rank_listed(const CollideParams &P, CtaStats *stats, int slot,
                                            uint32_t k, uint32_t j, uint32_t n, uint32_t M,
                                            uint32_t tcur, int rho)
{
    const uint32_t b = __umulhi(k, M), word = b >> 5;
    const uint32_t cw = S::cnt()[word];
    const uint32_t pw = slot ? (cw >> 16) : (cw & 0xFFFFu);
    const uint32_t at = atomicAdd(&stats->nlist[slot], 1u);
    if (at < (uint32_t)LCAP) {
        const uint32_t next = atomicExch(&stats->head[slot][word % kChains], at);
        S::lkey(slot)[at] = k;
        S::lwj(slot)[at] = (word << 13) | j;
        S::lpn(slot)[at] = (pw >> 1) | (next << 16);
        return;
    }
    const uint32_t rank = (pw >> 1) + brute_rank(P.seed, tcur, S::pid(), n, M, word, k, S::pid()[j], rho);   // the list is full
    S::ord(slot)[rank] = (uint16_t)j;
}

// Phase C2, one thread per list entry (the two lists side by side, each on its own half of the CTA): rank
// inside the dirty word = entries of the same word with a smaller (key, pid), found on the word's chain.
template <typename S, int LCAP, int THREADS>
__device__ __forceinline__ void rank_dirty(const CollideParams &P, const CtaStats *stats, uint32_t n, uint32_t M,
                                           uint32_t tcur, int rho0, bool two)
{
    constexpr int HALF = THREADS >= 64 ? THREADS / 2 : THREADS;
    const int slot = (THREADS >= 64 && (int)threadIdx.x >= HALF) ? 1 : 0;
    for (int pass = 0; pass < (THREADS >= 64 ? 1 : 2); ++pass) {
        const int sl = THREADS >= 64 ? slot : pass;
        if (sl == 1 && !two) break;
        const uint32_t nl = stats->nlist[sl];
        for (uint32_t i = threadIdx.x - (THREADS >= 64 ? sl * HALF : 0); i < min(nl, (uint32_t)LCAP); i += HALF) {
            const uint32_t k = S::lkey(sl)[i], wj = S::lwj(sl)[i];
            const uint32_t word = wj >> 13, j = wj & 0x1FFFu, id = S::pid()[j];
            uint32_t cnt = 0;
            if (nl <= (uint32_t)LCAP) {
                for (uint32_t q = stats->head[sl][word % kChains]; q != kNil; q = S::lpn(sl)[q] >> 16) {
                    const uint32_t wj2 = S::lwj(sl)[q], k2 = S::lkey(sl)[q];
                    if ((wj2 >> 13) == word && (k2 < k || (k2 == k && S::pid()[wj2 & 0x1FFFu] < id))) cnt += 1u;
                }
            } else {
                cnt = brute_rank(P.seed, tcur, S::pid(), n, M, word, k, id, rho0 + sl);   // some elements of the word may be missing from the list
            }
            S::ord(sl)[(S::lpn(sl)[i] & 0xFFFFu) + cnt] = (uint16_t)j;
        }
    }
}

// All R rounds of one staged cell, two per sweep (see above).  On entry: momenta and pids staged, both
// bitmaps, the duplicate counters, the list counters and chain heads cleared, a block barrier passed.
// keepE: the caller needs the energies of the final momenta in sE afterwards.
template <int THREADS, int ITEMS, int G, int CAP, int LCAP, bool TRACE>
__device__ __forceinline__ void run_sweeps(const CollideParams &P, uint32_t c, uint32_t n, int R, uint32_t tcur,
                                               bool hist, uint32_t *s_warp, CtaStats *stats
#ifdef CUBA_PHASE_CLOCKS
                                               , long long &g_last
#endif
                                               )
{
    using S = CellSmem<CAP, LCAP>;
    constexpr int NG = ITEMS / G;
    constexpr int PITEMS = (ITEMS + 1) / 2;          // pairs per thread
    constexpr int SCAN = ITEMS | 1;                  // words per thread in the scan (odd stride: no bank conflicts)
    const int tid = threadIdx.x;
    const uint32_t last = n - 1u;
    const uint32_t M = 32u * n;                      // bits of a bitmap: word = bit >> 5 < n
    uint32_t *bmA = S::bm(), *bmB = S::bm() + n;
    // items it of this warp with a particle in them: (tid & ~31) + it * THREADS < n
    const int nit = (int)min((uint32_t)ITEMS, (n + (uint32_t)THREADS - 1u - min(n, (uint32_t)(tid & ~31))) / (uint32_t)THREADS);
    for (int rho0 = 0; rho0 < R; rho0 += 2) {
        const bool two = rho0 + 1 < R;
        if (rho0 > 0) {
            // later sweeps: the energies (in the bitmaps' space) are dead again until the next pair phase
            __syncthreads();
#pragma unroll
            for (int it = 0; it < ITEMS; ++it) {
                const uint32_t j = tid + it * THREADS;
                if (j < n) { *reinterpret_cast<uint2 *>(S::bm() + 2 * j) = make_uint2(0u, 0u); S::cnt()[j] = 0; }
            }
            for (int e = tid; e < 2 * kChains; e += THREADS) (&stats->head[0][0])[e] = kNil;
            if (tid == 0) { stats->nlist[0] = 0; stats->nlist[1] = 0; }
            __syncthreads();
        }
        uint32_t keyA[ITEMS], keyB[ITEMS];
        // (A) shuffle keys of the two rounds (A7: words 2*(sweep mod 2), +1 of the call for rounds
        // 4*(rho div 4)..+3) and one atomicOr per element and round.  nit: items of this warp that hold
        // particles (warp-uniform): a warp does no Philox and no ranking for the padding of the class.
#pragma unroll
        for (int g = 0; g < NG; ++g) {
            if (g * G >= nit) break;
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const int it = g * G + i;
                keyA[it] = 0; keyB[it] = 0;
                if (it < nit) {
                    const uint32_t jc = min((uint32_t)(tid + it * THREADS), last);
                    const U4 w = drawk(P, tcur, S::pid()[jc], (uint32_t)rho0 >> 2, kTagShuf, 0);
                    keyA[it] = (rho0 & 2) ? w.z : w.x;
                    keyB[it] = (rho0 & 2) ? w.w : w.y;
                }
            }
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const int it = g * G + i;
                const uint32_t j = tid + it * THREADS;
                if (it < nit && j < n) {
                    const uint32_t bA = __umulhi(keyA[it], M), mA = 1u << (bA & 31u);
                    if (atomicOr(&bmA[bA >> 5], mA) & mA) atomicAdd(&S::cnt()[bA >> 5], 1u);
                    if (two) {
                        const uint32_t bB = __umulhi(keyB[it], M), mB = 1u << (bB & 31u);
                        if (atomicOr(&bmB[bB >> 5], mB) & mB) atomicAdd(&S::cnt()[bB >> 5], 0x10000u);
                    }
                }
            }
        }
        __syncthreads();
        CUBA_MARK(1);
        // (B) per word: elements = popc + duplicates, both rounds packed in one word; exclusive scan
        {
            const uint32_t chunk = ((n + THREADS - 1) / THREADS) | 1u;
            const uint32_t w0 = min(n, tid * chunk), w1 = min(n, w0 + chunk);
            uint32_t v[SCAN], sum = 0, dirty = 0;
#pragma unroll
            for (int q = 0; q < SCAN; ++q) {
                v[q] = 0;
                if (w0 + q < w1) {
                    const uint32_t cw = S::cnt()[w0 + q];
                    v[q] = (__popc(bmA[w0 + q]) + (cw & 0xFFFFu)) + ((__popc(bmB[w0 + q]) + (cw >> 16)) << 16);
                    dirty |= (((cw & 0xFFFFu) ? 1u : 0u) | ((cw >> 16) ? 2u : 0u)) << (2 * q);
                }
                sum += v[q];
            }
            uint32_t run = block_exclusive_scan_1b<THREADS>(sum, s_warp);   // its barrier separates the reads of cnt above from the writes below
            if (THREADS == 32) __syncwarp();
#pragma unroll
            for (int q = 0; q < SCAN; ++q) {
                if (w0 + q < w1) {
                    const uint32_t d = (dirty >> (2 * q)) & 3u;
                    S::cnt()[w0 + q] = (((run & 0xFFFFu) << 1) | (d & 1u)) | ((((run >> 16) << 1) | (d >> 1)) << 16);
                }
                run += v[q];
            }
        }
        __syncthreads();
        CUBA_MARK(2);
        // (C1) rank = prefix of the word + occupied bits below mine, all items of the thread in one straight-line
        // block; then every thread lists its elements of dirty words one after the other (about 5 % of the
        // elements: a warp loops two or three times instead of branching once per item and round)
        uint32_t listed = 0;
#pragma unroll
        for (int it = 0; it < ITEMS; ++it) {
            const uint32_t j = tid + it * THREADS;
            const bool valid = it < nit && j < n;
            listed |= (rank_clean<S, 0>(keyA[it], j, valid, n, M) ? 1u : 0u) << (2 * it);
            if (two) listed |= (rank_clean<S, 1>(keyB[it], j, valid, n, M) ? 2u : 0u) << (2 * it);
        }
        while (__any_sync(0xFFFFFFFFu, listed != 0u)) {
            if (listed) {
                const int e = __ffs(listed) - 1, it = e >> 1, sl = e & 1;
                listed &= listed - 1u;
                uint32_t k = 0;
#pragma unroll
                for (int q = 0; q < ITEMS; ++q) k = (q == it) ? (sl ? keyB[q] : keyA[q]) : k;
                rank_listed<S, LCAP>(P, stats, sl, k, tid + it * THREADS, n, M, tcur, rho0 + sl);
            }
        }
        __syncthreads();
        CUBA_MARK(3);
        // (C2) the listed elements, one thread each
        rank_dirty<S, LCAP, THREADS>(P, stats, n, M, tcur, rho0, two);
        __syncthreads();
        CUBA_MARK(4);
        // pair phases of the two rounds; energies appear in the first one
#pragma unroll 1
        for (int sl = 0; sl < (two ? 2 : 1); ++sl) {
            if (sl) { __syncthreads(); CUBA_MARK(5); }
            pair_phase<S, THREADS, PITEMS, TRACE>(P, c, n, tcur, rho0 + sl, sl, sl == 0, sl == 0 ? (two || hist) : hist, stats);
        }
    }
}

template <int THREADS, int ITEMS, int G, int CAP, int LCAP, bool TRACE, bool LOCAL, bool GRAPH>
__device__ __forceinline__ void collide_cell_smem(const CollideParams &P, uint32_t c, uint32_t lo, uint32_t n,
                                                  uint32_t *s_warp, CtaStats *stats,
                                                  uint32_t *s_seg, long long *s_esum,
                                                  uint32_t lo_next, uint32_t n_next
#ifdef CUBA_PHASE_CLOCKS
                                                  , long long &g_last
#endif
                                                  )
{
    static_assert(ITEMS % G == 0, "items are processed in groups of G");
    constexpr int NG = ITEMS / G;
    using S = CellSmem<CAP, LCAP>;
    const int tid = threadIdx.x;
    // step index: a constant-bank operand normally; a register loaded from device memory when the
    // kernel is a node of a replayed CUDA graph (small problems only, where registers are plentiful)
    const uint32_t tcur = GRAPH ? *P.t_dev : P.t;
    const bool hist = P.next_dt > 0.0;
    constexpr bool local = LOCAL;     // compile-time: the constant-sigma kernels carry none of its registers
    // rounds and scale (A5, A6): identical integer/fp64 results on every thread.  With the local
    // cross section the factor needs the cell's energy sum and is computed after staging.
    double base = P.base;
    const double cn = (n & 1u) ? (double)n : (double)(n - 1u);
    int R = 0;
    if (!local) {
        const double pmax = (2.0 * cn) * base;
        if (!(pmax <= 64.0)) { if (tid == 0) atomicOr(P.flags, kFlagRounds); R = 64; }
        else R = (pmax <= 1.0) ? 1 : (int)ceil(pmax);
        if (n < 2u) R = 0;          // a single particle has no partner; it is here for the fused histogram only
    }
    for (int e = tid; e < 2 * kChains; e += THREADS) (&stats->head[0][0])[e] = kNil;
    if (tid == 0) {
        stats->lo = lo;
        stats->nlist[0] = 0; stats->nlist[1] = 0;
        if (!local) {
            const double scale = (cn * base) / (double)R;
            stats->scale = scale; stats->hscale = 0.5 * scale;
        }
    }
    if (hist && tid < 32) hist_cell_setup(P.g, c, &stats->h, tid);
    const uint32_t last = n - 1u;
    const uint32_t M = 32u * n;                      // bits of a bitmap: word = bit >> 5 < n
    uint32_t *bmA = S::bm(), *bmB = S::bm() + n;
    double *sE = S::E();   // E[n] covers exactly the two bitmaps (2 n words)

    // ---- stage the cell: momenta and pids; clear the bitmaps and the duplicate counters ---------
    long long esum = 0;
#pragma unroll
    for (int g = 0; g < NG; ++g) {
        if ((uint32_t)(g * G * THREADS) >= n) break;
        double a[G], b[G], cc[G];
        uint32_t id[G];
#pragma unroll
        for (int i = 0; i < G; ++i) {
            const uint32_t jc = lo + min((uint32_t)(tid + (g * G + i) * THREADS), last);
            a[i] = P.px[jc]; b[i] = P.py[jc]; cc[i] = P.pz[jc]; id[i] = P.pid[jc];
        }
#pragma unroll
        for (int i = 0; i < G; ++i) {
            const uint32_t j = tid + (g * G + i) * THREADS;
            if (j < n) {
                S::pxy()[j] = make_double2(a[i], b[i]); S::pz()[j] = cc[i]; S::pid()[j] = id[i];
                *reinterpret_cast<uint2 *>(S::bm() + 2 * j) = make_uint2(0u, 0u); S::cnt()[j] = 0;
                if (local) esum += energy_fixed(energy(a[i], b[i], cc[i]));
            }
        }
    }
    if (hist)
        for (uint32_t e = tid; e < ((lo + n - 1u) / kTile - lo / kTile + 1u) * kDirs; e += THREADS) s_seg[e] = 0;
    if (local) block_sum_ll_post<THREADS>(esum, s_esum);
    __syncthreads();
    CUBA_MARK(0);
    if (local) {
        base = local_base(block_sum_ll_read<THREADS>(s_esum), n, P.dt, P.etas);
        const double pmax = (2.0 * cn) * base;
        if (!(pmax <= 64.0)) { if (tid == 0) atomicOr(P.flags, kFlagRounds); R = 64; }
        else R = (pmax <= 1.0) ? 1 : (int)ceil(pmax);
        if (n < 2u) R = 0;
        if (tid == 0) {             // read in the pair phases, several barriers from here
            const double scale = (cn * base) / (double)R;
            stats->scale = scale; stats->hscale = 0.5 * scale;
        }
    }
    // the CTA's next cell goes to L2 while this one is processed, so its load phase does not wait on DRAM
    for (uint32_t l = tid * 16u; n_next && l < n_next + 16u; l += THREADS * 16u) {   // one 128 B line of doubles per thread
        const uint32_t e = lo_next + min(l, n_next - 1u);
        prefetch_l2(P.px + e); prefetch_l2(P.py + e); prefetch_l2(P.pz + e);
        if ((l & 16u) == 0) prefetch_l2(P.pid + e);
        if (hist) { prefetch_l2(P.x + e); prefetch_l2(P.y + e); prefetch_l2(P.z + e); }
    }

#ifdef CUBA_PHASE_CLOCKS
    run_sweeps<THREADS, ITEMS, G, CAP, LCAP, TRACE>(P, c, n, R, tcur, hist, s_warp, stats, g_last);
#else
    run_sweeps<THREADS, ITEMS, G, CAP, LCAP, TRACE>(P, c, n, R, tcur, hist, s_warp, stats);
#endif
    if (R == 0 && hist && tid == 0) {     // a lone particle: no pair phase has computed its energy
        const double2 xy = S::pxy()[0];
        sE[0] = energy(xy.x, xy.y, S::pz()[0]);
    }
    __syncthreads();
    CUBA_MARK(6);
    const uint32_t lo_w = *reinterpret_cast<volatile uint32_t *>(&stats->lo);
    constexpr int HB = (ITEMS % 2 == 0) ? 2 : 1;
#pragma unroll 1
    for (uint32_t j = tid; j < n; j += THREADS) {
        const double2 xy = S::pxy()[j];
        P.px[lo_w + j] = xy.x; P.py[lo_w + j] = xy.y; P.pz[lo_w + j] = S::pz()[j];
    }
    if (tid == 0) { stats->pairs += (unsigned long long)R * (n >> 1); stats->rounds += (unsigned long long)R; }

    // ---- fused histogram of the next step (S1-S3 of step t+1 on the final momenta) ----------
    // The positions of group g + 1 are in flight while group g is worked on (the loads hit L2: the cell was
    // prefetched while the previous one was processed; their latency is what this phase used to wait for).
    if (hist) {
        const uint32_t T0 = lo_w / kTile;
        const HistCell &hc = stats->h;
        constexpr int NGH = ITEMS / HB;
        double xx[HB], yy[HB], zz[HB];
#pragma unroll
        for (int i = 0; i < HB; ++i) {
            const uint32_t jc = lo_w + min((uint32_t)(tid + i * THREADS), last);
            xx[i] = P.x[jc]; yy[i] = P.y[jc]; zz[i] = P.z[jc];
        }
#pragma unroll 1
        for (int g = 0; g < NGH; ++g) {
            if ((uint32_t)(g * HB * THREADS) >= n) break;
            double xn[HB], yn[HB], zn[HB];
            const bool more = g + 1 < NGH && (uint32_t)((g + 1) * HB * THREADS) < n;
#pragma unroll
            for (int i = 0; i < HB; ++i) {
                const uint32_t jc = lo_w + min((uint32_t)(tid + ((g + 1) * HB + i) * THREADS), last);
                xn[i] = xx[i]; yn[i] = yy[i]; zn[i] = zz[i];
                if (more) { xn[i] = P.x[jc]; yn[i] = P.y[jc]; zn[i] = P.z[jc]; }
            }
#pragma unroll
            for (int i = 0; i < HB; ++i) {
                const uint32_t j = tid + (g * HB + i) * THREADS, jj = min(j, last);
                const double2 xy = S::pxy()[jj];
                const int d = next_direction_guarded(P.g, P.next_dt, hc, xx[i], yy[i], zz[i], xy.x, xy.y, S::pz()[jj], sE[jj]);
                if (j < n && d != (int)kDirStay) {
                    if (d < 0) atomicOr(P.flags, kFlagMoved);
                    atomicAdd(&s_seg[((lo_w + j) / kTile - T0) * kDirs + (uint32_t)max(d, 0)], 1u);
                }
            }
#pragma unroll
            for (int i = 0; i < HB; ++i) { xx[i] = xn[i]; yy[i] = yn[i]; zz[i] = zn[i]; }
        }
        __syncthreads();
        CUBA_MARK(7);
        hist_fill_stay<THREADS>(lo_w, n, s_seg);
        __syncthreads();
        hist_publish<THREADS>(P, c, lo_w, n, s_seg);
    }
}

// Fused histogram for the overflow class: any n, one tile segment after the other.
template <int THREADS>
__device__ __forceinline__ void hist_cell_generic(const CollideParams &P, uint32_t c, uint32_t lo, uint32_t n,
                                                  const double *sE, uint32_t *s_run)
{
    const int tid = threadIdx.x;
    const uint32_t T0 = lo / kTile, nseg = (lo + n - 1u) / kTile - T0 + 1u;
    const int iz0 = (int)(c % (uint32_t)P.g.nc[2]);
    const int iy0 = (int)((c / (uint32_t)P.g.nc[2]) % (uint32_t)P.g.nc[1]);
    const int ix0 = (int)(c / ((uint32_t)P.g.nc[2] * (uint32_t)P.g.nc[1]));
    if (tid < kDirs) s_run[tid] = 0;
    __syncthreads();
    for (uint32_t k = 0; k < nseg; ++k) {
        if (tid < kDirs && (k > 0 || lo % kTile == 0)) P.carry[(size_t)(T0 + k) * kTileRec + tid] = s_run[tid];
        __syncthreads();
        const uint32_t j0 = max(lo, (T0 + k) * (uint32_t)kTile) - lo;
        const uint32_t j1 = min(lo + n, (T0 + k + 1u) * (uint32_t)kTile) - lo;
        for (uint32_t j = j0 + tid; j < j1; j += THREADS) {
            const int d = next_direction(P.g, P.next_dt, ix0, iy0, iz0, P.x[lo + j], P.y[lo + j], P.z[lo + j],
                                         P.px[lo + j], P.py[lo + j], P.pz[lo + j], sE[j]);
            if (d < 0) atomicOr(P.flags, kFlagMoved);
            atomicAdd(&s_run[max(d, 0)], 1u);
        }
        __syncthreads();
    }
    if (tid < kDirs) P.cnt[(size_t)tid * P.g.ncells + c] = s_run[tid];
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

// Shared-memory classes: CAP particles at most, 44 B of shared memory per particle.  The next
// work item is fetched one cell ahead and its momenta / pids are prefetched into L2 while
// the current cell is processed, so the load phase does not wait on DRAM.
template <int THREADS, int ITEMS, int CAP, int MIN_BLOCKS, bool TRACE, bool LOCAL, bool GRAPH>
__global__ void __launch_bounds__(THREADS, MIN_BLOCKS)
k_collide(CollideParams P)
{
    static_assert(CAP <= THREADS * ITEMS && CAP < 8192 && CAP % 32 == 0, "class capacity");
#ifndef CUBA_G6
#define CUBA_G6 3
#endif
    constexpr int G = (ITEMS == 6) ? CUBA_G6 : ((ITEMS % 2 == 0) ? 2 : ITEMS);
    constexpr int LCAP = collide_list_cap(CAP);
    constexpr int PITEMS = (ITEMS + 1) / 2;
    static_assert(collide_smem_bytes(CAP, THREADS, ITEMS) >= (size_t)CAP * 44 + 24 * (size_t)LCAP + (size_t)THREADS * PITEMS * 2, "carve");
    __shared__ uint32_t s_warp[32];
    __shared__ CtaStats s_stats;
    __shared__ uint32_t s_seg[((CAP + kTile - 2) / kTile + 1) * kDirs];   // a cell of CAP particles spans at most this many tiles
    __shared__ long long s_esum[32];

    // Dynamic work distribution, claimed one cell ahead so that the next cell can be prefetched
    // into L2.  (Measured alternatives, both slower because they lengthen the tail of the list:
    // a static round-robin, +0.10 ms at configs[2]; claiming three cells ahead, +0.09 ms.)
    const uint32_t nlist = *P.list_count;
    if (threadIdx.x == 0) { s_stats.near = 0; s_stats.hits = 0; s_stats.pairs = 0; s_stats.rounds = 0; }
    __shared__ uint32_t s_item[2];
    if (threadIdx.x == 0) { s_item[0] = atomicAdd(P.work, 1u); s_item[1] = 0xFFFFFFFFu; }
    __syncthreads();
    uint32_t item = s_item[0];
    uint4 cur = make_uint4(0u, 0u, 0u, 0u);
    if (item < nlist) cur = P.list[item];
    if (threadIdx.x == 0 && item < nlist) s_item[1] = atomicAdd(P.work, 1u);
    __syncthreads();
#ifdef CUBA_PHASE_CLOCKS
    long long g_last = clock64();
#endif
    // One block barrier per cell: thread 0 claims the cell after the next one at the END of a cell, so that the
    // barrier that frees the shared memory for the next cell also publishes the claim.
    for (int it = 0; item < nlist; ++it) {
        const uint32_t item_next = s_item[(it + 1) & 1];
        uint4 nxt = make_uint4(0u, 0u, 0u, 0u);
        if (item_next < nlist) nxt = P.list[item_next];   // first used after the staging barrier
#ifdef CUBA_PHASE_CLOCKS
        collide_cell_smem<THREADS, ITEMS, G, CAP, LCAP, TRACE, LOCAL, GRAPH>(P, cur.x, cur.y, cur.z, s_warp, &s_stats, s_seg, s_esum,
                                                                        nxt.y, nxt.z, g_last);
#else
        collide_cell_smem<THREADS, ITEMS, G, CAP, LCAP, TRACE, LOCAL, GRAPH>(P, cur.x, cur.y, cur.z, s_warp, &s_stats, s_seg, s_esum,
                                                                        nxt.y, nxt.z);
#endif
        if (threadIdx.x == 0) s_item[it & 1] = item_next < nlist ? atomicAdd(P.work, 1u) : 0xFFFFFFFFu;
        __syncthreads();
        CUBA_MARK(8);
        cur = nxt;
        item = item_next;
    }
    if (threadIdx.x == 0) {       // the loop ends with a block barrier
        if (s_stats.hits) atomicAdd(&P.counters[1], (unsigned long long)s_stats.hits);
        if (s_stats.pairs) atomicAdd(&P.counters[0], s_stats.pairs);
        if (s_stats.rounds) atomicAdd(&P.counters[2], s_stats.rounds);
        if (s_stats.near) atomicAdd(&P.counters[3], (unsigned long long)s_stats.near);
    }
}

// step index in device memory for graph replays
__global__ void k_set_t(uint32_t *t_dev, uint32_t v) { *t_dev = v; }
__global__ void k_bump_t(uint32_t *t_dev) { *t_dev += 1u; }

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
    __shared__ uint32_t s_run[32];
    __shared__ long long s_esum[32];
    const uint32_t nlist = *P.list_count;
    unsigned long long n_pairs = 0, n_coll = 0, n_near = 0;
    for (;;) {
        if (threadIdx.x == 0) s_item = atomicAdd(P.work, 1u);
        __syncthreads();
        const uint32_t item = s_item;
        if (item >= nlist) break;
        const uint4 ent = P.list[item];
        const uint32_t c = ent.x, lo = ent.y, n = ent.z;
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
                                            s_warp, s_esum, n_pairs, n_coll, n_near);
        __syncthreads();
        if (P.next_dt > 0.0) hist_cell_generic<1024>(P, c, lo, n, arena_E + b, s_run);
        __syncthreads();
    }
    flush_counters<1024>(P, n_pairs, n_coll, n_near);
}

}  // namespace cuba
