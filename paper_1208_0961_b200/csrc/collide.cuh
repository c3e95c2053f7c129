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

// Per-cell constants of the fused histogram, written by thread 0 when the cell is set up.
struct HistCell {
    int i0[3];            // cell coordinates (x slowest)
    double i0d[3];        // the same as doubles
    int lo_code[3];       // per-axis direction component of a particle that leaves through the lower face:
    int hi_code[3];       //   0 / 2, or 1 where that face is a wall (elastic reflection back into the cell, A12)
};

__device__ __forceinline__ void hist_cell_setup(const Geom &g, uint32_t c, HistCell *h)
{
    h->i0[2] = (int)(c % (uint32_t)g.nc[2]);
    h->i0[1] = (int)((c / (uint32_t)g.nc[2]) % (uint32_t)g.nc[1]);
    h->i0[0] = (int)(c / ((uint32_t)g.nc[2] * (uint32_t)g.nc[1]));
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        h->i0d[k] = (double)h->i0[k];
        h->lo_code[k] = h->i0[k] == 0 ? 1 : 0;
        h->hi_code[k] = h->i0[k] == g.nc[k] - 1 ? 1 : 2;
    }
}

__device__ __forceinline__ double rcp_approx(double a)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(a));   // ~20 good bits from the upper word
    return r;
}

// One axis of the guarded estimate: t = position after the move in units of the cell edge,
// relative to the cell's lower face (the cell is [0,1)).  Away from the faces (and dt < cell edge
// means |t - 0.5| < 1.5) the direction component follows from t alone: inside -> 1; beyond the
// upper face -> 2, beyond the lower -> 0, or 1 if that face is a wall (the reflected position lies
// in the same cell).  Within kHistEps of a face -- or anything unexpected, NaN included -- the
// caller redoes the particle with the exact operation order.
constexpr double kHistEps = 1e-4;   // the estimate is good to ~1e-9; the band is generous

__device__ __forceinline__ int axis_code(double t, int lo_code, int hi_code, bool &safe)
{
    const double a = fabs(t - 0.5);
    const bool inside = a < 0.5 - kHistEps;
    const bool outside = a > 0.5 + kHistEps && a < 1.5 - kHistEps;
    safe = safe && (inside || outside);
    return inside ? 1 : (t > 0.5 ? hi_code : lo_code);
}

// Direction code of a particle: the same value as next_direction(), computed without the fp64
// division (hardware reciprocal estimate + one Newton step, fused multiply-adds) wherever the
// outcome is not within kHistEps of changing.
__device__ __forceinline__ int next_direction_guarded(const Geom &g, double dt, const HistCell &h,
                                                      double x, double y, double z, double px, double py, double pz, double E)
{
    double r = rcp_approx(E);
    r = __fma_rn(r, __fma_rn(-E, r, 1.0), r);
    const double w = dt * r;
    bool safe = true;
    const int dx = axis_code(__fma_rn(__fma_rn(px, w, x), g.inv_d[0], -h.i0d[0]), h.lo_code[0], h.hi_code[0], safe);
    const int dy = axis_code(__fma_rn(__fma_rn(py, w, y), g.inv_d[1], -h.i0d[1]), h.lo_code[1], h.hi_code[1], safe);
    const int dz = axis_code(__fma_rn(__fma_rn(pz, w, z), g.inv_d[2], -h.i0d[2]), h.lo_code[2], h.hi_code[2], safe);
    if (CUBA_FORCE_SLOW_PATHS || !safe) return next_direction(g, dt, h.i0[0], h.i0[1], h.i0[2], x, y, z, px, py, pz, E);
    return dx * 9 + dy * 3 + dz;
}

// Tile segments of a cell: the flat passes work on tiles of kTile consecutive slots; segment k of
// the cell [lo, lo+n) is its intersection with tile (lo / kTile) + k.  s_seg[k][d] counts the
// cell's particles of segment k that move in direction d.  From it:
//   cnt[d][c]              = sum over all segments                      (what K_A accumulates)
//   carry[tile T0+k][d]    = sum over segments before k, k >= 1         (what k_carry derives)
//   carry[tile T0][d]      = 0 if the cell starts exactly at the tile start
// Every tile start lies in exactly one non-empty cell, so every carry row is written once.
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
// Same results as the generic routine above, organised for issue efficiency on sm_100a:
//   * every phase works on groups of G items per thread with clamped, unguarded loads so
//     that the G Philox / fp64 chains of a thread interleave (only stores are predicated);
//   * 2n buckets with 16-bit counters packed two per word; the keys themselves are parked in
//     bucket order, so an element ranks itself from five consecutive words (no indirection)
//     and buckets with more than four elements or equal 32-bit keys take a rare slow path;
//   * the Eq. 3 decision compares u*(EaEb)^2 with |d|^2*scale/2 (no division); only a
//     decision inside a 4e-9 band around the threshold is redone with the exact operation
//     order of the oracle, so the decisions (and the near-threshold counter, A16) are the
//     oracle's bit for bit; the division for s is paid by the pairs that collide;
//   * hits are compacted per warp, and a warp scatters its own hits right away: pairs are
//     disjoint, so no block barrier separates decision and scatter;
//   * the energy of an outgoing momentum is only recomputed when another round will read it.
// Five block barriers per round.

// 53-bit uniform from two Philox words, same value as u53(): both halves are exact integers
// below 2^27 placed in the mantissa of 2^52, so every operation below is exact.
__device__ __forceinline__ double u53_bits(uint32_t w0, uint32_t w1)
{
    const double hi = __hiloint2double(0x43300000, (int)(w0 >> 5)) - 4503599627370496.0;
    const double lo = __hiloint2double(0x43300000, (int)(w1 >> 6)) - 4503599627370496.0;
    return (hi * 67108864.0 + lo) * (1.0 / 9007199254740992.0);
}

// Marsaglia disc rejection (A11) with the key schedule from the parameters.
__device__ __forceinline__ void draw_direction_k(const CollideParams &P, uint32_t t, uint32_t pid, uint32_t rho,
                                                 double &nx, double &ny, double &nz)
{
    for (uint32_t call = 0; call < 65536u; ++call) {
        const U4 w = drawk(P, t, pid, rho, kTagDir, call);
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

// Exclusive block scan with one barrier; s_warp is next written a round (several barriers) later.
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


// Rare path of the in-bucket ranking: buckets with more than four elements, or equal 32-bit
// keys (then the pid decides, A7; the keys of the other particles are recomputed).
__device__ __noinline__ uint32_t slow_rank(uint64_t seed, uint32_t t, const uint32_t *spark, const uint32_t *spid,
                                           uint32_t n, uint32_t nb, uint32_t j, uint32_t k, uint32_t beg, int rho)
{
    const uint32_t b = __umulhi(k, nb);
    uint32_t rank = beg, same = 0;
    for (uint32_t q = beg; q < n; ++q) {
        const uint32_t kk = spark[q];
        if (__umulhi(kk, nb) != b) break;
        rank += kk < k ? 1u : 0u;
        same += kk == k ? 1u : 0u;
    }
    if (CUBA_FORCE_SLOW_PATHS || same > 1u) {
        const uint32_t id = spid[j];
        for (uint32_t i = 0; i < n; ++i) {
            const uint32_t id2 = spid[i];
            if (id2 < id && shuf_word(draw(seed, id2, t, (uint32_t)rho >> 2, kTagShuf, 0), rho) == k) rank += 1u;
        }
    }
    return rank;
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

// Per-CTA statistics in shared memory: [0] pairs, [1] collisions, [2] near-threshold decisions;
// and the constants of the current cell that are only needed at a few places (kept out of
// registers across the register-hungry phases).
struct CtaStats {
    double scale, hscale;     // Eq. 3 factor cn*base/R of the current cell, and half of it
    uint32_t lo;              // first slot of the current cell
    uint32_t near;            // near-threshold decisions of this CTA (A16; rare)
    HistCell h;               // fused histogram: constants of the current cell
};

// Per-thread accumulators over all cells of a CTA, flushed once at the end of the kernel.
struct ThreadStats {
    unsigned long long pairs, rounds;   // uniform over the CTA; thread 0 flushes
    uint32_t hits;                       // uniform over a warp; lane 0 flushes
};

template <int THREADS, int ITEMS, int G, bool TRACE, bool LOCAL, bool GRAPH>
__device__ __forceinline__ void collide_cell_smem(const CollideParams &P, uint32_t c, uint32_t lo, uint32_t n,
                                                  double *sp0, double *sp1, double *sp2, double *sE,
                                                  uint32_t *spid, uint32_t *spark, uint32_t *sbkt,
                                                  uint16_t *sord, uint32_t *s_warp, CtaStats *stats,
                                                  uint32_t *s_seg, long long *s_esum, ThreadStats &acc,
                                                  uint32_t lo_next, uint32_t n_next)
{
    static_assert(ITEMS % G == 0, "items are processed in groups of G");
    constexpr int NG = ITEMS / G;
    constexpr int PITEMS = (ITEMS + 1) / 2;          // pairs per thread
    constexpr int SCAN = ITEMS | 1;                  // words per thread in the scan (odd stride: no bank conflicts)
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
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
    if (tid == 0) {
        stats->lo = lo;
        if (!local) {
            const double scale = (cn * base) / (double)R;
            stats->scale = scale; stats->hscale = 0.5 * scale;
        }
        if (hist) hist_cell_setup(P.g, c, &stats->h);
    }
    const uint32_t npairs = n >> 1, nb = 2u * n, last = n - 1u;
    uint16_t *sb16 = reinterpret_cast<uint16_t *>(sbkt);
    uint16_t *shit = reinterpret_cast<uint16_t *>(spark) + wid * (PITEMS * 32);   // this warp's hit list
    uint32_t key[ITEMS], aux[ITEMS], keep[ITEMS];

    // ---- stage the cell: momenta, energies, pids; clear the bucket counters -----------------
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
            const double e = energy(a[i], b[i], cc[i]);
            if (j < n) {
                sp0[j] = a[i]; sp1[j] = b[i]; sp2[j] = cc[i]; sE[j] = e; spid[j] = id[i]; sbkt[j] = 0;
                if (local) esum += energy_fixed(e);
            }
        }
    }
    if (hist)
        for (uint32_t e = tid; e < ((lo + n - 1u) / kTile - lo / kTile + 1u) * kDirs; e += THREADS) s_seg[e] = 0;
    if (local) block_sum_ll_post<THREADS>(esum, s_esum);
    __syncthreads();
    if (local) {
        base = local_base(block_sum_ll_read<THREADS>(s_esum), n, P.dt, P.etas);
        const double pmax = (2.0 * cn) * base;
        if (!(pmax <= 64.0)) { if (tid == 0) atomicOr(P.flags, kFlagRounds); R = 64; }
        else R = (pmax <= 1.0) ? 1 : (int)ceil(pmax);
        if (n < 2u) R = 0;
        if (tid == 0) {             // read in phase (e1), several barriers from here
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

    uint32_t warp_hits = 0;
    for (int rho = 0; rho < R; ++rho) {
        // (a) shuffle keys (A7: word rho mod 4 of the call for rounds 4*(rho div 4)..+3; one call
        // serves two rounds, the second word is kept) and bucket counts
#pragma unroll
        for (int g = 0; g < NG; ++g) {
            if ((uint32_t)(g * G * THREADS) >= n) break;
            if ((rho & 1) == 0) {
#pragma unroll
                for (int i = 0; i < G; ++i) {
                    const int it = g * G + i;
                    const uint32_t jc = min((uint32_t)(tid + it * THREADS), last);
                    const U4 w = drawk(P, tcur, spid[jc], (uint32_t)rho >> 2, kTagShuf, 0);
                    key[it] = (rho & 2) ? w.z : w.x;
                    keep[it] = (rho & 2) ? w.w : w.y;
                }
            } else {
#pragma unroll
                for (int i = 0; i < G; ++i) key[g * G + i] = keep[g * G + i];
            }
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const int it = g * G + i;
                const uint32_t j = tid + it * THREADS;
                const uint32_t b = __umulhi(key[it], nb);
                const uint32_t sh = (b & 1u) * 16u;
                aux[it] = 0;
                if (j < n) aux[it] = (atomicAdd(&sbkt[b >> 1], 1u << sh) >> sh) & 0xFFFFu;   // arrival slot
            }
        }
        __syncthreads();
        // (b) exclusive scan of the 2n counters (n words), a contiguous chunk of words per thread
        {
            const uint32_t chunk = ((n + THREADS - 1) / THREADS) | 1u;
            const uint32_t w0 = min(n, tid * chunk), w1 = min(n, w0 + chunk);
            uint32_t v[SCAN], sum = 0;
#pragma unroll
            for (int q = 0; q < SCAN; ++q) {
                v[q] = (w0 + q < w1) ? sbkt[w0 + q] : 0u;
                sum += (v[q] & 0xFFFFu) + (v[q] >> 16);
            }
            uint32_t run = block_exclusive_scan_1b<THREADS>(sum, s_warp);
#pragma unroll
            for (int q = 0; q < SCAN; ++q) {
                const uint32_t mid = run + (v[q] & 0xFFFFu);
                if (w0 + q < w1) sbkt[w0 + q] = run | (mid << 16);
                run = mid + (v[q] >> 16);
            }
        }
        __syncthreads();
        // (c) park the key at bucket start + arrival slot; four sentinels behind the last key
#pragma unroll
        for (int g = 0; g < NG; ++g) {
            if ((uint32_t)(g * G * THREADS) >= n) break;
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const int it = g * G + i;
                const uint32_t j = tid + it * THREADS;
                const uint32_t beg = sb16[__umulhi(key[it], nb)];
                if (j < n) spark[beg + aux[it]] = key[it];
                aux[it] = (j < n) ? beg : 0u;
            }
        }
        if (tid < 4) spark[n + tid] = 0xFFFFFFFFu;
        __syncthreads();
        // (d) rank = bucket start + number of bucket mates with a smaller key.  Keys beyond the
        // bucket are larger (the bucket index is monotone in the key), so four words decide a
        // bucket of up to four; the fifth tells whether the bucket is bigger.
#pragma unroll
        for (int g = 0; g < NG; ++g) {
            if ((uint32_t)(g * G * THREADS) >= n) break;
            uint32_t rank[G];
            bool slow[G];
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const int it = g * G + i;
                const uint32_t k = key[it], beg = aux[it];
                const uint32_t k0 = spark[beg], k1 = spark[beg + 1], k2 = spark[beg + 2], k3 = spark[beg + 3],
                               k4 = spark[beg + 4];
                rank[i] = beg + (k0 < k ? 1u : 0u) + (k1 < k ? 1u : 0u) + (k2 < k ? 1u : 0u) + (k3 < k ? 1u : 0u);
                const uint32_t same = (k0 == k ? 1u : 0u) + (k1 == k ? 1u : 0u) + (k2 == k ? 1u : 0u) + (k3 == k ? 1u : 0u);
                slow[i] = (tid + it * THREADS < n) &&
                          (CUBA_FORCE_SLOW_PATHS || same != 1u || __umulhi(k4, nb) == __umulhi(k, nb));
            }
            bool any = false;
#pragma unroll
            for (int i = 0; i < G; ++i) any = any || slow[i];
            if (any) {
#pragma unroll
                for (int i = 0; i < G; ++i)
                    if (slow[i]) rank[i] = slow_rank(P.seed, tcur, spark, spid, n, nb, tid + (g * G + i) * THREADS,
                                                     key[g * G + i], aux[g * G + i], rho);
            }
#pragma unroll
            for (int i = 0; i < G; ++i) {
                const uint32_t j = tid + (g * G + i) * THREADS;
                if (j < n) {
                    sord[rank[i]] = (uint16_t)j;
                    sbkt[j] = 0;                 // the counters are free: clear them for the next round
                }
            }
        }
        __syncthreads();
        // (e1) pair order[2k] with order[2k+1]: Eq. 3 decision; this warp's hits go to its list
        uint32_t nh = 0;
        {
            const double scale = *reinterpret_cast<volatile double *>(&stats->scale);
            const double hscale = *reinterpret_cast<volatile double *>(&stats->hscale);
            double dd[PITEMS], ee[PITEMS], u[PITEMS];
            uint32_t ida[PITEMS];
#pragma unroll
            for (int it = 0; it < PITEMS; ++it) {
                const uint32_t kc = min((uint32_t)(tid + it * THREADS), npairs - 1u);
                const uint32_t ab = *reinterpret_cast<const uint32_t *>(sord + 2 * kc);
                const uint32_t a = ab & 0xFFFFu, b = ab >> 16;
                const double Ea = sE[a], Eb = sE[b];
                const double dx = Eb * sp0[a] - Ea * sp0[b];
                const double dy = Eb * sp1[a] - Ea * sp1[b];
                const double dz = Eb * sp2[a] - Ea * sp2[b];
                ida[it] = spid[a];
                ee[it] = Ea * Eb;
                dd[it] = (dx * dx + dy * dy) + dz * dz;
            }
#pragma unroll
            for (int it = 0; it < PITEMS; ++it) {
                const U4 w = drawk(P, tcur, ida[it], (uint32_t)rho, kTagDec, 0);
                u[it] = u53_bits(w.x, w.y);
            }
#pragma unroll
            for (int it = 0; it < PITEMS; ++it) {
                const uint32_t k = tid + it * THREADS;
                bool hit;
                if (TRACE) {
                    const double s = dd[it] / ee[it];         // (p_a+p_b)^2, A9
                    const double vrel = 0.5 * (s / ee[it]);   // s/(2 E_a E_b)
                    const double prob = vrel * scale;         // Eq. 3 * cn/R
                    hit = u[it] < prob;
                    if (k < npairs) {
                        if (fabs(u[it] - prob) <= 1e-12) atomicAdd(&stats->near, 1u);
                        const uint32_t ab = *reinterpret_cast<const uint32_t *>(sord + 2 * k);
                        const unsigned long long e = P.trace_off[c] + (unsigned long long)rho * npairs + k;
                        P.tr_cell[e] = c; P.tr_round[e] = (uint32_t)rho; P.tr_pa[e] = ida[it]; P.tr_pb[e] = spid[ab >> 16];
                        P.tr_P[e] = prob; P.tr_u[e] = u[it]; P.tr_dec[e] = hit ? 1 : 0;
                    }
                } else {
                    // sign(u - P) from u*(EaEb)^2 - |d|^2*scale/2; the exact form only inside a band
                    // far wider than the rounding error (it also catches NaN, inf and underflow)
                    const double ee2 = ee[it] * ee[it];
                    const double diff = u[it] * ee2 - dd[it] * hscale;
                    hit = diff < 0.0;
                    if (CUBA_FORCE_SLOW_PATHS || !(fabs(diff) > 4e-9 * ee2) || !(ee2 > 1e-280)) {
                        const uint32_t r = exact_decision(dd[it], ee[it], u[it], scale);
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
        // (e2) scatter this warp's colliding pairs, densely
        for (uint32_t h = lane; h < nh; h += 32) {
            const uint32_t k = shit[h];
            const uint32_t ab = *reinterpret_cast<const uint32_t *>(sord + 2 * k);
            const uint32_t a = ab & 0xFFFFu, b = ab >> 16;
            const double pax = sp0[a], pay = sp1[a], paz = sp2[a], Ea = sE[a];
            const double pbx = sp0[b], pby = sp1[b], pbz = sp2[b], Eb = sE[b];
            const double ee = Ea * Eb;
            const double dx = Eb * pax - Ea * pbx;
            const double dy = Eb * pay - Ea * pby;
            const double dz = Eb * paz - Ea * pbz;
            const double s = ((dx * dx + dy * dy) + dz * dz) / ee;
            double q[6];
            pair_scatter(P, tcur, spid[a], (uint32_t)rho, s, pax, pay, paz, Ea, pbx, pby, pbz, Eb, q);
            sp0[a] = q[0]; sp1[a] = q[1]; sp2[a] = q[2];
            sp0[b] = q[3]; sp1[b] = q[4]; sp2[b] = q[5];
            if (rho + 1 < R || hist) { sE[a] = energy(q[0], q[1], q[2]); sE[b] = energy(q[3], q[4], q[5]); }
        }
        warp_hits += nh;
        __syncwarp();   // the hit list is rewritten in the next round
    }
    __syncthreads();
    const uint32_t lo_w = *reinterpret_cast<volatile uint32_t *>(&stats->lo);
    // positions for the fused histogram: all loads of a thread in flight before anything waits on them
#ifndef CUBA_HB6
#define CUBA_HB6 2
#endif
    constexpr int HB = (ITEMS == 6) ? CUBA_HB6 : ((ITEMS % 2 == 0) ? 2 : 1);
    double xx[HB], yy[HB], zz[HB];
    if (hist && HB == ITEMS) {
#pragma unroll
        for (int it = 0; it < HB; ++it) {
            const uint32_t jc = lo_w + min((uint32_t)(tid + it * THREADS), last);
            xx[it] = P.x[jc]; yy[it] = P.y[jc]; zz[it] = P.z[jc];
        }
    }
#pragma unroll
    for (int g = 0; g < NG; ++g) {
        if ((uint32_t)(g * G * THREADS) >= n) break;
#pragma unroll
        for (int i = 0; i < G; ++i) {
            const uint32_t j = tid + (g * G + i) * THREADS;
            if (j < n) { P.px[lo_w + j] = sp0[j]; P.py[lo_w + j] = sp1[j]; P.pz[lo_w + j] = sp2[j]; }
        }
    }
    acc.hits += warp_hits;
    acc.pairs += (unsigned long long)R * npairs;
    acc.rounds += (unsigned long long)R;

    // ---- fused histogram of the next step (S1-S3 of step t+1 on the final momenta) ----------
    if (hist) {
        const uint32_t T0 = lo_w / kTile;
        const HistCell &hc = stats->h;
#pragma unroll
        for (int g = 0; g < ITEMS / HB; ++g) {
            if ((uint32_t)(g * HB * THREADS) >= n) break;
            if (HB != ITEMS) {
#pragma unroll
                for (int i = 0; i < HB; ++i) {
                    const uint32_t jc = lo_w + min((uint32_t)(tid + (g * HB + i) * THREADS), last);
                    xx[i] = P.x[jc]; yy[i] = P.y[jc]; zz[i] = P.z[jc];
                }
            }
#pragma unroll
            for (int i = 0; i < HB; ++i) {
                const uint32_t j = tid + (g * HB + i) * THREADS, jj = min(j, last);
                const int d = next_direction_guarded(P.g, P.next_dt, hc, xx[i], yy[i], zz[i],
                                                     sp0[jj], sp1[jj], sp2[jj], sE[jj]);
                const bool valid = j < n;
                if (valid && d < 0) atomicOr(P.flags, kFlagMoved);
                const uint32_t key = ((lo_w + jj) / kTile - T0) * kDirs + (uint32_t)max(d, 0);
                const uint32_t active = __ballot_sync(0xFFFFFFFFu, valid);
                if (valid) {
                    const uint32_t peers = __match_any_sync(active, key);
                    if ((peers & lanemask_lt()) == 0) atomicAdd(&s_seg[key], (uint32_t)__popc(peers));
                }
            }
        }
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

// Shared-memory classes: CAP particles at most, 46 B of shared memory per particle.  The next
// work item is fetched one cell ahead and its momenta / pids are prefetched into L2 while
// the current cell is processed, so the load phase does not wait on DRAM.
template <int THREADS, int ITEMS, int CAP, int MIN_BLOCKS, bool TRACE, bool LOCAL, bool GRAPH>
__global__ void __launch_bounds__(THREADS, MIN_BLOCKS)
k_collide(CollideParams P)
{
    static_assert(CAP <= THREADS * ITEMS && CAP < 65536, "class capacity");
#ifndef CUBA_G6
#define CUBA_G6 3
#endif
    constexpr int G = (ITEMS == 6) ? CUBA_G6 : ((ITEMS % 2 == 0) ? 2 : ITEMS);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *sp0 = reinterpret_cast<double *>(smem_raw);
    double *sp1 = sp0 + CAP, *sp2 = sp1 + CAP, *sE = sp2 + CAP;
    uint32_t *spid = reinterpret_cast<uint32_t *>(sE + CAP);
    uint32_t *spark = spid + CAP;                // CAP keys + 4 sentinels (+ pad); hit lists between (d) and (c)
    uint32_t *sbkt = spark + CAP + 8;            // CAP words = 2 CAP packed 16-bit counters
    uint16_t *sord = reinterpret_cast<uint16_t *>(sbkt + CAP + 8);
    __shared__ uint32_t s_warp[32];
    __shared__ CtaStats s_stats;
    __shared__ uint32_t s_seg[((CAP + kTile - 2) / kTile + 1) * kDirs];   // a cell of CAP particles spans at most this many tiles
    __shared__ long long s_esum[32];

    // Dynamic work distribution, claimed one cell ahead so that the next cell can be prefetched
    // into L2.  (Measured alternatives, both slower because they lengthen the tail of the list:
    // a static round-robin, +0.10 ms at configs[2]; claiming three cells ahead, +0.09 ms.)
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
        if (item < nlist) nxt = P.list[item];   // first used after the staging barrier
        collide_cell_smem<THREADS, ITEMS, G, TRACE, LOCAL, GRAPH>(P, cur.x, cur.y, cur.z, sp0, sp1, sp2, sE, spid, spark, sbkt, sord,
                                                    s_warp, &s_stats, s_seg, s_esum, acc, nxt.y, nxt.z);
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

// step index in device memory for graph replays
__global__ void k_set_t(uint32_t *t_dev, uint32_t v) { *t_dev = v; }
__global__ void k_bump_t(uint32_t *t_dev) { *t_dev += 1u; }

constexpr size_t collide_smem_bytes(int cap) { return (size_t)cap * 46 + 64; }

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
