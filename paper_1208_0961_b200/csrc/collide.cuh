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
            const uint32_t k = shuf_word(draw(P.seed, spid[j], P.t, (uint32_t)rho >> 2, kTagShuf, 0), rho);
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

// One pair: Eq. 3 decision.  Returns hit; s (Mandelstam) through s_out.
__device__ __forceinline__ bool pair_decide(const CollideParams &P, uint32_t ida, uint32_t rho, double scale,
                                            double pax, double pay, double paz, double Ea,
                                            double pbx, double pby, double pbz, double Eb,
                                            double &s_out, double &prob_out, double &u_out)
{
    const double ee = Ea * Eb;
    const double dx = Eb * pax - Ea * pbx;
    const double dy = Eb * pay - Ea * pby;
    const double dz = Eb * paz - Ea * pbz;
    const double s = ((dx * dx + dy * dy) + dz * dz) / ee;   // (p_a+p_b)^2, A9
    const double vrel = 0.5 * (s / ee);                       // s/(2 E_a E_b)
    const double prob = vrel * scale;                         // Eq. 3 * cn/R
    const U4 w = draw(P.seed, ida, P.t, rho, kTagDec, 0);
    const double u = u53(w.x, w.y);
    s_out = s; prob_out = prob; u_out = u;
    return u < prob;
}

// Boost to the CM frame, isotropic direction, boost back (closed form A10).
__device__ __forceinline__ void pair_scatter(const CollideParams &P, uint32_t ida, uint32_t rho, double s,
                                             double pax, double pay, double paz, double Ea,
                                             double pbx, double pby, double pbz, double Eb,
                                             double q[6])
{
    double nx, ny, nz;
    draw_direction(P.seed, ida, P.t, rho, nx, ny, nz);
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

// Shared-memory classes: THREADS threads, at most THREADS*ITEMS particles, compile-time trip
// counts.  Differences to the generic routine, all invisible in the results:
//   * 2n buckets with 16-bit counters packed two per word (expected occupancy 1/2);
//   * pairs that collide are compacted into a list first, so the expensive scatter path runs
//     on full warps instead of on the ~25 % of lanes that hit in a round.
template <int THREADS, int ITEMS, bool TRACE>
__device__ __forceinline__ void collide_cell_smem(const CollideParams &P, uint32_t c, uint32_t lo, uint32_t n,
                                                  double *sp0, double *sp1, double *sp2, double *sE,
                                                  uint32_t *spid, uint32_t *skey, uint32_t *sbkt,
                                                  uint16_t *sord, uint16_t *stmp, uint32_t *s_warp,
                                                  uint32_t *s_nhit,
                                                  unsigned long long &n_pairs, unsigned long long &n_coll,
                                                  unsigned long long &n_near)
{
    const int tid = threadIdx.x, lane = tid & 31;
    const double cn = (n & 1u) ? (double)n : (double)(n - 1u);
    const double pmax = (2.0 * cn) * P.base;
    int R;
    if (!(pmax <= 64.0)) { if (tid == 0) atomicOr(P.flags, kFlagRounds); R = 64; }
    else R = (pmax <= 1.0) ? 1 : (int)ceil(pmax);
    const double scale = (cn * P.base) / (double)R;
    const uint32_t npairs = n >> 1;
    const uint32_t nb = 2u * n;
    uint16_t *sb16 = reinterpret_cast<uint16_t *>(sbkt);
    double *sS = reinterpret_cast<double *>(skey);   // Mandelstam s of the colliding pairs (skey is dead by then)
    U4 shuf[ITEMS];                                  // shuffle words of my particles: one Philox call per 4 rounds

#pragma unroll
    for (int it = 0; it < ITEMS; ++it) {
        const uint32_t j = tid + it * THREADS;
        if (j < n) {
            const double a = P.px[lo + j], b = P.py[lo + j], cc = P.pz[lo + j];
            sp0[j] = a; sp1[j] = b; sp2[j] = cc;
            sE[j] = energy(a, b, cc);
            spid[j] = P.pid[lo + j];
            sbkt[j] = 0;
        }
    }
    if (tid == 0) { sbkt[n] = 0; *s_nhit = 0; }
    __syncthreads();

    for (int rho = 0; rho < R; ++rho) {
        // (a) keys, bucket counts; the arrival slot only serves to park the element
#pragma unroll
        for (int it = 0; it < ITEMS; ++it) {
            const uint32_t j = tid + it * THREADS;
            if (j < n) {
                if ((rho & 3) == 0) shuf[it] = draw(P.seed, spid[j], P.t, (uint32_t)rho >> 2, kTagShuf, 0);
                const uint32_t k = shuf_word(shuf[it], rho);
                skey[j] = k;
                const uint32_t b = __umulhi(k, nb);
                const uint32_t sh = (b & 1u) * 16u;
                const uint32_t old = atomicAdd(&sbkt[b >> 1], 1u << sh);
                sord[j] = (uint16_t)((old >> sh) & 0xFFFFu);
            }
        }
        __syncthreads();
        // (b) exclusive scan of the 2n counters (n words), contiguous chunk of words per thread
        {
            const uint32_t chunk = (n + THREADS - 1) / THREADS;
            const uint32_t w0 = min(n, tid * chunk), w1 = min(n, w0 + chunk);
            uint32_t sum = 0;
            for (uint32_t w = w0; w < w1; ++w) { const uint32_t v = sbkt[w]; sum += (v & 0xFFFFu) + (v >> 16); }
            uint32_t total;
            uint32_t run = block_exclusive_scan<THREADS>(sum, s_warp, total);
            for (uint32_t w = w0; w < w1; ++w) {
                const uint32_t v = sbkt[w];
                const uint32_t mid = run + (v & 0xFFFFu);
                sbkt[w] = run | (mid << 16);
                run = mid + (v >> 16);
            }
            if (tid == 0) sbkt[n] = n;   // start of the sentinel bucket 2n
        }
        __syncthreads();
        // (c) park element j at its arrival slot inside its bucket
#pragma unroll
        for (int it = 0; it < ITEMS; ++it) {
            const uint32_t j = tid + it * THREADS;
            if (j < n) stmp[(uint32_t)sb16[__umulhi(skey[j], nb)] + (uint32_t)sord[j]] = (uint16_t)j;
        }
        __syncthreads();
        // (d) final rank = bucket start + number of bucket mates with a smaller (key, pid).
        // Buckets hold 1.5 elements on average (own bucket), so the first four slots are
        // compared in straight-line code on full warps; bigger buckets and equal 32-bit keys
        // (2^-32 per mate) take the loop.
#pragma unroll
        for (int it = 0; it < ITEMS; ++it) {
            const uint32_t j = tid + it * THREADS;
            if (j < n) {
                const uint32_t k = skey[j];
                const uint32_t b = __umulhi(k, nb);
                const uint32_t beg = sb16[b], cnt = (uint32_t)sb16[b + 1] - beg;
                const uint32_t last = n - 1u;
                const uint32_t k0 = skey[stmp[beg]];
                const uint32_t k1 = skey[stmp[min(beg + 1u, last)]];
                const uint32_t k2 = skey[stmp[min(beg + 2u, last)]];
                const uint32_t k3 = skey[stmp[min(beg + 3u, last)]];
                uint32_t rank = beg + (k0 < k ? 1u : 0u) + ((cnt > 1u && k1 < k) ? 1u : 0u) +
                                ((cnt > 2u && k2 < k) ? 1u : 0u) + ((cnt > 3u && k3 < k) ? 1u : 0u);
                const uint32_t same = (k0 == k ? 1u : 0u) + ((cnt > 1u && k1 == k) ? 1u : 0u) +
                                      ((cnt > 2u && k2 == k) ? 1u : 0u) + ((cnt > 3u && k3 == k) ? 1u : 0u);
                if (cnt > 4u || same > 1u) {
                    const uint32_t id = spid[j];
                    rank = beg;
                    for (uint32_t q = beg; q < beg + cnt; ++q) {
                        const uint32_t jj = stmp[q];
                        const uint32_t kk = skey[jj];
                        rank += (kk < k || (kk == k && spid[jj] < id)) ? 1u : 0u;
                    }
                }
                sord[rank] = (uint16_t)j;   // arrival slots in sord are dead after (c)
            }
        }
        __syncthreads();
        // (e1) pair order[2k] with order[2k+1]: Eq. 3 decision; colliding pairs go to a list
#pragma unroll
        for (int it = 0; it < (ITEMS + 1) / 2; ++it) {
            const uint32_t k = tid + it * THREADS;
            bool hit = false;
            double s = 0.0;
            if (k < npairs) {
                const uint32_t a = sord[2 * k], b = sord[2 * k + 1];
                const uint32_t ida = spid[a];
                double prob, u;
                hit = pair_decide(P, ida, (uint32_t)rho, scale, sp0[a], sp1[a], sp2[a], sE[a],
                                  sp0[b], sp1[b], sp2[b], sE[b], s, prob, u);
                n_pairs += 1;
                if (fabs(u - prob) <= 1e-12) n_near += 1;
                if (TRACE) {
                    const unsigned long long e = P.trace_off[c] + (unsigned long long)rho * npairs + k;
                    P.tr_cell[e] = c; P.tr_round[e] = (uint32_t)rho; P.tr_pa[e] = ida; P.tr_pb[e] = spid[b];
                    P.tr_P[e] = prob; P.tr_u[e] = u; P.tr_dec[e] = hit ? 1 : 0;
                }
            }
            const uint32_t hm = __ballot_sync(0xFFFFFFFFu, hit);
            if (hm) {
                uint32_t basep = 0;
                if (lane == 0) basep = atomicAdd(s_nhit, (uint32_t)__popc(hm));
                basep = __shfl_sync(0xFFFFFFFFu, basep, 0);
                if (hit) {
                    const uint32_t pos = basep + __popc(hm & lanemask_lt());
                    stmp[pos] = (uint16_t)k;      // stmp and skey are dead after (d)
                    sS[k] = s;
                }
            }
        }
        // the bucket counters are free from here on: clear them for the next round
#pragma unroll
        for (int it = 0; it < ITEMS; ++it) {
            const uint32_t j = tid + it * THREADS;
            if (j < n) sbkt[j] = 0;
        }
        if (tid == 0) sbkt[n] = 0;
        __syncthreads();
        // (e2) scatter the colliding pairs, densely
        const uint32_t nhit = *s_nhit;
        for (uint32_t h = tid; h < nhit; h += THREADS) {
            const uint32_t k = stmp[h];
            const uint32_t a = sord[2 * k], b = sord[2 * k + 1];
            double q[6];
            pair_scatter(P, spid[a], (uint32_t)rho, sS[k], sp0[a], sp1[a], sp2[a], sE[a],
                         sp0[b], sp1[b], sp2[b], sE[b], q);
            sp0[a] = q[0]; sp1[a] = q[1]; sp2[a] = q[2]; sE[a] = energy(q[0], q[1], q[2]);
            sp0[b] = q[3]; sp1[b] = q[4]; sp2[b] = q[5]; sE[b] = energy(q[3], q[4], q[5]);
        }
        if (tid == 0) n_coll += nhit;
        __syncthreads();
        if (tid == 0) *s_nhit = 0;
    }
#pragma unroll
    for (int it = 0; it < ITEMS; ++it) {
        const uint32_t j = tid + it * THREADS;
        if (j < n) { P.px[lo + j] = sp0[j]; P.py[lo + j] = sp1[j]; P.pz[lo + j] = sp2[j]; }
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

__device__ __forceinline__ void prefetch_l2(const void *p)
{
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// Shared-memory classes: CAP particles at most, 48 B of shared memory per particle.  The next
// work item is fetched one cell ahead and its momenta / pids are prefetched into L2 while
// the current cell is processed, so the load phase does not wait on DRAM.
template <int THREADS, int ITEMS, int CAP, int MIN_BLOCKS, bool TRACE>
__global__ void __launch_bounds__(THREADS, MIN_BLOCKS)
k_collide(CollideParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *sp0 = reinterpret_cast<double *>(smem_raw);
    double *sp1 = sp0 + CAP, *sp2 = sp1 + CAP, *sE = sp2 + CAP;
    uint32_t *spid = reinterpret_cast<uint32_t *>(sE + CAP);
    uint32_t *skey = spid + CAP;
    uint32_t *sbkt = skey + CAP;                 // CAP + 2 words = 2 CAP + 4 packed counters
    uint16_t *sord = reinterpret_cast<uint16_t *>(sbkt + CAP + 2);
    uint16_t *stmp = sord + CAP;
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_item[2];
    __shared__ uint32_t s_nhit;

    const uint32_t nlist = *P.list_count;
    unsigned long long n_pairs = 0, n_coll = 0, n_near = 0;
    if (threadIdx.x == 0) s_item[0] = atomicAdd(P.work, 1u);
    __syncthreads();
    uint32_t item = s_item[0];
    for (int it = 0; item < nlist; ++it) {
        if (threadIdx.x == 0) s_item[(it + 1) & 1] = atomicAdd(P.work, 1u);
        __syncthreads();
        const uint32_t next = s_item[(it + 1) & 1];
        if (next < nlist) {
            const uint32_t c2 = P.list[next];
            const uint32_t lo2 = P.cell_start[c2], n2 = P.cell_start[c2 + 1] - lo2;
            for (uint32_t l = threadIdx.x * 16u; l < n2 + 16u; l += THREADS * 16u) {   // one 128 B line per thread
                const uint32_t e = lo2 + min(l, n2 - 1u);
                prefetch_l2(P.px + e); prefetch_l2(P.py + e); prefetch_l2(P.pz + e);
                if ((l & 16u) == 0) prefetch_l2(P.pid + e);
            }
        }
        const uint32_t c = P.list[item];
        const uint32_t lo = P.cell_start[c], n = P.cell_start[c + 1] - lo;
        collide_cell_smem<THREADS, ITEMS, TRACE>(P, c, lo, n, sp0, sp1, sp2, sE, spid, skey, sbkt, sord,
                                                 stmp, s_warp, &s_nhit, n_pairs, n_coll, n_near);
        __syncthreads();
        item = next;
    }
    flush_counters<THREADS>(P, n_pairs, n_coll, n_near);
}

constexpr size_t collide_smem_bytes(int cap) { return (size_t)cap * 48 + 32; }

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
