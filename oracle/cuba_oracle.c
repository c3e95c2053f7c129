/*
 * cuba_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded CPU statement of the per-timestep particle-in-cell
 * Boltzmann step of CuBA/BAMPS (arXiv:1208.0961; /root/reference/PAPER.md), written from
 * the paper step by step in the paper's order.  It shares no code, header, table or helper
 * with the CUDA library in paper_1208_0961_b200/ and neither imports the other.  Only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call it.
 *
 * Build:  gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (see oracle/__init__.py).
 * -ffp-contract=off is part of the arithmetic contract (reading A2): every
 * written + - * / sqrt rounds once, in the written order, no fused multiply-add.
 *
 * Passages followed (PAPER.md line : what):
 *   32      PIC: volume divided into cells V_cell = dx dy dz, each particle has r and p
 *   34-36   Eq. 2  x -> x + c^2 p_x/E dt (same for y, z)                       -> S1
 *   38      collisions are binary, only between particles in the same cell    -> S3-S5
 *   40      Eq. 3  P22 = v_rel (sigma/N_test) (dt/V_cell)                     -> S5
 *   42      v_rel = s/(2 E1 E2), s = (p1+p2)^2, sigma isotropic               -> S5
 *   44      testparticles (P22 reduced by r_test); boost to CM, choose the momentum
 *           randomly, boost back; elastic reflection off the six walls        -> S2, S5
 *   66      total energy is conserved                                         -> observables
 *   62-72   energy density / flow of the Riemann problem, viscosity            -> LRF observables
 *   98      "implement the parameter dt as variable"                           -> oracle_step_adaptive
 *   80,108  "local cross section" / constant eta/s of ref. [1]                 -> oracle_step_etas
 * Where the paper is silent (pair enumeration, shuffle, RNG, order inside a step, odd
 * cells, P > 1) the readings A1..A19 of DESIGN.md are followed; each is named at its use.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Philox vs cuRAND's host generator;
 * wall reflection |p| preservation and hand-built mirror cases; per-collision
 * four-momentum conservation and agreement with an explicit 4x4 Lorentz-matrix boost;
 * run-level energy conservation; collision rate vs the closed form; isotropy (KS);
 * thermal box stays Boltzmann (KS); initial energy density 3nT; free-streaming Riemann
 * closed form; counting sort vs brute force; pairing uniform over perfect matchings;
 * Landau matching vs numpy's eigen-decomposition, hand-built slabs, tracelessness, and a
 * boosted thermal ensemble (e = 3 n T, v = beta); variable dt: reduces to the fixed step where
 * the rule does not bind, keeps every traced probability <= 1 without extra rounds, and leaves the
 * collision rate per unit time at the closed form; local cross section: traced probabilities
 * against Eq. 3 assembled with math.fsum, collision rate per particle 0.3 T/(hbarc eta/s)
 * independent of the density, independence of the array order.
 * Parity unpinned: the paper's Fig. 2-4 curves and the BAMPS overlay (images and BAMPS
 * are not available).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define TAG_SHUF 0u
#define TAG_DEC 1u
#define TAG_DIR 2u
#define R_CAP 64          /* DESIGN.md A6: more rounds than this is an error */
#define DIR_CALL_CAP 65536 /* sub index is 16 bits wide (A11) */

#define ORC_OK 0
#define ORC_ERR_ARG (-1)
#define ORC_ERR_ROUNDS (-9)
#define ORC_ERR_STATE (-6)
#define ORC_ERR_CFL (-7)

/* ------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), the counter-based generator
 * north_star prescribes ("counter-based Philox streams keyed by (seed, step,
 * particle/pair id)").  Ten rounds; each round multiplies counter words 0 and 2 by two
 * fixed odd constants, keeps high and low halves, mixes in the key; the key is bumped by
 * the two Weyl constants between rounds.
 * ---------------------------------------------------------------------------------- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t prod0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t prod1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(prod0 >> 32), lo0 = (uint32_t)prod0;
        uint32_t hi1 = (uint32_t)(prod1 >> 32), lo1 = (uint32_t)prod1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* The method's stream layout ("RNG"): key = seed (low, high word); counter =
 * {particle id, global step t, round rho, tag<<16 | sub}.  Every (id,t,rho,tag,sub) is
 * used at most once. */
static void draw(uint64_t seed, uint32_t id, uint32_t t, uint32_t rho, uint32_t tag,
                 uint32_t sub, uint32_t w[4])
{
    uint32_t ctr[4] = { id, t, rho, (tag << 16) | sub };
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    oracle_philox4x32_10(ctr, key, w);
}

/* 53-bit uniform in [0,1): 27 high bits of w0 and 26 high bits of w1 (exact in fp64). */
double oracle_u53(uint32_t w0, uint32_t w1)
{
    return ((double)(w0 >> 5) * 67108864.0 + (double)(w1 >> 6)) * (1.0 / 9007199254740992.0);
}

/* E = |p| for a massless gluon (north_star: "massless gluons E=|p|"). */
static double energy(double px, double py, double pz)
{
    return sqrt((px * px + py * py) + pz * pz);
}

/* ------------------------------------------------------------------------------------
 * S1 free streaming, Eq. 2 with c = 1:  x -> x + (p_x/E) dt, same for y, z.
 * S2 wall reflection, "elastically reflected": walls at 0 and L (A12); the
 * position is mirrored and the normal momentum component negated, so |p| keeps its bits.
 * wall_dp (optional) accumulates the momentum the walls hand to the gas, sum of -2 p_k.
 * ---------------------------------------------------------------------------------- */
static void reflect_axis(double *x, double *p, double L, double *wall_dp)
{
    if (*x < 0.0) {
        *x = -*x;
        if (wall_dp) *wall_dp += -2.0 * *p;
        *p = -*p;
    } else if (*x > L) {
        *x = 2.0 * L - *x;
        if (wall_dp) *wall_dp += -2.0 * *p;
        *p = -*p;
    }
}

void oracle_stream_reflect(int64_t n, double *x, double *y, double *z,
                           double *px, double *py, double *pz,
                           double dt, const double box[3], double wall_dp[3])
{
    for (int64_t i = 0; i < n; ++i) {
        double E = energy(px[i], py[i], pz[i]);
        double w = dt / E;
        x[i] = x[i] + px[i] * w;
        y[i] = y[i] + py[i] * w;
        z[i] = z[i] + pz[i] * w;
        reflect_axis(&x[i], &px[i], box[0], wall_dp ? &wall_dp[0] : 0);
        reflect_axis(&y[i], &py[i], box[1], wall_dp ? &wall_dp[1] : 0);
        reflect_axis(&z[i], &pz[i], box[2], wall_dp ? &wall_dp[2] : 0);
    }
}

/* ------------------------------------------------------------------------------------
 * S3 cell index, PAPER.md:32 (cells of volume dx dy dz): ix = min(int(x/dx), nx-1) with
 * 1/dx precomputed; c = (ix*ny + iy)*nz + iz, x slowest.  x == L is legal after a
 * reflection and is clamped into the last cell (A12).
 * ---------------------------------------------------------------------------------- */
static uint32_t axis_index(double x, double inv_d, int ncell)
{
    int i = (int)(x * inv_d);
    if (i > ncell - 1) i = ncell - 1;
    if (i < 0) i = 0; /* unreachable for validated input; keeps the index in range */
    return (uint32_t)i;
}

void oracle_cell_index(int64_t n, const double *x, const double *y, const double *z,
                       const double box[3], const int ncell[3], uint32_t *cell)
{
    double inv_dx = 1.0 / (box[0] / (double)ncell[0]);
    double inv_dy = 1.0 / (box[1] / (double)ncell[1]);
    double inv_dz = 1.0 / (box[2] / (double)ncell[2]);
    for (int64_t i = 0; i < n; ++i) {
        uint32_t ix = axis_index(x[i], inv_dx, ncell[0]);
        uint32_t iy = axis_index(y[i], inv_dy, ncell[1]);
        uint32_t iz = axis_index(z[i], inv_dz, ncell[2]);
        cell[i] = (ix * (uint32_t)ncell[1] + iy) * (uint32_t)ncell[2] + iz;
    }
}

/* ------------------------------------------------------------------------------------
 * S4 stable counting sort by cell (north_star: "cell binning by stable counting sort"):
 * count, exclusive scan, place in ascending previous index (A8).  perm[k] = previous
 * index of the particle now at k; cell_start has ncells+1 entries.
 * ---------------------------------------------------------------------------------- */
void oracle_counting_sort(int64_t n, int64_t ncells, const uint32_t *cell,
                          uint32_t *cell_start, int64_t *perm)
{
    int64_t *cursor = (int64_t *)calloc((size_t)ncells + 1, sizeof(int64_t));
    for (int64_t i = 0; i < n; ++i) cursor[cell[i]] += 1;
    int64_t run = 0;
    for (int64_t c = 0; c < ncells; ++c) {
        int64_t cnt = cursor[c];
        cell_start[c] = (uint32_t)run;
        cursor[c] = run;
        run += cnt;
    }
    cell_start[ncells] = (uint32_t)run;
    for (int64_t i = 0; i < n; ++i) perm[cursor[cell[i]]++] = i;
    free(cursor);
}

/* ------------------------------------------------------------------------------------
 * Pair kinematics: s = (p1+p2)^2, v_rel = s/(2 E1 E2).  Reading A9: for
 * massless on-shell momenta s = |E_b p_a - E_a p_b|^2/(E_a E_b), a sum of squares (never
 * negative, accurate for near-collinear pairs).
 * ---------------------------------------------------------------------------------- */
void oracle_pair_kinematics(const double pa[3], const double pb[3],
                            double *Ea_out, double *Eb_out, double *s_out, double *vrel_out)
{
    double Ea = energy(pa[0], pa[1], pa[2]);
    double Eb = energy(pb[0], pb[1], pb[2]);
    double ee = Ea * Eb;
    double dx = Eb * pa[0] - Ea * pb[0];
    double dy = Eb * pa[1] - Ea * pb[1];
    double dz = Eb * pa[2] - Ea * pb[2];
    double s = ((dx * dx + dy * dy) + dz * dz) / ee;
    double vrel = 0.5 * (s / ee);
    *Ea_out = Ea; *Eb_out = Eb; *s_out = s; *vrel_out = vrel;
}

/* Isotropic direction in the CM frame, "choose the momentum randomly",
 * PAPER.md:42 sigma "isotropic".  Reading A11: Marsaglia's disc rejection, strict q < 1,
 * words (W0,W1) of call m>>1 for even attempts m and (W2,W3) for odd ones.
 * Returns the number of attempts used. */
int oracle_direction(uint64_t seed, uint32_t pid, uint32_t t, uint32_t rho, double nhat[3])
{
    for (int m = 0; m < 2 * DIR_CALL_CAP; ++m) {
        uint32_t w[4];
        draw(seed, pid, t, rho, TAG_DIR, (uint32_t)(m >> 1), w);
        uint32_t wa = (m & 1) ? w[2] : w[0];
        uint32_t wb = (m & 1) ? w[3] : w[1];
        double a = ((double)wa + 0.5) * (1.0 / 2147483648.0) - 1.0;
        double b = ((double)wb + 0.5) * (1.0 / 2147483648.0) - 1.0;
        double q = a * a + b * b;
        if (q < 1.0) {
            double h = sqrt(1.0 - q);
            nhat[0] = (2.0 * a) * h;
            nhat[1] = (2.0 * b) * h;
            nhat[2] = 1.0 - 2.0 * q;
            return m + 1;
        }
    }
    nhat[0] = 0.0; nhat[1] = 0.0; nhat[2] = 1.0; /* probability (1-pi/4)^131072: never */
    return 2 * DIR_CALL_CAP;
}

/* Boost to the CM frame, new direction, boost back.  Reading A10: for an
 * isotropic cross section only sqrt(s) and the boost back matter; with gamma = E_t/sqrt(s)
 * and gamma*beta = P/sqrt(s) the boost of (sqrt(s)/2)(1, +-n) closes to
 *   p'_{a,b} = 1/2 [ +-sqrt(s) n + P (1 +- (P.n)/(E_t + sqrt(s))) ]. */
void oracle_scatter(const double pa[3], const double pb[3], double Ea, double Eb, double s,
                    const double nhat[3], double pa_new[3], double pb_new[3])
{
    double rs = sqrt(s);
    double Pvx = pa[0] + pb[0], Pvy = pa[1] + pb[1], Pvz = pa[2] + pb[2];
    double Et = Ea + Eb;
    double Pn = (Pvx * nhat[0] + Pvy * nhat[1]) + Pvz * nhat[2];
    double al = Pn / (Et + rs);
    double f1 = 1.0 + al;
    double f2 = 1.0 - al;
    pa_new[0] = 0.5 * (rs * nhat[0] + Pvx * f1);
    pa_new[1] = 0.5 * (rs * nhat[1] + Pvy * f1);
    pa_new[2] = 0.5 * (rs * nhat[2] + Pvz * f1);
    pb_new[0] = 0.5 * (Pvx * f2 - rs * nhat[0]);
    pb_new[1] = 0.5 * (Pvy * f2 - rs * nhat[1]);
    pb_new[2] = 0.5 * (Pvz * f2 - rs * nhat[2]);
}

/* ------------------------------------------------------------------------------------
 * State of a run.
 * ---------------------------------------------------------------------------------- */
typedef struct {
    uint32_t cell, round, pid_a, pid_b;
    double P, u;
    uint8_t decided;
} pair_rec;

typedef struct oracle_state {
    int64_t n, ncells;
    double box[3];
    int ncell[3];
    double n_test;
    uint64_t seed;
    uint32_t t; /* global step index: the only RNG state */
    double *x, *y, *z, *px, *py, *pz;
    uint32_t *pid;
    uint32_t *cell;       /* cell of each slot after the last binning */
    uint32_t *cell_start; /* ncells + 1 */
    /* counters */
    uint64_t steps, pairs, collisions, rounds, near_threshold, dir_attempts;
    uint32_t max_occupancy;
    double wall_dp[3];
    /* trace of the last step (when enabled) */
    int trace_on;
    pair_rec *trace;
    int64_t trace_len, trace_cap;
    /* per-collision log of (n_z, phi-free) direction cosines for the isotropy pin */
    int dirlog_on;
    double *dirlog; /* 3 doubles per collision */
    int64_t dirlog_len, dirlog_cap;
} oracle_state;

static void bin_and_sort(oracle_state *st)
{
    int64_t n = st->n;
    oracle_cell_index(n, st->x, st->y, st->z, st->box, st->ncell, st->cell);
    int64_t *perm = (int64_t *)malloc((size_t)n * sizeof(int64_t));
    oracle_counting_sort(n, st->ncells, st->cell, st->cell_start, perm);
    double *tmp = (double *)malloc((size_t)n * sizeof(double));
    double *cols[6] = { st->x, st->y, st->z, st->px, st->py, st->pz };
    for (int k = 0; k < 6; ++k) {
        for (int64_t j = 0; j < n; ++j) tmp[j] = cols[k][perm[j]];
        memcpy(cols[k], tmp, (size_t)n * sizeof(double));
    }
    uint32_t *tmpu = (uint32_t *)tmp;
    for (int64_t j = 0; j < n; ++j) tmpu[j] = st->pid[perm[j]];
    memcpy(st->pid, tmpu, (size_t)n * sizeof(uint32_t));
    for (int64_t j = 0; j < n; ++j) tmpu[j] = st->cell[perm[j]];
    memcpy(st->cell, tmpu, (size_t)n * sizeof(uint32_t));
    free(tmp);
    free(perm);
}

/* cuba_init's counterpart.  Copies the caller's arrays, assigns the persistent ids
 * pid[i] = i, validates (positions inside [0,L], momenta finite, |p| > 0) and bins the
 * initial positions with S3 + S4 (reading A19: the state is cell-sorted from the start). */
oracle_state *oracle_init(const double box[3], const int ncell[3], int64_t n,
                          const double *x, const double *y, const double *z,
                          const double *px, const double *py, const double *pz,
                          double n_test, uint64_t seed, int *err)
{
    *err = ORC_ERR_ARG;
    if (n < 1 || n >= ((int64_t)1 << 32) || !(n_test > 0.0)) return 0;
    for (int k = 0; k < 3; ++k)
        if (!(box[k] > 0.0) || ncell[k] < 1) return 0;
    int64_t ncells = (int64_t)ncell[0] * ncell[1] * ncell[2];
    if (ncells >= ((int64_t)1 << 27)) return 0;
    for (int64_t i = 0; i < n; ++i) {
        double E = energy(px[i], py[i], pz[i]);
        if (!(x[i] >= 0.0 && x[i] <= box[0] && y[i] >= 0.0 && y[i] <= box[1] &&
              z[i] >= 0.0 && z[i] <= box[2]) || !(E > 0.0) || !isfinite(E)) {
            *err = ORC_ERR_STATE;
            return 0;
        }
    }
    oracle_state *st = (oracle_state *)calloc(1, sizeof(oracle_state));
    st->n = n; st->ncells = ncells; st->n_test = n_test; st->seed = seed; st->t = 0;
    for (int k = 0; k < 3; ++k) { st->box[k] = box[k]; st->ncell[k] = ncell[k]; }
    size_t bytes = (size_t)n * sizeof(double);
    st->x = (double *)malloc(bytes); memcpy(st->x, x, bytes);
    st->y = (double *)malloc(bytes); memcpy(st->y, y, bytes);
    st->z = (double *)malloc(bytes); memcpy(st->z, z, bytes);
    st->px = (double *)malloc(bytes); memcpy(st->px, px, bytes);
    st->py = (double *)malloc(bytes); memcpy(st->py, py, bytes);
    st->pz = (double *)malloc(bytes); memcpy(st->pz, pz, bytes);
    st->pid = (uint32_t *)malloc((size_t)n * sizeof(uint32_t));
    st->cell = (uint32_t *)malloc((size_t)n * sizeof(uint32_t));
    st->cell_start = (uint32_t *)malloc(((size_t)ncells + 1) * sizeof(uint32_t));
    for (int64_t i = 0; i < n; ++i) st->pid[i] = (uint32_t)i;
    bin_and_sort(st);
    *err = ORC_OK;
    return st;
}

void oracle_destroy(oracle_state *st)
{
    if (!st) return;
    free(st->x); free(st->y); free(st->z); free(st->px); free(st->py); free(st->pz);
    free(st->pid); free(st->cell); free(st->cell_start); free(st->trace); free(st->dirlog);
    free(st);
}

void oracle_set_trace(oracle_state *st, int on) { st->trace_on = on; }
void oracle_set_dirlog(oracle_state *st, int on) { st->dirlog_on = on; }

static void trace_push(oracle_state *st, pair_rec r)
{
    if (st->trace_len == st->trace_cap) {
        st->trace_cap = st->trace_cap ? 2 * st->trace_cap : 4096;
        st->trace = (pair_rec *)realloc(st->trace, (size_t)st->trace_cap * sizeof(pair_rec));
    }
    st->trace[st->trace_len++] = r;
}

static void dirlog_push(oracle_state *st, const double nhat[3])
{
    if (st->dirlog_len == st->dirlog_cap) {
        st->dirlog_cap = st->dirlog_cap ? 2 * st->dirlog_cap : 4096;
        st->dirlog = (double *)realloc(st->dirlog, (size_t)st->dirlog_cap * 3 * sizeof(double));
    }
    memcpy(st->dirlog + 3 * st->dirlog_len, nhat, 3 * sizeof(double));
    st->dirlog_len++;
}

typedef struct { uint64_t key; int64_t slot; } shuf_item;

static int cmp_shuf(const void *a, const void *b)
{
    uint64_t ka = ((const shuf_item *)a)->key, kb = ((const shuf_item *)b)->key;
    return (ka > kb) - (ka < kb);
}

/* ------------------------------------------------------------------------------------
 * S5 collisions inside one cell holding slots [lo, hi).
 *   - pairs: A4/A7 per round, order the cell by the key (a Philox word keyed by the
 *     persistent pid: word rho mod 4 of the call with counter {pid, t, rho div 4, SHUF})
 *     << 32 | pid and pair order[2k] with order[2k+1];
 *   - P22 of Eq. 3 scaled by cn = n(n-1)/(2 floor(n/2)) so that floor(n/2) tested pairs
 *     carry the rate of all n(n-1)/2 pairs (north_star "(n_cell-1)"; A5 for odd n);
 *   - A6: if the largest possible scaled P (v_rel <= 2) exceeds 1, split the step into R
 *     rounds, each with a fresh shuffle and P/R.
 * Returns ORC_OK or ORC_ERR_ROUNDS.
 * ---------------------------------------------------------------------------------- */
static int collide_cell(oracle_state *st, uint32_t c, int64_t lo, int64_t hi, double base)
{
    int64_t n = hi - lo;
    if (n < 2) return ORC_OK;
    double cn = (n & 1) ? (double)n : (double)(n - 1);
    double pmax = (2.0 * cn) * base;
    if (!(pmax <= (double)R_CAP)) return ORC_ERR_ROUNDS;
    int R = (pmax <= 1.0) ? 1 : (int)ceil(pmax);
    double scale = (cn * base) / (double)R;
    shuf_item *order = (shuf_item *)malloc((size_t)n * sizeof(shuf_item));
    st->rounds += (uint64_t)R;
    for (int rho = 0; rho < R; ++rho) {
        for (int64_t j = 0; j < n; ++j) {
            uint32_t w[4];
            draw(st->seed, st->pid[lo + j], st->t, (uint32_t)rho >> 2, TAG_SHUF, 0, w);
            order[j].key = ((uint64_t)w[rho & 3] << 32) | (uint64_t)st->pid[lo + j];
            order[j].slot = lo + j;
        }
        qsort(order, (size_t)n, sizeof(shuf_item), cmp_shuf); /* keys are unique (pid is) */
        for (int64_t k = 0; k < n / 2; ++k) {
            int64_t a = order[2 * k].slot, b = order[2 * k + 1].slot;
            double pa[3] = { st->px[a], st->py[a], st->pz[a] };
            double pb[3] = { st->px[b], st->py[b], st->pz[b] };
            double Ea, Eb, s, vrel;
            oracle_pair_kinematics(pa, pb, &Ea, &Eb, &s, &vrel);
            double P = vrel * scale;
            uint32_t w[4];
            draw(st->seed, st->pid[a], st->t, (uint32_t)rho, TAG_DEC, 0, w);
            double u = oracle_u53(w[0], w[1]);
            int hit = (u < P);
            st->pairs += 1;
            if (fabs(u - P) <= 1e-12) st->near_threshold += 1; /* A16 */
            if (st->trace_on) {
                pair_rec r = { c, (uint32_t)rho, st->pid[a], st->pid[b], P, u, (uint8_t)hit };
                trace_push(st, r);
            }
            if (hit) {
                double nhat[3], qa[3], qb[3];
                st->dir_attempts += (uint64_t)oracle_direction(st->seed, st->pid[a], st->t,
                                                               (uint32_t)rho, nhat);
                oracle_scatter(pa, pb, Ea, Eb, s, nhat, qa, qb);
                st->px[a] = qa[0]; st->py[a] = qa[1]; st->pz[a] = qa[2];
                st->px[b] = qb[0]; st->py[b] = qb[1]; st->pz[b] = qb[2];
                st->collisions += 1;
                if (st->dirlog_on) dirlog_push(st, nhat);
            }
        }
    }
    free(order);
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------
 * S5 on selected cells of a caller-supplied, cell-sorted state: an entry point
 * to collide_cell() above for parity checks at sizes where only some cells can be re-collided
 * (tests/test_gpu_large.py).  pid/px/py/pz are whole arrays in array order; cell k of the
 * selection holds slots [lo[k], hi[k]) and is collided in place with step index t and the Eq. 3
 * factor `base`.  counters (may be NULL) receives {pairs, collisions, rounds}.  No arithmetic of
 * its own.
 * ---------------------------------------------------------------------------------- */
int oracle_collide_cells(uint64_t seed, uint32_t t, double base, int64_t ncell_sel,
                         const int64_t *lo, const int64_t *hi, const uint32_t *cell_id,
                         uint32_t *pid, double *px, double *py, double *pz, uint64_t counters[3])
{
    oracle_state st;
    memset(&st, 0, sizeof(st));
    st.seed = seed; st.t = t; st.pid = pid; st.px = px; st.py = py; st.pz = pz;
    int rc = ORC_OK;
    for (int64_t k = 0; k < ncell_sel; ++k) {
        int r = collide_cell(&st, cell_id ? cell_id[k] : (uint32_t)k, lo[k], hi[k], base);
        if (r != ORC_OK) rc = r;
    }
    if (counters) { counters[0] = st.pairs; counters[1] = st.collisions; counters[2] = st.rounds; }
    return rc;
}

/* ------------------------------------------------------------------------------------
 * Local ("per-cell") cross section for a constant shear viscosity to entropy density ratio
 * (Fig. 3 caption "local cross section"; the constant-eta/s runs of ref. [1],
 * PAPER.md:108; sigma_cell from the cell's n and <E>).  Reading A24
 * (DESIGN.md): for an isotropic cross section and a massless Boltzmann gas eta = (6/5) T/sigma
 * and s = 4 n, so eta/s fixes  sigma_cell = (3/10) T / (n (eta/s))  with, per cell,
 * T = <E>/3 (in fm^-1: divided by hbar c = 0.197327 GeV fm) and n = n_cell/(r_test V_cell).
 * Eq. 3 without v_rel then reads
 *     base_cell = sigma_cell dt/(r_test V_cell) = ((0.1 S) dt) / (((hbarc (n n)) etas)),
 * S = sum of the cell's energies at the start of S5.  So that S does not depend on the order of
 * summation (R(n) and every P must be identical in any implementation), it is DEFINED as the
 * exact fixed-point sum  S = (sum_i rint(E_i 2^40)) 2^-40  (64-bit integers; rint = to nearest,
 * ties to even; E < 2^22 GeV).
 * ---------------------------------------------------------------------------------- */
#define ORC_HBARC 0.197327
double oracle_local_base(int64_t n, const double *px, const double *py, const double *pz, double dt, double etas)
{
    int64_t acc = 0;
    for (int64_t i = 0; i < n; ++i) acc += (int64_t)llrint(energy(px[i], py[i], pz[i]) * 1099511627776.0);
    double S = (double)acc * (1.0 / 1099511627776.0);
    double nn = (double)n * (double)n;
    return ((0.1 * S) * dt) / ((ORC_HBARC * nn) * etas);
}

/* One step, reading A1 (Fig. 1 is missing): stream -> reflect -> bin -> pair -> collide.
 * etas > 0 selects the local cross section (sigma is then ignored). */
static int step_once_mode(oracle_state *st, double dt, double sigma, double etas);
static int step_once(oracle_state *st, double dt, double sigma) { return step_once_mode(st, dt, sigma, 0.0); }

static int step_once_mode(oracle_state *st, double dt, double sigma, double etas)
{
    double dmin = st->box[0] / st->ncell[0];
    for (int k = 1; k < 3; ++k)
        if (st->box[k] / st->ncell[k] < dmin) dmin = st->box[k] / st->ncell[k];
    if (!(dt > 0.0) || !(sigma >= 0.0)) return ORC_ERR_ARG;
    if (!(dt < dmin)) return ORC_ERR_CFL; /* PAPER.md:62 "dt is always chosen smaller than dx" */
    double dx = st->box[0] / (double)st->ncell[0];
    double dy = st->box[1] / (double)st->ncell[1];
    double dz = st->box[2] / (double)st->ncell[2];
    double V = (dx * dy) * dz;
    double base = (sigma * dt) / (st->n_test * V); /* Eq. 3 without v_rel; A3: divide by r_test */
    st->trace_len = 0;
    oracle_stream_reflect(st->n, st->x, st->y, st->z, st->px, st->py, st->pz, dt, st->box,
                          st->wall_dp);
    bin_and_sort(st);
    int rc = ORC_OK;
    for (int64_t c = 0; c < st->ncells; ++c) {
        int64_t lo = st->cell_start[c], hi = st->cell_start[c + 1];
        if ((uint32_t)(hi - lo) > st->max_occupancy) st->max_occupancy = (uint32_t)(hi - lo);
        double b = base;
        if (etas > 0.0 && hi - lo >= 2) b = oracle_local_base(hi - lo, st->px + lo, st->py + lo, st->pz + lo, dt, etas);
        int r = collide_cell(st, (uint32_t)c, lo, hi, b);
        if (r != ORC_OK) rc = r;
    }
    st->t += 1;
    st->steps += 1;
    return rc;
}

int oracle_step(oracle_state *st, int nsteps, double dt, double sigma)
{
    for (int i = 0; i < nsteps; ++i) {
        int rc = step_once(st, dt, sigma);
        if (rc != ORC_OK) return rc;
    }
    return ORC_OK;
}

int oracle_step_etas(oracle_state *st, int nsteps, double dt, double etas)
{
    if (!(etas > 0.0)) return ORC_ERR_ARG;
    for (int i = 0; i < nsteps; ++i) {
        int rc = step_once_mode(st, dt, 0.0, etas);
        if (rc != ORC_OK) return rc;
    }
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------
 * Variable time step ("implement the parameter dt as variable"; SURVEY.md 8(f)-3:
 * dt chosen per step from the largest scaled collision probability of the state the step starts
 * from).  Reading A23: with n_max the population of the fullest cell of the current,
 * cell-sorted store (A19) and cn(n) the pair-count factor of A5,
 *     g = sigma / (r_test * V_cell);   lim = (1 - 2^-10) / ((2 cn(n_max)) g);   dt = min(dt_max, lim),
 * i.e. the dt for which the bound 2 cn base of A6 (v_rel <= 2) reaches 1 - 2^-10 in that cell: no
 * extra round, with a margin far above the rounding of the bound (landing on 1 itself would let
 * one ulp decide between one round and two); dt = dt_max if sigma = 0 or no cell holds two particles.  A cell that
 * grows beyond n_max in the step's own binning still gets R > 1 rounds (A6 stays in force).
 * dt_used (nsteps entries, may be NULL) receives the steps taken; *elapsed their sum, added
 * in step order.
 * ---------------------------------------------------------------------------------- */
double oracle_adaptive_dt(const oracle_state *st, double dt_max, double sigma)
{
    uint32_t nmax = 0;
    for (int64_t c = 0; c < st->ncells; ++c) {
        uint32_t m = st->cell_start[c + 1] - st->cell_start[c];
        if (m > nmax) nmax = m;
    }
    if (nmax < 2 || !(sigma > 0.0)) return dt_max;
    double dx = st->box[0] / (double)st->ncell[0];
    double dy = st->box[1] / (double)st->ncell[1];
    double dz = st->box[2] / (double)st->ncell[2];
    double V = (dx * dy) * dz;
    double cn = (nmax & 1u) ? (double)nmax : (double)(nmax - 1u);
    double g = sigma / (st->n_test * V);
    double lim = 0.9990234375 / ((2.0 * cn) * g);   /* 1 - 2^-10 */
    return lim < dt_max ? lim : dt_max;
}

int oracle_step_adaptive(oracle_state *st, int nsteps, double dt_max, double sigma,
                         double *dt_used, double *elapsed)
{
    double sum = 0.0;
    if (!(dt_max > 0.0) || !(sigma >= 0.0)) return ORC_ERR_ARG;
    for (int i = 0; i < nsteps; ++i) {
        double dt = oracle_adaptive_dt(st, dt_max, sigma);
        int rc = step_once(st, dt, sigma);
        if (rc != ORC_OK) return rc;
        if (dt_used) dt_used[i] = dt;
        sum = sum + dt;
    }
    if (elapsed) *elapsed = sum;
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------
 * Observables, PAPER.md:66 (total energy) and PAPER.md:68-70 Fig. 2 (energy density along
 * x).  total = (sum E, sum px, sum py, sum pz); edens[j] = sum_{i in slab j} E_i /
 * (r_test * V_slab), the lab-frame T^00 (A15).  Neumaier-compensated sums.
 * ---------------------------------------------------------------------------------- */
typedef struct { double s, c; } ksum;
static void kadd(ksum *k, double v)
{
    double t = k->s + v;
    if (fabs(k->s) >= fabs(v)) k->c += (k->s - t) + v; else k->c += (v - t) + k->s;
    k->s = t;
}

void oracle_observables(const oracle_state *st, double total[4], int nslab, double *edens)
{
    ksum tot[4] = { {0, 0}, {0, 0}, {0, 0}, {0, 0} };
    ksum *slab = (ksum *)calloc((size_t)nslab, sizeof(ksum));
    double inv_w = (double)nslab / st->box[0];
    for (int64_t i = 0; i < st->n; ++i) {
        double E = energy(st->px[i], st->py[i], st->pz[i]);
        kadd(&tot[0], E); kadd(&tot[1], st->px[i]); kadd(&tot[2], st->py[i]); kadd(&tot[3], st->pz[i]);
        int j = (int)(st->x[i] * inv_w);
        if (j > nslab - 1) j = nslab - 1;
        if (j < 0) j = 0;
        kadd(&slab[j], E);
    }
    for (int k = 0; k < 4; ++k) total[k] = tot[k].s + tot[k].c;
    double vol = ((st->n_test * (st->box[0] / (double)nslab)) * st->box[1]) * st->box[2];
    for (int j = 0; j < nslab; ++j) edens[j] = (slab[j].s + slab[j].c) / vol;
    free(slab);
}

/* ------------------------------------------------------------------------------------
 * Local-rest-frame observables (the quantities the Riemann profiles of
 * PAPER.md:66-72 and the viscosity discussion of PAPER.md:62-64, 74-82 are about).
 * Kinetic energy-momentum tensor of the testparticles of slab j (transversely homogeneous
 * set-up):  T^{mu nu}_j = sum_{i in j} p_i^mu p_i^nu / E_i / (r_test V_slab),
 * components T00, T0x, Txx, Tyy, Tzz (T0y, T0z, Txy... vanish by symmetry on average and are
 * not used).  Per particle: w = 1/E, contributions E, px, (px*px)*w, (py*py)*w, (pz*pz)*w.
 * Landau matching for a flow along x (reading A22): the energy density in the local
 * rest frame is the timelike eigenvalue of T^mu_nu restricted to (t, x),
 *     e = ((T00 - Txx) + sqrt((T00 + Txx)^2 - 4 T0x^2)) / 2,   v = T0x / (e + Txx),
 *     P_L = (e - T00) + Txx  (minus the other eigenvalue),      P_T = (Tyy + Tzz) / 2.
 * A negative discriminant (rounding) counts as 0; e + Txx = 0 (empty slab) gives v = 0.
 * ---------------------------------------------------------------------------------- */
void oracle_landau_match(double T00, double T0x, double Txx, double Tyy, double Tzz, double out[4])
{
    double tr = T00 + Txx;
    double disc = tr * tr - 4.0 * (T0x * T0x);
    if (!(disc > 0.0)) disc = 0.0;
    double e = 0.5 * ((T00 - Txx) + sqrt(disc));
    double den = e + Txx;
    out[0] = e;
    out[1] = (den > 0.0) ? T0x / den : 0.0;
    out[2] = (e - T00) + Txx;
    out[3] = 0.5 * (Tyy + Tzz);
}

/* T: 5*nslab doubles (T00[nslab], T0x[nslab], Txx, Tyy, Tzz); lrf: 4*nslab (e, v, P_L, P_T) */
void oracle_observables_lrf(const oracle_state *st, int nslab, double *T, double *lrf)
{
    ksum *acc = (ksum *)calloc((size_t)5 * nslab, sizeof(ksum));
    double inv_w = (double)nslab / st->box[0];
    for (int64_t i = 0; i < st->n; ++i) {
        double px = st->px[i], py = st->py[i], pz = st->pz[i];
        double E = energy(px, py, pz);
        double w = 1.0 / E;
        int j = (int)(st->x[i] * inv_w);
        if (j > nslab - 1) j = nslab - 1;
        if (j < 0) j = 0;
        kadd(&acc[0 * nslab + j], E);
        kadd(&acc[1 * nslab + j], px);
        kadd(&acc[2 * nslab + j], (px * px) * w);
        kadd(&acc[3 * nslab + j], (py * py) * w);
        kadd(&acc[4 * nslab + j], (pz * pz) * w);
    }
    double vol = ((st->n_test * (st->box[0] / (double)nslab)) * st->box[1]) * st->box[2];
    for (int k = 0; k < 5 * nslab; ++k) T[k] = (acc[k].s + acc[k].c) / vol;
    for (int j = 0; j < nslab; ++j) {
        double o[4];
        oracle_landau_match(T[j], T[nslab + j], T[2 * nslab + j], T[3 * nslab + j], T[4 * nslab + j], o);
        for (int k = 0; k < 4; ++k) lrf[k * nslab + j] = o[k];
    }
    free(acc);
}

/* ------------------------------------------------------------------------------------
 * Accessors for the tests.
 * ---------------------------------------------------------------------------------- */
void oracle_get_particles(const oracle_state *st, uint32_t *pid, double *x, double *y, double *z,
                          double *px, double *py, double *pz)
{
    size_t b = (size_t)st->n * sizeof(double);
    if (pid) memcpy(pid, st->pid, (size_t)st->n * sizeof(uint32_t));
    if (x) memcpy(x, st->x, b);
    if (y) memcpy(y, st->y, b);
    if (z) memcpy(z, st->z, b);
    if (px) memcpy(px, st->px, b);
    if (py) memcpy(py, st->py, b);
    if (pz) memcpy(pz, st->pz, b);
}

void oracle_get_cells(const oracle_state *st, uint32_t *cell_of_slot, uint32_t *cell_start)
{
    if (cell_of_slot) memcpy(cell_of_slot, st->cell, (size_t)st->n * sizeof(uint32_t));
    if (cell_start) memcpy(cell_start, st->cell_start, ((size_t)st->ncells + 1) * sizeof(uint32_t));
}

/* out[0..7] = steps, pairs, collisions, rounds, near_threshold, max_occupancy,
 * direction attempts, global step index */
void oracle_counters(const oracle_state *st, uint64_t out[8], double wall_dp[3])
{
    out[0] = st->steps; out[1] = st->pairs; out[2] = st->collisions; out[3] = st->rounds;
    out[4] = st->near_threshold; out[5] = st->max_occupancy; out[6] = st->dir_attempts;
    out[7] = st->t;
    if (wall_dp) memcpy(wall_dp, st->wall_dp, 3 * sizeof(double));
}

int64_t oracle_trace_len(const oracle_state *st) { return st->trace_len; }

void oracle_trace_copy(const oracle_state *st, uint32_t *cell, uint32_t *round, uint32_t *pid_a,
                       uint32_t *pid_b, double *P, double *u, uint8_t *decided)
{
    for (int64_t i = 0; i < st->trace_len; ++i) {
        cell[i] = st->trace[i].cell; round[i] = st->trace[i].round;
        pid_a[i] = st->trace[i].pid_a; pid_b[i] = st->trace[i].pid_b;
        P[i] = st->trace[i].P; u[i] = st->trace[i].u; decided[i] = st->trace[i].decided;
    }
}

int64_t oracle_dirlog_len(const oracle_state *st) { return st->dirlog_len; }
void oracle_dirlog_copy(const oracle_state *st, double *out)
{
    memcpy(out, st->dirlog, (size_t)st->dirlog_len * 3 * sizeof(double));
}

/* Shuffle order of one hypothetical cell (for the pairing pin P12): pids in, order out. */
void oracle_shuffle_order(uint64_t seed, uint32_t t, uint32_t rho, int64_t n,
                          const uint32_t *pids, uint32_t *order_pids)
{
    shuf_item *o = (shuf_item *)malloc((size_t)n * sizeof(shuf_item));
    for (int64_t j = 0; j < n; ++j) {
        uint32_t w[4];
        draw(seed, pids[j], t, rho >> 2, TAG_SHUF, 0, w);
        o[j].key = ((uint64_t)w[rho & 3] << 32) | (uint64_t)pids[j];
        o[j].slot = j;
    }
    qsort(o, (size_t)n, sizeof(shuf_item), cmp_shuf);
    for (int64_t j = 0; j < n; ++j) order_pids[j] = pids[o[j].slot];
    free(o);
}
