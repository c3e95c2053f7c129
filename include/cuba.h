/*
 * cuba.h -- C ABI of the B200-native CuBA hot path (arXiv:1208.0961, "CuBA - a CUDA
 * implementation of BAMPS"; citations are /root/reference/PAPER.md line numbers).
 *
 * One call sequence, one GPU:   cuba_init -> cuba_step* -> cuba_observables -> cuba_destroy
 *
 * What a step computes (section 2; order per DESIGN.md reading A1):
 *   S1  free streaming      x -> x + c^2 p_x/E dt, same for y,z        PAPER.md:34 Eq. 2
 *   S2  wall reflection     elastic, off the six walls of the box
 *   S3  cell index          cells of volume dx dy dz
 *   S4  stable counting sort of the particle store by cell             north_star (3)
 *   S5  per cell: Philox-keyed shuffle, pair 2k with 2k+1, collide with
 *       P22 = v_rel (sigma/N_test)(dt/V_cell) * n(n-1)/(2 floor(n/2)),
 *       v_rel = s/(2 E1 E2), s = (p1+p2)^2; on a hit boost to the CM frame,
 *       draw an isotropic direction, boost back                        PAPER.md:38-44 Eq. 3
 * All arithmetic is IEEE fp64, one rounding per written operation, no FMA contraction
 * (A2), so a trajectory is a pure function of (initial state, seed).
 *
 * Conventions: c = 1; lengths fm, time fm/c, momenta and energies GeV, sigma in fm^2
 * (10 GeV^-2 = 0.389379 fm^2 with hbar c = 0.197327 GeV fm).  Massless gluons: E = |p| is
 * never stored.  `n_test` is the testparticle multiplier r_test of PAPER.md:44 (the divisor
 * in Eq. 3, A3).
 *
 * Memory: every pointer is labelled DEVICE or HOST.  The caller (PyTorch in the shipped
 * binding) allocates all device memory; the library allocates no device memory on the cuba_step
 * path (for problems of up to 2^20 particles the first cuba_step of a given (dt, sigma) instantiates
 * a CUDA graph of two steps once -- a driver-side allocation; CUBA_OPT_GRAPH = 0 avoids it).
 * Errors: every call returns 0 or a negative CUBA_ERR_* code; nothing throws or aborts.
 * There is no CPU fallback: without a CUDA device every call fails with CUBA_ERR_CUDA.
 */
#ifndef CUBA_H
#define CUBA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CUBA_OK 0
#define CUBA_ERR_NULL (-1)        /* a required pointer is null                              */
#define CUBA_ERR_SIZE (-2)        /* n < 1, n >= 2^32, ncell < 1, ncells >= 2^27, nslab < 1   */
#define CUBA_ERR_VALUE (-3)       /* non-positive box / n_test / dt, negative sigma           */
#define CUBA_ERR_WORKSPACE (-4)   /* workspace smaller than cuba_workspace_bytes or misaligned */
#define CUBA_ERR_CUDA (-5)        /* a CUDA runtime call failed (cuba_last_cuda_error)        */
#define CUBA_ERR_STATE (-6)       /* a particle outside [0,L], non-finite, or with p = 0      */
#define CUBA_ERR_CFL (-7)         /* dt not below the smallest cell edge        */
#define CUBA_ERR_MOVED (-8)       /* device check: a particle crossed more than one cell      */
#define CUBA_ERR_ROUNDS (-9)      /* a cell needs more than CUBA_MAX_ROUNDS rounds (A6)       */
#define CUBA_ERR_TRACE (-10)      /* trace capacity too small                                 */
#define CUBA_ERR_HALO (-11)       /* device check: a halo buffer's header is not the count given */

#define CUBA_MAX_ROUNDS 64

typedef struct cuba_ctx cuba_ctx; /* opaque; owned by the library, freed by cuba_destroy */

/* Device pointers to the current particle store (SoA, array order = cell-sorted order). */
typedef struct cuba_soa {
    double *x, *y, *z, *px, *py, *pz; /* DEVICE, n doubles each */
    uint32_t *pid;                    /* DEVICE, n: persistent id = index in the arrays given to cuba_init */
    uint32_t *cell_start;             /* DEVICE, ncells+1: slots [cell_start[c], cell_start[c+1]) hold cell c */
} cuba_soa;

typedef struct cuba_counters_t {
    uint64_t steps;          /* steps done since cuba_init                                   */
    uint64_t pairs;          /* collision-pair evaluations (sum over steps, cells, rounds)   */
    uint64_t collisions;     /* pairs that collided                                          */
    uint64_t rounds;         /* sum over steps and cells with n >= 2 of R(n) (A6)            */
    uint64_t near_threshold; /* decisions with |u - P| <= 1e-12 (A16)                        */
    uint64_t max_occupancy;  /* largest cell population seen                                 */
    uint64_t overflow_cells; /* cells too large for shared memory, done by the global path   */
    uint64_t device_flags;   /* sticky device error bits (0 when healthy)                    */
} cuba_counters_t;

/* Trace of ONE step for the bit-exact parity check.  All arrays are HOST memory owned by
 * the caller.  Pairs are listed in (cell, round, k) order, k = index in the shuffled
 * order; pair k of a round joins order[2k] (pid_a) and order[2k+1] (pid_b). */
typedef struct cuba_trace {
    uint32_t *cell_of_pid; /* HOST, n: cell index of every particle after S3, by pid       */
    int64_t pair_capacity; /* in: entries available in the arrays below                    */
    int64_t n_pairs;       /* out: pairs evaluated in this step                            */
    uint32_t *pair_cell;   /* HOST, pair_capacity                                          */
    uint32_t *pair_round;  /* HOST                                                         */
    uint32_t *pid_a;       /* HOST                                                         */
    uint32_t *pid_b;       /* HOST                                                         */
    double *P;             /* HOST: scaled collision probability of Eq. 3                  */
    double *u;             /* HOST: the uniform it was compared with                       */
    uint8_t *decided;      /* HOST: 1 iff u < P                                            */
} cuba_trace;

/* Bytes of DEVICE workspace cuba_init needs for n particles on an ncell[0..2] grid
 * (second copy of the particle store for the out-of-place sort, pid arrays, cell tables,
 * sort scratch).  Returns 0 for invalid arguments.  The workspace must be 256-byte aligned. */
size_t cuba_workspace_bytes(int64_t n, const int ncell[3]);

/* Adopt a particle store.  PAPER.md:32 (cells, per-particle r and p), PAPER.md:44 (box with
 * six walls at 0 and L; N_test).  x..pz are DEVICE arrays of n doubles (16-byte aligned), adopted in place and
 * to be kept alive (with `workspace`) until cuba_destroy.  Assigns pid[i] = i, validates the
 * state on the device (CUBA_ERR_STATE), and bins the initial positions with S3+S4 so that
 * the store is cell-sorted from the start (A19); on return the caller's arrays
 * hold the sorted state.  `cuda_stream` is a cudaStream_t (NULL = default stream); all later
 * work is enqueued on it.  Synchronises once. */
int cuba_init(cuba_ctx **out, const double box[3], const int ncell[3], int64_t n,
              double *x, double *y, double *z, double *px, double *py, double *pz,
              double n_test, uint64_t seed, void *workspace, size_t workspace_bytes,
              void *cuda_stream);

/* Advance nsteps steps of S1..S5 with time step dt (fm/c) and total cross section sigma
 * (fm^2).  Asynchronous: kernels are enqueued on the context's stream, no host
 * synchronisation.  cuba_step(k) == k x cuba_step(1) bit for bit (the global step index is
 * the only RNG state).  After the call the current store alternates between the caller's
 * arrays and the workspace copy: ask cuba_state() where it is.  Errors: CUBA_ERR_VALUE,
 * CUBA_ERR_CFL synchronously; device-side conditions (CUBA_ERR_MOVED, CUBA_ERR_ROUNDS)
 * surface at the next synchronising call. */
int cuba_step(cuba_ctx *ctx, int nsteps, double dt, double sigma);

/* Local ("per-cell") cross section for a constant shear viscosity to entropy density ratio
 * ("local cross section", constant-eta/s runs of ref. [1] PAPER.md:108; DESIGN.md
 * reading A24).  As cuba_step, but in every cell the total cross section of Eq. 3 is
 *     sigma_cell = (3/10) T / (n * eta_over_s),  T = <E>/3 of the cell's particles (GeV / 0.197327
 *     GeV fm), n = n_cell / (n_test * V_cell)
 * (eta = (6/5) T/sigma and s = 4 n for an isotropic cross section and a massless Boltzmann gas);
 * the cell's energy sum is the exact fixed-point sum (sum rint(E 2^40)) 2^-40, so the result does
 * not depend on any summation order.  Errors as cuba_step; eta_over_s <= 0: CUBA_ERR_VALUE. */
int cuba_step_local_sigma(cuba_ctx *ctx, int nsteps, double dt, double eta_over_s);

/* Variable time step ("implement the parameter dt as variable"; DESIGN.md reading
 * A23).  Before each of the nsteps steps, with n_max the population of the fullest cell of the
 * current store and cn = n_max (odd) or n_max - 1 (even),
 *     dt = min(dt_max, (1 - 2^-10) / ((2 cn) * sigma / (n_test * V_cell)))
 * (dt_max if sigma = 0 or no cell holds two particles): the scaled Eq. 3 probability stays below
 * 1 in that cell without extra rounds; cells that outgrow it in the step's own binning still get
 * extra rounds.  Then the step runs exactly as cuba_step(ctx, 1, dt, sigma).  dt_used (HOST,
 * nsteps doubles, may be NULL) receives the steps taken, *elapsed (HOST, may be NULL) their sum
 * in step order.  Synchronises once per step (a 4-byte read-back of n_max).  Errors as
 * cuba_step; the CFL check applies to every dt actually taken. */
int cuba_step_adaptive(cuba_ctx *ctx, int nsteps, double dt_max, double sigma, double *dt_used, double *elapsed);

/* Execution options (results are bit-identical for every setting; they only change how the
 * step is scheduled on the device).  CUBA_OPT_FUSE_HIST (default 1): the collision kernel of
 * step t also performs S1-S3 of step t+1 on the momenta it holds on chip and writes the
 * (cell, direction) histogram of the counting sort, so that consecutive steps with the same
 * dt skip the separate streaming/histogram pass; a step whose dt differs from the previous
 * one (or that follows cuba_init / cuba_step_traced) runs that pass.  value 0 always runs the
 * separate pass.  Errors: CUBA_ERR_NULL, CUBA_ERR_VALUE (unknown option or value; in a slab context
 * (cuba_slab_init) a non-zero value for CUBA_OPT_FUSE_HIST, CUBA_OPT_GRAPH or CUBA_OPT_SLOTS: those
 * schedules are not available there and stay off). */
#define CUBA_OPT_FUSE_HIST 1
/* CUBA_OPT_GRAPH (default 1): for problems of up to 2^20 particles, whose step is bound by the host
 * cost of its launches, cuba_step replays a CUDA graph of two steps (captured on first use for the
 * given dt and sigma) instead of launching the kernels one by one -- provided the context's stream
 * can be captured (not the legacy default stream or cudaStreamPerThread) and per-kernel profiling
 * is off.  value 0: plain launches.  Results are identical either way. */
#define CUBA_OPT_GRAPH 2
/* CUBA_OPT_SLOTS (default 0): schedule of cuba_step.  0: the compact schedule (histogram, scan, scatter,
 * collide) on the caller's arrays and workspace only.  1: a call of at least 4 steps on a problem that is
 * not launch-bound runs on the slotted store (one kernel per step and size class);
 * 2: every call does.  The slotted store is device memory allocated BY THE LIBRARY on first use (two
 * copies of ncells * slots-per-cell * 52 bytes, 7 GB at 25M particles) and freed by cuba_destroy -- the
 * one exception to "the caller owns all device memory", which is why it is opt-in; if the allocation
 * fails the compact schedule runs.  Measured at 25M particles: 1.57 vs 1.61 ms per step.  Results are
 * bit-identical for every setting. */
#define CUBA_OPT_SLOTS 3
/* CUBA_OPT_SLOT_MARGIN (default 100): per cent by which the segment capacities of the slotted store
 * are scaled, 1..1000.  A run that outgrows a capacity is detected at the next synchronising call and
 * redone on the compact schedule from the state it started from; small values exist to test that.
 * Synchronises if a slotted run is still unverified; releases the slotted store. */
#define CUBA_OPT_SLOT_MARGIN 4
int cuba_set_option(cuba_ctx *ctx, int option, int value);
/* Diagnostics of the slotted schedule (CUBA_OPT_SLOTS): HOST out[0] = calls of cuba_step that ran on the
 * slotted store since cuba_init, out[1] = those that outgrew a segment and were redone on the compact
 * schedule.  Verifies a pending run first (synchronises then).  Errors: CUBA_ERR_NULL, or what the
 * redone run returned. */
int cuba_slot_stats(cuba_ctx *ctx, uint64_t out[2]);

/* PAPER.md:66 (total energy) and PAPER.md:68-70 Fig. 2 (energy density along x).
 * total = (sum E, sum px, sum py, sum pz) in GeV; edens[j] = sum_{i in slab j} E_i /
 * (n_test * V_slab) in GeV/fm^3 for nslab equal slabs along x (lab-frame T^00, A15).
 * HOST outputs; synchronises the stream and reports pending device errors. */
int cuba_observables(cuba_ctx *ctx, double total[4], int nslab, double *edens);

/* Local-rest-frame observables (the quantities behind the Riemann profiles
 * and the viscosity discussion of PAPER.md:62-72).  Kinetic energy-momentum tensor of the
 * testparticles per x-slab, T^{mu nu} = sum p^mu p^nu / E / (n_test * V_slab) in GeV/fm^3:
 *   T   HOST, 5*nslab doubles: T00[nslab], T0x[nslab], Txx[nslab], Tyy[nslab], Tzz[nslab];
 *   lrf HOST, 4*nslab doubles: e[nslab] (energy density in the local rest frame, Landau matching
 *       for a flow along x: e = ((T00-Txx) + sqrt((T00+Txx)^2 - 4 T0x^2))/2), v[nslab] (flow
 *       velocity T0x/(e+Txx), 0 for an empty slab), P_L[nslab] = e - T00 + Txx, P_T[nslab] =
 *       (Tyy+Tzz)/2.
 * 1 <= nslab <= 256 (CUBA_ERR_SIZE otherwise).  Synchronises; reports pending device errors. */
int cuba_observables_lrf(cuba_ctx *ctx, int nslab, double *T, double *lrf);

/* The totals and the energy density per x-slab of cuba_observables (Fig. 2), for
 * callers that are not allowed to allocate GPU memory or to wait for the GPU: code that runs inside somebody
 * else's memory budget (a plug-in of a host application that owns the allocator, a process sharing the GPU
 * under a fixed memory reservation), an in-situ analysis hook called between steps of a running loop, where an
 * allocation or a free can stall every stream of the device, or a service that pre-allocates everything at start-up and
 * treats a later allocation as a fault.  cuba_observables needs a context (cuba_init allocates pinned host
 * memory, streams and events) and keeps its per-block partial sums in the workspace; this call needs neither.
 * It takes no context, calls no cudaMalloc / cudaFree / cudaMallocHost and no library routine that allocates,
 * does not synchronise and copies nothing to the host: it enqueues two kernels on `cuda_stream` and returns.
 *
 *   n                      particles, 1 <= n < 2^32
 *   x, px, py, pz          DEVICE, n doubles each (8-byte aligned), read only, owned by the caller; any order
 *                          works, a cell-sorted store (cuba_state) is what the kernel is fast on
 *   box[3], n_test         HOST: box edges in fm and the testparticle multiplier, as given to cuba_init
 *   nslab                  1 .. CUBA_NOALLOC_MAX_SLABS equal slabs along x
 *   result                 DEVICE, 4 + nslab doubles, owned by the caller, written in stream order:
 *                          sum E, sum px, sum py, sum pz, then edens[nslab] = slab energy / (n_test V_slab)
 *   cuda_stream            a cudaStream_t (NULL = default stream)
 *
 * Where the partial sums go: a fixed array inside the library image (static __device__, 592 x (4 +
 * CUBA_NOALLOC_MAX_SLABS) doubles = 625,152 bytes).  Every GPU on which the library is loaded holds that array
 * until the process exits, used or not -- which is why the limit on nslab is modest.  Consequences:
 *   - nslab > CUBA_NOALLOC_MAX_SLABS returns CUBA_ERR_SIZE and launches nothing (use cuba_observables, whose
 *     limit is 1024, if you can afford a context);
 *   - the FIRST call on each device looks up the array's device address (cudaGetSymbolAddress with that device
 *     current; the result is remembered per device).  Make that first call during set-up, outside any stream
 *     capture; the call uses whatever device is current and `cuda_stream` must belong to it;
 *   - all calls on a device share the one array.  Nothing in it has to be zero beforehand (every block
 *     overwrites its whole row before the second kernel reads it, so the previous call's contents do not
 *     matter), but two calls whose kernels can overlap on the GPU -- different streams without an ordering
 *     between them, or two host threads -- race on it and give wrong sums.  Calls on one stream are safe.
 * The arithmetic, grid and summation order are those of cuba_observables for nslab <= 2 nx: same bits there,
 * within 1e-12 relative elsewhere.  Errors: CUBA_ERR_NULL, CUBA_ERR_SIZE (n, nslab), CUBA_ERR_VALUE (box,
 * n_test, more than 64 devices), CUBA_ERR_WORKSPACE (misaligned pointer), CUBA_ERR_CUDA (no device; launch
 * failed).  Device-side problems in the inputs (non-finite values) are not checked: the sums carry them. */
#define CUBA_NOALLOC_MAX_SLABS 128
int cuba_observables_noalloc(int64_t n, const double *x, const double *px, const double *py, const double *pz,
                             const double box[3], double n_test, int nslab, double *result, void *cuda_stream);

/* Where the current state lives (DEVICE pointers, valid until the next cuba_step). */
int cuba_state(cuba_ctx *ctx, cuba_soa *out);

/* Copy the current state to HOST arrays in array order (any pointer may be null). Synchronises. */
int cuba_get_particles(cuba_ctx *ctx, uint32_t *pid, double *x, double *y, double *z,
                       double *px, double *py, double *pz);

/* Copy cell_start (ncells+1 entries) of the current state to HOST memory.  Synchronises. */
int cuba_get_cells(cuba_ctx *ctx, uint32_t *cell_start);

/* One step with the parity trace filled (slow path: allocates temporary device memory,
 * synchronises).  The state advances exactly as with cuba_step(ctx, 1, dt, sigma) -- also when
 * the records cannot be taken: with CUBA_ERR_TRACE (out->n_pairs then holds the capacity that
 * was needed; cell_of_pid is filled) or after a failed temporary allocation the step is completed
 * without records, so the context stays valid and one step further; a retry traces the NEXT step. */
int cuba_step_traced(cuba_ctx *ctx, double dt, double sigma, cuba_trace *out);

/* Counters since cuba_init.  Synchronises. */
int cuba_counters(cuba_ctx *ctx, cuba_counters_t *out);

/* End-to-end convenience for HOST-resident data: allocates device memory, uploads the six
 * HOST arrays (n doubles each), runs cuba_init + cuba_step(nsteps) + cuba_observables,
 * optionally downloads the final state into the same HOST arrays (pid_out may be null;
 * download != 0 to copy back), frees everything.  Device memory comes from a memory pool owned
 * by the library (kept between calls so that a second call of the same size maps nothing new;
 * the process-wide default pool is not touched).  Used for the bench's e2e number. */
int cuba_run_host(const double box[3], const int ncell[3], int64_t n,
                  double *x, double *y, double *z, double *px, double *py, double *pz,
                  double n_test, uint64_t seed, int nsteps, double dt, double sigma,
                  double total[4], int nslab, double *edens, uint32_t *pid_out, int download);

/* Per-kernel timing for the roofline report.  cuba_profile_enable(ctx, 1) makes cuba_step
 * record a CUDA event on the context's stream after every kernel it launches (host cost
 * ~1 us per event, no device-side serialisation beyond the stream's own order);
 * cuba_profile_read synchronises and returns, for each of the CUBA_PROFILE_GROUPS kernel
 * groups, the summed device time in milliseconds and the number of launches since the last
 * enable, then clears the log.  HOST outputs of CUBA_PROFILE_GROUPS entries each.
 * Mode 1 times the collision kernels as one group (the size classes run concurrently on
 * internal streams, as in normal operation); mode 2 serialises them on the caller's stream and
 * times every class by itself (diagnostic: slower than normal operation); 0 switches off. */
#define CUBA_PROFILE_GROUPS 21
int cuba_profile_enable(cuba_ctx *ctx, int on);
int cuba_profile_read(cuba_ctx *ctx, double *ms_sum, uint64_t *launches);
const char *cuba_profile_name(int group);

/* ---- x-slab decomposition over several GPUs (collisions happen inside a
 * cell only: dt below the cell edge) ----------------------------------------------------------------
 * One context per rank.  A rank OWNS the cell layers [layer_lo, layer_hi) along x of the global grid and keeps a
 * copy (ghost) of the adjacent boundary layer of each neighbour, all in the coordinates and cell numbering of
 * the whole problem, so that every operation rounds exactly as on one GPU.  Protocol of one step, the same on
 * every rank:  cuba_step(ctx, 1, dt, sigma)  ->  cuba_slab_count / cuba_slab_pack for side 0 (lowest owned layer)
 * and side 1 (highest)  ->  send each buffer to that neighbour, receive theirs (torch.distributed / NCCL: the
 * library does not communicate)  ->  cuba_slab_unpack.  The owned ranges of all ranks, concatenated in rank
 * order, are the one-GPU store bit for bit (array order, positions, momenta, pids); counters add up.
 *
 * cuba_slab_init: like cuba_init, but the DEVICE arrays x..pz hold `capacity` doubles (room for the ghosts and for
 * fluctuations), the first n entries given: ALL particles of the problem whose cell lies in the layers
 * [layer_lo - 1, layer_hi + 1), in ascending order of their global index, and pid (DEVICE, n) those global
 * indices.  workspace: cuba_workspace_bytes(capacity, ncell).  Every rank passes the same box, ncell, n_test, seed.
 * In a slab context: cuba_step takes nsteps <= 1; the fused histogram, the CUDA graph and the slotted schedule
 * are off; cuba_step_traced and cuba_step_adaptive return CUBA_ERR_VALUE; cuba_observables(_lrf) cover the owned
 * particles only (add the ranks' results); cuba_get_particles / cuba_state give the whole local store, of which
 * cuba_slab_owned names the owned part.  Errors as cuba_init, plus CUBA_ERR_SIZE (n > capacity) and
 * CUBA_ERR_VALUE (layers). */
int cuba_slab_init(cuba_ctx **out, const double box[3], const int ncell[3], int64_t capacity, int64_t n,
                   double *x, double *y, double *z, double *px, double *py, double *pz, const uint32_t *pid,
                   double n_test, uint64_t seed, void *workspace, size_t workspace_bytes, void *cuda_stream,
                   int layer_lo, int layer_hi);
/* The cell layer along x of every particle, exactly as S3 computes it on the device (the cells the
 * particles are sorted into; the same inline function as the kernels, compiled for the host: trunc(x * (1 /
 * (box_x / nx))) clamped to [0, nx - 1]).  HOST in, HOST out, no device needed: x (n doubles), layer (n int32).
 * This is what decides which rank is given a particle at the start (cuba_slab_init wants the particles of the
 * layers [layer_lo - 1, layer_hi + 1)) and what the cuts are balanced with; a particle on a layer face goes where
 * the device would bin it.  Errors: CUBA_ERR_NULL, CUBA_ERR_SIZE (n < 0, nx < 1), CUBA_ERR_VALUE (box_x). */
int cuba_slab_layer_index(double box_x, int nx, int64_t n, const double *x, int32_t *layer);
/* HOST out[4] = first slot of the owned part of the current store, its length, particles in the store, capacity.
 * Synchronises (reads four words back) once after a step. */
int cuba_slab_owned(cuba_ctx *ctx, int64_t out[4]);
/* HOST *count = particles in the owned boundary layer on `side` (0: layer_lo, 1: layer_hi - 1). */
int cuba_slab_count(cuba_ctx *ctx, int side, int64_t *count);
/* Bytes of a halo buffer for `count` particles: 16-byte header {count, cells per layer}, six double arrays,
 * the pids, the population of every cell of the layer. */
size_t cuba_slab_buffer_bytes(int64_t count, const int ncell[3]);
/* Copies the owned boundary layer on `side` into `buffer` (DEVICE, 16-byte aligned, at least
 * cuba_slab_buffer_bytes(cuba_slab_count)); stream-ordered.  CUBA_ERR_SIZE if the buffer is too small. */
int cuba_slab_pack(cuba_ctx *ctx, int side, void *buffer, size_t buffer_bytes);
/* Rebuilds the store as [lo_buffer's particles][owned cells][hi_buffer's particles] and its cell table; the
 * buffers are what the lower / upper neighbour packed for its side 1 / side 0 (DEVICE; null exactly where there
 * is no neighbour), the counts those of cuba_slab_count there.  Stream-ordered after one synchronisation.
 * CUBA_ERR_SIZE if the capacity is exceeded, CUBA_ERR_VALUE for a buffer where no neighbour is (or none where
 * one is).  The header {count, cells per layer} that cuba_slab_pack wrote into each buffer is compared on the
 * device with the count given here and with this grid; a mismatch (a buffer paired with the wrong count, a
 * truncated transfer) surfaces as CUBA_ERR_HALO at the next synchronising call -- the store is then invalid. */
int cuba_slab_unpack(cuba_ctx *ctx, const void *lo_buffer, int64_t lo_count, const void *hi_buffer, int64_t hi_count);

/* fp64 leg of the roofline (fp64-pipe utilisation against a measured peak; no passage of
 * the paper: a timing probe).  Launches a kernel of dependent DFMA chains (8 per thread, 8 x SM count
 * CTAs of 256 threads) `repeats` times (1..64) after one warm-up on `cuda_stream` (a cudaStream_t, may
 * be null = default stream), times each with CUDA events and writes the best rate to the HOST double
 * *dfma_per_s: thread-level fp64 FMA instructions per second of the whole device (x 2 = FLOP/s,
 * / 32 = warp instructions/s).  Allocates and frees its own small device buffer; synchronises.
 * Errors: CUBA_ERR_NULL, CUBA_ERR_SIZE, CUBA_ERR_CUDA (*dfma_per_s = 0). */
int cuba_probe_fp64(void *cuda_stream, int repeats, double *dfma_per_s);

void cuba_destroy(cuba_ctx *ctx);
const char *cuba_strerror(int code);
/* Text of the last CUDA runtime error seen by this library in the calling process. */
const char *cuba_last_cuda_error(void);
/* Number of kernel launches this library has issued in the calling process. */
uint64_t cuba_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* CUBA_H */
