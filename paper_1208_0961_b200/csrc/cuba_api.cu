// cuba_api.cu -- the C ABI of include/cuba.h: argument validation, workspace carving and
// stream-ordered kernel launches.  No CPU fallback: every entry point needs a CUDA device.
#include "../../include/cuba.h"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "bin.cuh"
#include "collide.cuh"
#include "common.cuh"
#include "init_sort.cuh"
#include "observe.cuh"
#include "slots.cuh"
#include "probe.cuh"

using namespace cuba;

namespace {

std::atomic<uint64_t> g_launches{0};
thread_local char g_cuda_err[256] = "";

bool cuda_ok(cudaError_t e, const char *what)
{
    if (e == cudaSuccess) return true;
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", what, cudaGetErrorString(e));
    return false;
}
#define CU(call) do { if (!cuda_ok((call), #call)) return CUBA_ERR_CUDA; } while (0)
#define LAUNCHED() do { g_launches.fetch_add(1, std::memory_order_relaxed); if (!cuda_ok(cudaGetLastError(), "kernel launch")) return CUBA_ERR_CUDA; } while (0)

// Size classes of the collision kernels: X(index, threads per CTA, items per thread, capacity
// in particles, min CTAs per SM).  A cell goes to the first class whose capacity holds it; a
// cell beyond the last capacity goes to the global-memory overflow kernel.  Thread counts are
// about a quarter of the capacity so that every thread owns <= 4 particles and <= 2 pairs.
// Listed (and launched) biggest first: the big cells are the long poles.
#ifndef CUBA_C4_T   // class 4 (the ~1350-particle hot cells of the 25M-particle Riemann problem) is tunable at build time
#define CUBA_C4_T 256
#define CUBA_C4_I 6
#define CUBA_C4_CAP 1536
#define CUBA_C4_MB 3
#endif
#ifndef CUBA_C1_MB   // resident CTAs per SM asked for the two smallest classes (latency bound: occupancy over registers)
#define CUBA_C1_MB 12
#endif
#ifndef CUBA_C0_MB
#define CUBA_C0_MB 16
#endif
#ifndef CUBA_C2_MB
#define CUBA_C2_MB 8
#endif
#ifndef CUBA_C3_MB
#define CUBA_C3_MB 4
#endif
#define CUBA_FOR_EACH_CLASS(X) \
    X(6, 1024, 5, 4544, 1)     \
    X(5, 512, 4, 2048, 2)      \
    X(4, CUBA_C4_T, CUBA_C4_I, CUBA_C4_CAP, CUBA_C4_MB) \
    X(3, 224, 4, 896, CUBA_C3_MB) \
    X(2, 128, 4, 512, CUBA_C2_MB) \
    X(1, 64, 4, 256, CUBA_C1_MB) \
    X(0, 32, 4, 128, CUBA_C0_MB)
constexpr int kSmemClasses = 7;
static_assert(kSmemClasses + 1 == kNumClasses, "class table");

size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

struct Layout {
    size_t setB[6], pidA, pidB, cnt, count_new, cell_start, block_sum, tile_rec, carry, class_list,
        zero, counters, flags, tdev, max_occ, obs_partial, obs_result, arena32, arenaE, rsH, rsSums, total;
    int64_t ntiles, nblocks_cells, rs_blocks, arena_entries;
};

constexpr int kObsGrid = 148 * 4;   // resident CTAs: 4 per SM at 64 registers
constexpr int kZeroWords = 32;   // class_count[8], work[8], arena cursor (u64 = 2 words), [20] fullest cell of this binning, pad
constexpr int kStepMaxWord = 20;

Layout make_layout(int64_t n, int64_t ncells)
{
    Layout L{};
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
    L.ntiles = (n + kTile - 1) / kTile;
    L.nblocks_cells = (ncells + 255) / 256;
    L.rs_blocks = (n + kRsTile - 1) / kRsTile;
    L.arena_entries = n + 2 * ncells + 8;
    for (int k = 0; k < 6; ++k) L.setB[k] = take((size_t)n * 8);
    L.pidA = take((size_t)n * 4);
    L.pidB = take((size_t)n * 4);
    L.cnt = take((size_t)kDirs * ncells * 4);
    L.count_new = take((size_t)ncells * 4);
    L.cell_start = take((size_t)(ncells + 1) * 4);
    L.block_sum = take((size_t)L.nblocks_cells * 4);
    L.tile_rec = take((size_t)L.ntiles * kTileRec * 4);
    L.carry = take((size_t)L.ntiles * kTileRec * 4);
    L.class_list = take((size_t)kNumClasses * ncells * 16);
    L.zero = take(kZeroWords * 4);
    L.counters = take(8 * 8);
    L.flags = take(4);
    L.tdev = take(4);
    L.max_occ = take(8);
    constexpr size_t obs_words = (4 + kObsMaxSlabs) > kLrfComp * kLrfMaxSlabs ? (4 + kObsMaxSlabs) : kLrfComp * kLrfMaxSlabs;
    constexpr size_t res_words = (4 + kObsMaxSlabs) > 9 * kLrfMaxSlabs ? (4 + kObsMaxSlabs) : 9 * kLrfMaxSlabs;
    L.obs_partial = take((size_t)kObsGrid * obs_words * 8);
    L.obs_result = take(res_words * 8);
    L.arena32 = take((size_t)L.arena_entries * 16);   // also the init sort's key/value double buffers
    L.arenaE = take((size_t)L.arena_entries * 8);
    L.rsH = take((size_t)256 * L.rs_blocks * 4);
    L.rsSums = take(((size_t)256 * L.rs_blocks / kScanChunk + 2) * 4);
    L.total = o;
    return L;
}

}  // namespace

struct cuba_ctx {
    Geom g;
    int64_t n;           // particles in the store (x-slab decomposition: changes with every halo exchange)
    int64_t cap;         // particles the arrays and the workspace were sized for
    // x-slab decomposition (cuba_slab_*): this context owns the cell layers [layer_lo, layer_hi) = the cells
    // [own_lo, own_hi); its store also holds a copy of the neighbours' boundary layers (ghosts)
    bool slab = false;
    int layer_lo = 0, layer_hi = 0;
    uint32_t own_lo = 0, own_hi = 0;
    bool own_valid = false;                 // own_cs below is current
    uint32_t own_cs[4] = {0, 0, 0, 0};      // cell_start at own_lo, end of the first owned layer, start of the last one, own_hi
    double n_test;
    double box[3];
    uint64_t seed;
    uint32_t t;          // global step index
    uint64_t steps;
    cudaStream_t stream;
    Layout lay;
    unsigned char *ws;
    Soa set[2];          // [0] caller's arrays + pidA, [1] workspace copy + pidB
    int cur;
    int grid_cls[kSmemClasses], grid_o, grid_hist, grid_scat;
    double *h_obs;       // pinned staging for observables
    cudaStream_t cls_stream[kNumClasses] = {};   // the collision classes run concurrently, fenced into `stream`
    cudaEvent_t ev_fork = nullptr, ev_join[kNumClasses] = {};
    uint32_t nmax_cur = 0;   // population of the fullest cell of the current store (variable time step, A23)
    bool nmax_valid = false; // false after steps that did not read it back
    uint32_t *h_u32 = nullptr;   // pinned word for that read-back
    bool use_graph = true;   // CUBA_OPT_GRAPH
    bool capturing = false;  // launches go into a stream capture: GRAPH kernel instantiations, no profiling marks
    cudaGraphExec_t graph_exec = nullptr;   // two steps (the store alternates between its two copies) for (graph_dt, graph_sigma)
    double graph_dt = 0.0, graph_sigma = -1.0;
    uint64_t graph_kernels = 0;             // kernel launches one replay stands for (cuba_launch_count)
    bool fuse_hist = true;   // CUBA_OPT_FUSE_HIST
    double pre_dt = 0.0;     // > 0: cnt / carry already hold the histogram of the next step for this dt
    // ---- slotted schedule (slots.cuh): one kernel per step on a store with a fixed region per cell ----
    int slot_mode = 0;            // CUBA_OPT_SLOTS: 0 never (default), 1 for calls of >= kSlotMinSteps steps, 2 for every call
    double slot_margin = 1.0;     // CUBA_OPT_SLOT_MARGIN (percent): scales the segment capacities (tests force overflows)
    double slot_boost = 1.0;      // grows after an overflow so that the next geometry is roomier
    double slot_margin_built = 0.0;   // slot_margin * slot_boost the current store was laid out with
    unsigned char *slot_mem = nullptr;   // library-owned device memory: two slotted copies + the counter backup
    size_t slot_bytes = 0;
    SlotGeom slot_geom{};
    SlotStore slot_st[2]{};
    unsigned char *slot_backup = nullptr;  // counters (64 B), max_occ (8 B), flags (4 B) at the start of the pending run
    uint32_t slot_nmax = 0;       // what the geometry was sized for
    double slot_dt = 0.0;
    int grid_slot[kSmemClasses] = {};
    bool slot_grids = false;
    bool slot_unavailable = false;   // the allocation failed once: stay on the compact path
    uint64_t slot_runs = 0, slot_replays = 0;
    // an enqueued slotted run whose overflow flag has not been read back yet: the compact copy it started
    // from is untouched (the run packs into the other copy), so it can be redone on the compact path
    bool pend = false;
    int pend_cur = 0, pend_n = 0;
    uint32_t pend_t = 0;
    uint64_t pend_steps = 0;
    double pend_dt = 0.0, pend_sigma = 0.0;
    int prof_mode = 0;   // 0 off, 1 events per kernel (collision classes as one concurrent group), 2 classes serialised
    bool prof_on = false;
    std::vector<cudaEvent_t> prof_pool;          // reused events
    std::vector<std::pair<cudaEvent_t, int>> prof_log;   // (event, group) in stream order; group -1 = step start
    template <typename T> T *at(size_t off) const { return reinterpret_cast<T *>(ws + off); }
};

// The exported functions take C linkage from their declarations in cuba.h.

const char *cuba_strerror(int code)
{
    switch (code) {
    case CUBA_OK: return "ok";
    case CUBA_ERR_NULL: return "null pointer";
    case CUBA_ERR_SIZE: return "size out of range";
    case CUBA_ERR_VALUE: return "value out of range";
    case CUBA_ERR_WORKSPACE: return "workspace too small or misaligned";
    case CUBA_ERR_CUDA: return "CUDA runtime error";
    case CUBA_ERR_STATE: return "invalid particle state";
    case CUBA_ERR_CFL: return "dt not below the smallest cell edge";
    case CUBA_ERR_MOVED: return "a particle crossed more than one cell in a step";
    case CUBA_ERR_ROUNDS: return "a cell needs more than 64 collision rounds";
    case CUBA_ERR_TRACE: return "trace capacity too small";
    case CUBA_ERR_HALO: return "halo buffer does not hold the number of particles given to cuba_slab_unpack";
    default: return "unknown error";
    }
}

const char *cuba_last_cuda_error(void) { return g_cuda_err; }
uint64_t cuba_launch_count(void) { return g_launches.load(); }

static int check_grid(int64_t n, const int ncell[3], int64_t *ncells_out)
{
    if (!ncell) return CUBA_ERR_NULL;
    if (n < 1 || n >= ((int64_t)1 << 32)) return CUBA_ERR_SIZE;
    for (int k = 0; k < 3; ++k) if (ncell[k] < 1) return CUBA_ERR_SIZE;
    const int64_t ncells = (int64_t)ncell[0] * ncell[1] * ncell[2];
    if (ncells >= ((int64_t)1 << 27)) return CUBA_ERR_SIZE;
    *ncells_out = ncells;
    return CUBA_OK;
}

size_t cuba_workspace_bytes(int64_t n, const int ncell[3])
{
    int64_t ncells;
    if (check_grid(n, ncell, &ncells) != CUBA_OK) return 0;
    return make_layout(n, ncells).total;
}

static int device_flags_to_error(uint32_t f)
{
    if (f & kFlagState) return CUBA_ERR_STATE;
    if (f & kFlagMoved) return CUBA_ERR_MOVED;
    if (f & kFlagRounds) return CUBA_ERR_ROUNDS;
    if (f & kFlagTrace) return CUBA_ERR_TRACE;
    if (f & kFlagHalo) return CUBA_ERR_HALO;
    return CUBA_OK;
}

static int sync_and_check(cuba_ctx *ctx)
{
    uint32_t f = 0;
    CU(cudaMemcpyAsync(&f, ctx->at<uint32_t>(ctx->lay.flags), 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return device_flags_to_error(f);
}

enum { G_MEMSET = 0, G_STREAM_HIST, G_GATHER, G_SCAN, G_CELL_START, G_CARRY, G_DEST_BASE, G_SCATTER, G_COLLIDE_ALL, G_COLLIDE0,
       G_SLOT_UNPACK = G_COLLIDE0 + kNumClasses, G_SLOT_CLASSIFY, G_SLOT_STEP, G_SLOT_PACK, G_END };
static_assert(G_END == CUBA_PROFILE_GROUPS, "profile groups");

static void prof_mark(cuba_ctx *ctx, int group)
{
    if (!ctx->prof_on || ctx->capturing) return;
    cudaEvent_t e;
    if (ctx->prof_pool.empty()) { if (cudaEventCreate(&e) != cudaSuccess) return; }
    else { e = ctx->prof_pool.back(); ctx->prof_pool.pop_back(); }
    cudaEventRecord(e, ctx->stream);
    ctx->prof_log.emplace_back(e, group);
}

template <typename K>
static int occupancy_grid(K kernel, int threads, size_t smem, int sms, int *grid)
{
    if (smem > 32 * 1024)
        CU(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int per_sm = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem));
    if (per_sm < 1) per_sm = 1;
    *grid = per_sm * sms;
    return CUBA_OK;
}

// cuba_init and cuba_slab_init.  cap: particles the arrays and the workspace hold; n <= cap of them are
// given.  pid_global (DEVICE, n; null: pid = index) names the particles of a slab by their index in the
// whole problem; [layer_lo, layer_hi) are the owned cell layers along x.
static int init_impl(cuba_ctx **out, const double box[3], const int ncell[3], int64_t cap, int64_t n,
                     double *x, double *y, double *z, double *px, double *py, double *pz,
                     double n_test, uint64_t seed, void *workspace, size_t workspace_bytes,
                     void *cuda_stream, const uint32_t *pid_global, int layer_lo, int layer_hi, bool slab,
                     cudaEvent_t momenta_ready = nullptr)   // non-null: px, py, pz are being written on another stream until this event
{
    if (!out || !box || !ncell || !x || !y || !z || !px || !py || !pz || !workspace) return CUBA_ERR_NULL;
    *out = nullptr;
    int64_t ncells;
    int rc = check_grid(cap, ncell, &ncells);
    if (rc != CUBA_OK) return rc;
    if (n < 1 || n > cap) return CUBA_ERR_SIZE;
    if (layer_lo < 0 || layer_hi > ncell[0] || layer_lo >= layer_hi) return CUBA_ERR_VALUE;
    for (int k = 0; k < 3; ++k) if (!(box[k] > 0.0) || !std::isfinite(box[k])) return CUBA_ERR_VALUE;
    if (!(n_test > 0.0) || !std::isfinite(n_test)) return CUBA_ERR_VALUE;
    Layout lay = make_layout(cap, ncells);
    if (workspace_bytes < lay.total || (reinterpret_cast<uintptr_t>(workspace) & 255u)) return CUBA_ERR_WORKSPACE;
    for (const double *a : {x, y, z, px, py, pz})
        if (reinterpret_cast<uintptr_t>(a) & 15u) return CUBA_ERR_WORKSPACE;   // bulk copies need 16-byte alignment

    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));

    cuba_ctx *ctx = new (std::nothrow) cuba_ctx();
    if (!ctx) return CUBA_ERR_CUDA;
    ctx->n = n; ctx->cap = cap; ctx->n_test = n_test; ctx->seed = seed; ctx->t = 0; ctx->steps = 0;
    ctx->slab = slab; ctx->layer_lo = layer_lo; ctx->layer_hi = layer_hi;
    ctx->own_lo = (uint32_t)layer_lo * (uint32_t)(ncell[1] * ncell[2]);
    ctx->own_hi = (uint32_t)layer_hi * (uint32_t)(ncell[1] * ncell[2]);
    if (slab) {          // every step is followed by a halo exchange that rebuilds the store: plain compact steps
        ctx->fuse_hist = false; ctx->use_graph = false; ctx->slot_mode = 0;
    }
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    ctx->lay = lay;
    ctx->ws = static_cast<unsigned char *>(workspace);
    for (int k = 0; k < 3; ++k) {
        ctx->box[k] = box[k];
        ctx->g.L[k] = box[k];
        ctx->g.nc[k] = ncell[k];
        ctx->g.inv_d[k] = 1.0 / (box[k] / (double)ncell[k]);
    }
    ctx->g.ncells = (uint32_t)ncells;
    ctx->set[0] = Soa{x, y, z, px, py, pz, ctx->at<uint32_t>(lay.pidA)};
    ctx->set[1] = Soa{ctx->at<double>(lay.setB[0]), ctx->at<double>(lay.setB[1]), ctx->at<double>(lay.setB[2]),
                      ctx->at<double>(lay.setB[3]), ctx->at<double>(lay.setB[4]), ctx->at<double>(lay.setB[5]),
                      ctx->at<uint32_t>(lay.pidB)};
    ctx->cur = 0;
    ctx->h_obs = nullptr;
    auto fail = [&](int code) {
        if (ctx->h_obs) cudaFreeHost(ctx->h_obs);
        if (ctx->h_u32) cudaFreeHost(ctx->h_u32);
        if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
        for (int k = 0; k < kNumClasses; ++k) {
            if (ctx->cls_stream[k]) cudaStreamDestroy(ctx->cls_stream[k]);
            if (ctx->ev_join[k]) cudaEventDestroy(ctx->ev_join[k]);
        }
        delete ctx;
        return code;
    };
    if (!cuda_ok(cudaMallocHost(&ctx->h_obs, (9 * kLrfMaxSlabs > 4 + kObsMaxSlabs ? 9 * kLrfMaxSlabs : 4 + kObsMaxSlabs) * sizeof(double)), "cudaMallocHost")) return fail(CUBA_ERR_CUDA);
    if (!cuda_ok(cudaMallocHost(&ctx->h_u32, 64), "cudaMallocHost")) return fail(CUBA_ERR_CUDA);
    if (!cuda_ok(cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming), "cudaEventCreate")) return fail(CUBA_ERR_CUDA);
    for (int k = 0; k < kNumClasses; ++k) {
        if (!cuda_ok(cudaStreamCreateWithFlags(&ctx->cls_stream[k], cudaStreamNonBlocking), "cudaStreamCreate")) return fail(CUBA_ERR_CUDA);
        if (!cuda_ok(cudaEventCreateWithFlags(&ctx->ev_join[k], cudaEventDisableTiming), "cudaEventCreate")) return fail(CUBA_ERR_CUDA);
    }

#define CUBA_OCC(K, T, I, C, MB)                                                                                          \
    if (rc == CUBA_OK) rc = occupancy_grid(k_collide<T, I, C, MB, true, false, false>, T, collide_smem_bytes(C, T, I), sms, &ctx->grid_cls[K]); \
    if (rc == CUBA_OK) rc = occupancy_grid(k_collide<T, I, C, MB, false, true, false>, T, collide_smem_bytes(C, T, I), sms, &ctx->grid_cls[K]); \
    if (rc == CUBA_OK) rc = occupancy_grid(k_collide<T, I, C, MB, false, false, true>, T, collide_smem_bytes(C, T, I), sms, &ctx->grid_cls[K]); \
    if (rc == CUBA_OK) rc = occupancy_grid(k_collide<T, I, C, MB, false, false, false>, T, collide_smem_bytes(C, T, I), sms, &ctx->grid_cls[K]);
    rc = CUBA_OK;
    CUBA_FOR_EACH_CLASS(CUBA_OCC)
#undef CUBA_OCC
    if (rc == CUBA_OK) rc = occupancy_grid(k_stream_hist, kTileThreads, 2 * sizeof(TileStage<6>), sms, &ctx->grid_hist);
    if (rc == CUBA_OK) rc = occupancy_grid(k_scatter<true>, kTileThreads, 2 * sizeof(TileStage<7>), sms, &ctx->grid_scat);
    if (rc == CUBA_OK) rc = occupancy_grid(k_scatter<false>, kTileThreads, 2 * sizeof(TileStage<7>), sms, &ctx->grid_scat);
    if (rc != CUBA_OK) return fail(rc);
#ifdef CUBA_DEBUG_KNOBS   // experiment builds only (-DCUBA_DEBUG_KNOBS): resident CTAs per SM of class 4 / of the scatter
    if (const char *e = getenv("CUBA_DEBUG_GRID_C4")) ctx->grid_cls[4] = std::max(1, atoi(e)) * sms;
    if (const char *e = getenv("CUBA_DEBUG_GRID_SCAT")) ctx->grid_scat = std::max(1, atoi(e)) * sms;
#endif
    ctx->grid_o = sms;
    if (!cuda_ok(cudaFuncSetAttribute(k_observe_partial<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      kObsWarps * kObsMaxSlabs * 8), "cudaFuncSetAttribute")) return fail(CUBA_ERR_CUDA);
    if (!cuda_ok(cudaFuncSetAttribute(k_observe_partial<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      kObsWarps * kLrfComp * kLrfMaxSlabs * 8), "cudaFuncSetAttribute")) return fail(CUBA_ERR_CUDA);
    if (!cuda_ok(cudaFuncSetAttribute(k_observe_partial<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      kObsWarps * (kObsMaxSlabs + kObsWindowMax * 32) * 8), "cudaFuncSetAttribute")) return fail(CUBA_ERR_CUDA);
    if (!cuda_ok(cudaFuncSetAttribute(k_observe_partial<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      kObsWarps * kLrfComp * (kLrfMaxSlabs + kLrfWindowMax * 32) * 8), "cudaFuncSetAttribute")) return fail(CUBA_ERR_CUDA);

    cudaStream_t st = ctx->stream;
    auto body = [&]() -> int {
        CU(cudaMemsetAsync(ctx->at<void>(lay.zero), 0, kZeroWords * 4, st));
        CU(cudaMemsetAsync(ctx->at<void>(lay.counters), 0, 64, st));
        CU(cudaMemsetAsync(ctx->at<void>(lay.flags), 0, 4, st));
        CU(cudaMemsetAsync(ctx->at<void>(lay.max_occ), 0, 8, st));
        // S3 keys + persistent ids, then the general stable sort (A19)
        uint32_t *kv = ctx->at<uint32_t>(lay.arena32);
        uint32_t *keys[2] = {kv, kv + n}, *vals[2] = {kv + 2 * n, kv + 3 * n};
        const unsigned gb = (unsigned)((n + 255) / 256);
        k_init_keys<<<gb, 256, 0, st>>>(ctx->g, n, ctx->set[0], keys[0], vals[0], ctx->at<uint32_t>(lay.flags));
        LAUNCHED();
        int bits = 0;
        while (bits < 32 && (((uint64_t)ncells - 1) >> bits) != 0) ++bits;
        const int passes = bits == 0 ? 1 : (bits + 7) / 8;
        uint32_t *H = ctx->at<uint32_t>(lay.rsH);
        const uint32_t nb = (uint32_t)((n + kRsTile - 1) / kRsTile);
        int src = 0;
        for (int p = 0; p < passes; ++p) {
            k_rs_hist<<<nb, kRsThreads, 0, st>>>(keys[src], n, 8 * p, nb, H);
            LAUNCHED();
            {
                const int64_t total = (int64_t)256 * nb;
                const unsigned nchunks = (unsigned)((total + kScanChunk - 1) / kScanChunk);
                uint32_t *sums = ctx->at<uint32_t>(lay.rsSums);
                k_chunk_sums<<<nchunks, kScanThreads, 0, st>>>(H, total, sums);
                LAUNCHED();
                k_scan_blocks<<<1, 1024, 0, st>>>(sums, (int)nchunks, nullptr, 0);
                LAUNCHED();
                k_chunk_scan<<<nchunks, kScanThreads, 0, st>>>(H, total, sums);
                LAUNCHED();
            }
            k_rs_scatter<<<nb, kRsThreads, 0, st>>>(keys[src], vals[src], keys[1 - src], vals[1 - src], n, 8 * p, nb, H);
            LAUNCHED();
            src = 1 - src;
        }
        if (momenta_ready) CU(cudaStreamWaitEvent(st, momenta_ready, 0));
        k_gather_perm<<<gb, 256, 0, st>>>(n, vals[src], ctx->set[0], ctx->set[1], ctx->at<uint32_t>(lay.flags));
        LAUNCHED();
        if (pid_global) {
            k_map_pid<<<gb, 256, 0, st>>>(n, ctx->set[1].pid, pid_global);
            LAUNCHED();
        }
        k_starts_from_sorted<<<gb, 256, 0, st>>>(n, (uint32_t)ncells, keys[src], ctx->at<uint32_t>(lay.cell_start));
        LAUNCHED();
        // hand the sorted store back to the caller's arrays: the current set is 0 after init
        const double *from[6] = {ctx->set[1].x, ctx->set[1].y, ctx->set[1].z, ctx->set[1].px, ctx->set[1].py, ctx->set[1].pz};
        double *to[6] = {x, y, z, px, py, pz};
        for (int k = 0; k < 6; ++k) CU(cudaMemcpyAsync(to[k], from[k], (size_t)n * 8, cudaMemcpyDeviceToDevice, st));
        CU(cudaMemcpyAsync(ctx->set[0].pid, ctx->set[1].pid, (size_t)n * 4, cudaMemcpyDeviceToDevice, st));
        int r = sync_and_check(ctx);
        if (r != CUBA_OK) return r;
        // fullest cell of the initial binning (start of a variable-dt run); init is synchronous anyway
        std::vector<uint32_t> start((size_t)ncells + 1);
        CU(cudaMemcpy(start.data(), ctx->at<uint32_t>(lay.cell_start), ((size_t)ncells + 1) * 4, cudaMemcpyDeviceToHost));
        uint32_t m = 0;
        for (int64_t c = 0; c < ncells; ++c) m = std::max(m, start[c + 1] - start[c]);
        ctx->nmax_cur = m; ctx->nmax_valid = true;
        return CUBA_OK;
    };
    rc = body();
    if (rc != CUBA_OK) return fail(rc);
    *out = ctx;
    return CUBA_OK;
}

int cuba_init(cuba_ctx **out, const double box[3], const int ncell[3], int64_t n,
              double *x, double *y, double *z, double *px, double *py, double *pz,
              double n_test, uint64_t seed, void *workspace, size_t workspace_bytes,
              void *cuda_stream)
{
    if (!ncell) return CUBA_ERR_NULL;
    return init_impl(out, box, ncell, n, n, x, y, z, px, py, pz, n_test, seed, workspace, workspace_bytes, cuda_stream,
                     nullptr, 0, ncell[0] > 0 ? ncell[0] : 1, false);
}

int cuba_slab_init(cuba_ctx **out, const double box[3], const int ncell[3], int64_t capacity, int64_t n,
                   double *x, double *y, double *z, double *px, double *py, double *pz, const uint32_t *pid,
                   double n_test, uint64_t seed, void *workspace, size_t workspace_bytes, void *cuda_stream,
                   int layer_lo, int layer_hi)
{
    if (!pid) return CUBA_ERR_NULL;
    return init_impl(out, box, ncell, capacity, n, x, y, z, px, py, pz, n_test, seed, workspace, workspace_bytes, cuda_stream,
                     pid, layer_lo, layer_hi, true);
}

void cuba_destroy(cuba_ctx *ctx)
{
    if (!ctx) return;
    cudaStreamSynchronize(ctx->stream);
    if (ctx->graph_exec) cudaGraphExecDestroy(ctx->graph_exec);
    if (ctx->slot_mem) cudaFree(ctx->slot_mem);
    if (ctx->h_obs) cudaFreeHost(ctx->h_obs);
    if (ctx->h_u32) cudaFreeHost(ctx->h_u32);
    for (int k = 0; k < kNumClasses; ++k) {
        if (ctx->cls_stream[k]) { cudaStreamSynchronize(ctx->cls_stream[k]); cudaStreamDestroy(ctx->cls_stream[k]); }
        if (ctx->ev_join[k]) cudaEventDestroy(ctx->ev_join[k]);
    }
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    for (auto &pe : ctx->prof_log) cudaEventDestroy(pe.first);
    for (auto e : ctx->prof_pool) cudaEventDestroy(e);
    delete ctx;
}

// trace device buffers (cuba_step_traced only)
struct TraceDev {
    unsigned long long *off = nullptr;
    uint32_t *cell = nullptr, *round = nullptr, *pa = nullptr, *pb = nullptr, *cell_of_pid = nullptr;
    double *P = nullptr, *u = nullptr;
    uint8_t *dec = nullptr;
};

template <bool TRACE>
static int launch_collide(cuba_ctx *ctx, double base, const TraceDev *td, double next_dt, double etas = 0.0, double dt = 0.0)
{
    const Layout &lay = ctx->lay;
    Soa &cur = ctx->set[ctx->cur];
    CollideParams P{};
    P.seed = ctx->seed; P.t = ctx->t; P.base = base;
    P.next_dt = next_dt; P.g = ctx->g;
    P.etas = etas; P.dt = dt;
    P.t_dev = ctx->capturing ? ctx->at<uint32_t>(lay.tdev) : nullptr;
    P.x = cur.x; P.y = cur.y; P.z = cur.z;
    P.cnt = ctx->at<uint32_t>(lay.cnt); P.carry = ctx->at<uint32_t>(lay.carry);
    if (next_dt > 0.0) {      // the scatter of this step has consumed the offsets; empty cells must read as zero
        CU(cudaMemsetAsync(P.cnt, 0, (size_t)kDirs * ctx->g.ncells * 4, ctx->stream));
        prof_mark(ctx, G_MEMSET);
    }
    for (uint32_t r = 0; r < 10; ++r) {               // Philox4x32-10 key schedule (Salmon et al., SC'11)
        P.rk[2 * r] = (uint32_t)ctx->seed + r * 0x9E3779B9u;
        P.rk[2 * r + 1] = (uint32_t)(ctx->seed >> 32) + r * 0xBB67AE85u;
    }
    P.cell_start = ctx->at<uint32_t>(lay.cell_start);
    P.px = cur.px; P.py = cur.py; P.pz = cur.pz; P.pid = cur.pid;
    P.counters = ctx->at<unsigned long long>(lay.counters);
    P.flags = ctx->at<uint32_t>(lay.flags);
    P.arena = ctx->at<uint32_t>(lay.arena32);
    if (TRACE) {
        P.trace_off = td->off; P.tr_cell = td->cell; P.tr_round = td->round; P.tr_pa = td->pa; P.tr_pb = td->pb;
        P.tr_P = td->P; P.tr_u = td->u; P.tr_dec = td->dec;
    }
    uint32_t *zero = ctx->at<uint32_t>(lay.zero);
    uint4 *lists = ctx->at<uint4>(lay.class_list);
    auto cls = [&](int k) { P.list = lists + (size_t)k * ctx->g.ncells; P.list_count = zero + k; P.work = zero + 8 + k; };
    // The classes are independent (disjoint cells): fork them onto their own streams so that
    // small classes fill the tail of the big ones, then join back into the caller's stream.
    // Profile mode 2 serialises them on the caller's stream to time each class by itself.
    const bool serial = ctx->prof_mode == 2;
    cudaStream_t main = ctx->stream;
    if (!serial) CU(cudaEventRecord(ctx->ev_fork, main));
#define CUBA_LAUNCH(K, T, I, C, MB)                                                              \
    {                                                                                            \
        cudaStream_t st = serial ? main : ctx->cls_stream[K];                                    \
        if (!serial) CU(cudaStreamWaitEvent(st, ctx->ev_fork, 0));                               \
        cls(K);                                                                                  \
        if (!TRACE && ctx->capturing) k_collide<T, I, C, MB, false, false, true><<<ctx->grid_cls[K], T, collide_smem_bytes(C, T, I), st>>>(P); \
        else if (!TRACE && etas > 0.0) k_collide<T, I, C, MB, false, true, false><<<ctx->grid_cls[K], T, collide_smem_bytes(C, T, I), st>>>(P); \
        else k_collide<T, I, C, MB, TRACE, false, false><<<ctx->grid_cls[K], T, collide_smem_bytes(C, T, I), st>>>(P);    \
        LAUNCHED();                                                                              \
        if (serial) prof_mark(ctx, G_COLLIDE0 + K);                                              \
        else { CU(cudaEventRecord(ctx->ev_join[K], st)); CU(cudaStreamWaitEvent(main, ctx->ev_join[K], 0)); } \
    }
    CUBA_FOR_EACH_CLASS(CUBA_LAUNCH)
#undef CUBA_LAUNCH
    {
        cudaStream_t st = serial ? main : ctx->cls_stream[kSmemClasses];
        if (!serial) CU(cudaStreamWaitEvent(st, ctx->ev_fork, 0));
        cls(kSmemClasses);
        k_collide_overflow<TRACE><<<ctx->grid_o, 1024, 0, st>>>(P, reinterpret_cast<unsigned long long *>(zero + 16),
                                                               ctx->at<double>(lay.arenaE));
        LAUNCHED();
        if (serial) prof_mark(ctx, G_COLLIDE0 + kSmemClasses);
        else { CU(cudaEventRecord(ctx->ev_join[kSmemClasses], st)); CU(cudaStreamWaitEvent(main, ctx->ev_join[kSmemClasses], 0)); }
    }
    if (!serial) prof_mark(ctx, G_COLLIDE_ALL);
    return CUBA_OK;
}

static int check_step_args(const cuba_ctx *ctx, double dt, double sigma, double *base)
{
    if (!(dt > 0.0) || !std::isfinite(dt) || !(sigma >= 0.0) || !std::isfinite(sigma)) return CUBA_ERR_VALUE;
    const double dx = ctx->box[0] / (double)ctx->g.nc[0];
    const double dy = ctx->box[1] / (double)ctx->g.nc[1];
    const double dz = ctx->box[2] / (double)ctx->g.nc[2];
    const double dmin = std::fmin(dx, std::fmin(dy, dz));
    if (!(dt < dmin)) return CUBA_ERR_CFL;
    const double V = (dx * dy) * dz;
    *base = (sigma * dt) / (ctx->n_test * V);         // Eq. 3 without v_rel; A3
    return CUBA_OK;
}

// S1-S4 of one step: leaves the streamed, cell-sorted store in set[1-cur] and flips cur
static int enqueue_bin(cuba_ctx *ctx, double dt, uint32_t *cell_of_pid)
{
    const Layout &lay = ctx->lay;
    cudaStream_t st = ctx->stream;
    const int64_t n = ctx->n;
    const int64_t ntiles = (n + kTile - 1) / kTile;      // (the layout is sized for the capacity)
    const uint32_t ncells = ctx->g.ncells;
    Soa &in = ctx->set[ctx->cur], &outp = ctx->set[1 - ctx->cur];
    uint32_t *cnt = ctx->at<uint32_t>(lay.cnt);
    uint32_t *zero = ctx->at<uint32_t>(lay.zero);
    const bool have_hist = ctx->pre_dt > 0.0 && ctx->pre_dt == dt;   // written by the previous step's collision kernel
    ctx->pre_dt = 0.0;
    prof_mark(ctx, -1);
    if (!have_hist) {
        CU(cudaMemsetAsync(cnt, 0, (size_t)kDirs * ncells * 4, st));
        prof_mark(ctx, G_MEMSET);
        k_stream_hist<<<ctx->grid_hist, kTileThreads, 2 * sizeof(TileStage<6>), st>>>(ctx->g, dt, n, ntiles, in, cnt, ctx->at<uint32_t>(lay.tile_rec),
                                                                      ctx->at<uint32_t>(lay.flags));
        LAUNCHED();
        prof_mark(ctx, G_STREAM_HIST);
    }
    k_gather<<<(unsigned)lay.nblocks_cells, kGatherThreads, 0, st>>>(ctx->g, cnt, ctx->at<uint32_t>(lay.count_new),
                                                          ctx->at<uint32_t>(lay.block_sum));
    LAUNCHED();
    prof_mark(ctx, G_GATHER);
    k_scan_blocks<<<1, 1024, 0, st>>>(ctx->at<uint32_t>(lay.block_sum), (int)lay.nblocks_cells, zero, kZeroWords);
    LAUNCHED();
    prof_mark(ctx, G_SCAN);
    ClassTable ct{};
#define CUBA_CAP(K, T, I, C, MB) ct.max_n[K] = C;
    CUBA_FOR_EACH_CLASS(CUBA_CAP)
#undef CUBA_CAP
    ct.max_n[kSmemClasses] = 0xFFFFFFFFu;
    ct.c_lo = ctx->own_lo; ct.c_hi = ctx->own_hi;
    k_cell_start<<<(unsigned)lay.nblocks_cells, 256, 0, st>>>(ncells, ctx->at<uint32_t>(lay.count_new),
                                                              ctx->at<uint32_t>(lay.block_sum), ctx->at<uint32_t>(lay.cell_start),
                                                              ct, zero, ctx->at<uint4>(lay.class_list),
                                                              ctx->at<unsigned long long>(lay.max_occ), zero + kStepMaxWord);
    LAUNCHED();
    prof_mark(ctx, G_CELL_START);
    if (!have_hist) {
        k_carry<<<(unsigned)((ntiles + 7) / 8), 256, 0, st>>>((int)ntiles, ctx->at<uint32_t>(lay.tile_rec),
                                                                  ctx->at<uint32_t>(lay.carry));
        LAUNCHED();
        prof_mark(ctx, G_CARRY);
    }
    k_dest_base<<<dim3((unsigned)lay.nblocks_cells, kDirs), 256, 0, st>>>(ctx->g, cnt, ctx->at<uint32_t>(lay.cell_start));
    LAUNCHED();
    prof_mark(ctx, G_DEST_BASE);
    if (cell_of_pid)
        k_scatter<true><<<ctx->grid_scat, kTileThreads, 2 * sizeof(TileStage<7>), st>>>(ctx->g, dt, n, ntiles, in, outp, cnt,
                                                                       ctx->at<uint32_t>(lay.carry), cell_of_pid);
    else
        k_scatter<false><<<ctx->grid_scat, kTileThreads, 2 * sizeof(TileStage<7>), st>>>(ctx->g, dt, n, ntiles, in, outp, cnt,
                                                                        ctx->at<uint32_t>(lay.carry), nullptr);
    LAUNCHED();
    prof_mark(ctx, G_SCATTER);
    ctx->cur = 1 - ctx->cur;
    return CUBA_OK;
}

// fixed time step; etas > 0 selects the local cross section (sigma is then unused)
// one step by plain launches (also what a stream capture records)
static int step_once(cuba_ctx *ctx, double dt, double base, double etas)
{
    int rc = enqueue_bin(ctx, dt, nullptr);
    if (rc != CUBA_OK) return rc;
    const double next_dt = ctx->fuse_hist ? dt : 0.0;
    rc = launch_collide<false>(ctx, base, nullptr, next_dt, etas, dt);
    if (rc != CUBA_OK) return rc;
    ctx->pre_dt = next_dt;
    return CUBA_OK;
}

static void graph_drop(cuba_ctx *ctx)
{
    if (ctx->graph_exec) cudaGraphExecDestroy(ctx->graph_exec);
    ctx->graph_exec = nullptr;
    ctx->graph_sigma = -1.0;
}

// Small problems are bound by the host cost of the ~13 launches and the stream fork/join of a
// step, not by device time (78 us per step at 13.8k particles).  In the steady state of the fused
// schedule two consecutive steps differ only in which copy of the store is read and in the step
// index, so TWO steps are captured once into a CUDA graph (step index read from device memory and
// bumped by a one-thread kernel after each step) and replayed.
constexpr int64_t kGraphMaxParticles = 1 << 20;

static int graph_capture(cuba_ctx *ctx, double dt, double sigma, double base)
{
    graph_drop(ctx);
    const int cur0 = ctx->cur;
    const double pre0 = ctx->pre_dt;
    const uint64_t l0 = g_launches.load();
    cudaGraph_t graph = nullptr;
    uint32_t *t_dev = ctx->at<uint32_t>(ctx->lay.tdev);
    CU(cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal));
    ctx->capturing = true;
    int rc = CUBA_OK;
    for (int k = 0; k < 2 && rc == CUBA_OK; ++k) {
        rc = step_once(ctx, dt, base, 0.0);
        if (rc == CUBA_OK) { k_bump_t<<<1, 1, 0, ctx->stream>>>(t_dev); g_launches.fetch_add(1, std::memory_order_relaxed); }
    }
    ctx->capturing = false;
    const cudaError_t e = cudaStreamEndCapture(ctx->stream, &graph);
    ctx->graph_kernels = g_launches.load() - l0;
    g_launches.store(l0);                       // nothing has run yet
    ctx->cur = cur0; ctx->pre_dt = pre0;        // two steps bring both back to where they were
    if (rc != CUBA_OK || !cuda_ok(e, "cudaStreamEndCapture")) {
        if (graph) cudaGraphDestroy(graph);
        return rc != CUBA_OK ? rc : CUBA_ERR_CUDA;
    }
    const bool ok = cuda_ok(cudaGraphInstantiate(&ctx->graph_exec, graph, 0), "cudaGraphInstantiate");
    cudaGraphDestroy(graph);
    if (!ok) { ctx->graph_exec = nullptr; return CUBA_ERR_CUDA; }
    ctx->graph_dt = dt; ctx->graph_sigma = sigma;
    return CUBA_OK;
}


// ---- slotted schedule (slots.cuh) ---------------------------------------------------------------
// A call of cuba_step with enough steps converts the compact store into the slotted one (k_slot_unpack),
// runs the steps as one kernel per step and size class (k_slot_step), and converts back (k_slot_pack)
// into the OTHER compact copy.  The copy the run started from is left untouched until the run has been
// verified (no segment overflowed: kFlagSlots clear) at the next synchronising call; if the flag is
// set the run is redone from that copy on the compact path -- the results never depend on the
// capacities.  All of it is stream-ordered; only the verification synchronises.
constexpr int kSlotMinSteps = 4;        // below this the two conversion passes cost more than they save
constexpr size_t kSlotBackupBytes = 128;

// Capacities of the 27 inbox segments for cells of up to nmax particles and time step dt.  A massless
// particle moves dt in a step, so the share of a cell that leaves through a face is 1/4 dt/d for an
// isotropic distribution (dt/d if everything flies the same way), through an edge or a corner the
// product of two or three such factors.  Sized for twice the isotropic share plus six standard
// deviations plus a constant; the stay segment for nmax plus an eighth.  An overflow is not an
// error (see above), only slow.
static SlotGeom slot_geometry(const cuba_ctx *ctx, uint32_t nmax, double dt, double margin)
{
    SlotGeom sg{};
    double r[3];
    for (int k = 0; k < 3; ++k) r[k] = dt * ctx->g.inv_d[k];
    uint32_t off = 0;
    for (int s = 0; s < kDirs; ++s) {
        const int o[3] = {s / 9 - 1, (s / 3) % 3 - 1, s % 3 - 1};
        int m = 0;
        double frac = 1.0;
        for (int k = 0; k < 3; ++k) if (o[k] != 0) { ++m; frac *= r[k]; }
        double want;
        if (m == 0) want = 1.125 * (double)nmax + 64.0;
        else {
            const double mean = (m == 1 ? 0.5 : (m == 2 ? 0.25 : 0.125)) * frac * (double)nmax;
            want = mean + 6.0 * std::sqrt(mean) + (m == 1 ? 16.0 : 8.0);
        }
        uint32_t cap = (uint32_t)std::ceil(want * margin);
        cap = std::max(cap, 4u);
        cap = (cap + 3u) / 4u * 4u;                      // 32-byte sectors of the fp64 arrays
        if (s == (int)kDirStay) off = (off + 15u) / 16u * 16u;   // the big segment starts on a 128-byte line
        sg.seg_off[s] = off;
        off += cap;
    }
    sg.seg_off[kDirs] = off;
    sg.slots = (off + 15u) / 16u * 16u;
    return sg;
}

static void slot_release(cuba_ctx *ctx)
{
    if (ctx->slot_mem) cudaFree(ctx->slot_mem);
    ctx->slot_mem = nullptr; ctx->slot_bytes = 0; ctx->slot_nmax = 0; ctx->slot_dt = 0.0; ctx->slot_margin_built = 0.0;
}

// Make sure a slotted store fit for (nmax, dt) exists.  Returns false (and leaves the compact path in
// charge) when it cannot be had.
static bool slot_prepare(cuba_ctx *ctx, uint32_t nmax, double dt)
{
    if (ctx->slot_unavailable) return false;
    const double margin = ctx->slot_margin * ctx->slot_boost;
    // reuse the store only if it was laid out with at least the margin asked for now: after a run outgrew a
    // segment settle() raises slot_boost, and the next call must get the roomier geometry, not the old one
    if (ctx->slot_mem && nmax <= ctx->slot_nmax && dt <= ctx->slot_dt && margin <= ctx->slot_margin_built) return true;
    slot_release(ctx);
    const uint32_t size_n = nmax + nmax / 16u;             // a little head room so that small fluctuations do not reallocate
    const SlotGeom sg = slot_geometry(ctx, size_n, dt, margin);
    const uint64_t total_slots = (uint64_t)ctx->g.ncells * sg.slots;
    if (total_slots >= (1ull << 32)) { ctx->slot_unavailable = true; return false; }
    const size_t arr8 = align_up((size_t)total_slots * 8), arr4 = align_up((size_t)total_slots * 4);
    const size_t cntb = align_up((size_t)ctx->g.ncells * kDirs * 4);
    const size_t per_copy = 6 * arr8 + arr4 + cntb;
    const size_t bytes = 2 * per_copy + kSlotBackupBytes;
    void *mem = nullptr;
    if (cudaMalloc(&mem, bytes) != cudaSuccess) {
        cudaGetLastError();                                // not an error of the step
        ctx->slot_unavailable = true;
        return false;
    }
    ctx->slot_mem = static_cast<unsigned char *>(mem);
    ctx->slot_bytes = bytes;
    for (int c = 0; c < 2; ++c) {
        unsigned char *b = ctx->slot_mem + (size_t)c * per_copy;
        SlotStore &st = ctx->slot_st[c];
        double **arr[6] = {&st.x, &st.y, &st.z, &st.px, &st.py, &st.pz};
        for (int k = 0; k < 6; ++k) *arr[k] = reinterpret_cast<double *>(b + (size_t)k * arr8);
        st.pid = reinterpret_cast<uint32_t *>(b + 6 * arr8);
        st.cnt = reinterpret_cast<uint32_t *>(b + 6 * arr8 + arr4);
        // counts of segments whose source cell lies outside the box are never written: they stay zero
        if (cudaMemsetAsync(st.cnt, 0, cntb, ctx->stream) != cudaSuccess) { cudaGetLastError(); slot_release(ctx); ctx->slot_unavailable = true; return false; }
    }
    ctx->slot_backup = ctx->slot_mem + 2 * per_copy;
    ctx->slot_geom = sg;
    ctx->slot_nmax = size_n;
    ctx->slot_dt = dt;
    ctx->slot_margin_built = margin;
    return true;
}

static int slot_grids(cuba_ctx *ctx)
{
    if (ctx->slot_grids) return CUBA_OK;
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    int rc = CUBA_OK;
#define CUBA_OCC(K, T, I, C, MB) \
    if (rc == CUBA_OK) rc = occupancy_grid(k_slot_step<T, I, C, MB, kSlotFirst>, T, collide_smem_bytes(C, T, I), sms, &ctx->grid_slot[K]); \
    if (rc == CUBA_OK) rc = occupancy_grid(k_slot_step<T, I, C, MB, kSlotLast>, T, collide_smem_bytes(C, T, I), sms, &ctx->grid_slot[K]); \
    if (rc == CUBA_OK) rc = occupancy_grid(k_slot_step<T, I, C, MB, kSlotMiddle>, T, collide_smem_bytes(C, T, I), sms, &ctx->grid_slot[K]);
    CUBA_FOR_EACH_CLASS(CUBA_OCC)
#undef CUBA_OCC
    if (rc == CUBA_OK) ctx->slot_grids = true;
    return rc;
}

// nsteps steps on the slotted store, from and back to the compact one: nsteps + 1 passes (slots.cuh).
// Preconditions: no pending run, slot_prepare() succeeded.
static int slot_run(cuba_ctx *ctx, int nsteps, double dt, double sigma, double base)
{
    const Layout &lay = ctx->lay;
    cudaStream_t main = ctx->stream;
    const uint32_t ncells = ctx->g.ncells;
    int rc = slot_grids(ctx);
    if (rc != CUBA_OK) return rc;
    uint32_t *zero = ctx->at<uint32_t>(lay.zero);
    uint32_t *flags = ctx->at<uint32_t>(lay.flags);
    uint4 *lists = ctx->at<uint4>(lay.class_list);
    uint32_t *cell_start = ctx->at<uint32_t>(lay.cell_start);
    // what a replay needs: counters and flags as they are now, and where the state is
    CU(cudaMemcpyAsync(ctx->slot_backup, ctx->at<void>(lay.counters), 64, cudaMemcpyDeviceToDevice, main));
    CU(cudaMemcpyAsync(ctx->slot_backup + 64, ctx->at<void>(lay.max_occ), 8, cudaMemcpyDeviceToDevice, main));
    CU(cudaMemcpyAsync(ctx->slot_backup + 72, flags, 4, cudaMemcpyDeviceToDevice, main));
    ctx->pend = true; ctx->pend_cur = ctx->cur; ctx->pend_n = nsteps; ctx->pend_t = ctx->t; ctx->pend_steps = ctx->steps;
    ctx->pend_dt = dt; ctx->pend_sigma = sigma;
    ctx->slot_runs += 1;
    ctx->pre_dt = 0.0;

    ClassTable ct{};
#define CUBA_CAP(K, T, I, C, MB) ct.max_n[K] = C;
    CUBA_FOR_EACH_CLASS(CUBA_CAP)
#undef CUBA_CAP
    ct.max_n[kSmemClasses] = 0xFFFFFFFFu;
    ct.c_lo = 0; ct.c_hi = ncells;

    CollideParams P{};
    P.seed = ctx->seed; P.base = base; P.g = ctx->g;
    for (uint32_t r = 0; r < 10; ++r) {
        P.rk[2 * r] = (uint32_t)ctx->seed + r * 0x9E3779B9u;
        P.rk[2 * r + 1] = (uint32_t)(ctx->seed >> 32) + r * 0xBB67AE85u;
    }
    P.counters = ctx->at<unsigned long long>(lay.counters);
    P.flags = flags;
    SlotParams Q{};
    Q.sg = ctx->slot_geom; Q.dt = dt;
    const bool serial = ctx->prof_mode == 2;
    const Soa &from = ctx->set[ctx->cur], &to = ctx->set[1 - ctx->cur];
    const SlotStore compact_in{from.x, from.y, from.z, from.px, from.py, from.pz, from.pid, nullptr};
    const SlotStore compact_out{to.x, to.y, to.z, to.px, to.py, to.pz, to.pid, nullptr};

    // the size classes of one pass, forked onto their own streams
    auto launch_pass = [&](int mode) -> int {
        if (!serial) CU(cudaEventRecord(ctx->ev_fork, main));
#define CUBA_LAUNCH(K, T, I, C, MB)                                                              \
        {                                                                                        \
            cudaStream_t st = serial ? main : ctx->cls_stream[K];                                \
            if (!serial) CU(cudaStreamWaitEvent(st, ctx->ev_fork, 0));                           \
            P.list = lists + (size_t)K * ncells; P.list_count = zero + K; P.work = zero + 8 + K; \
            const size_t sm = collide_smem_bytes(C, T, I);                                       \
            if (mode == kSlotFirst) k_slot_step<T, I, C, MB, kSlotFirst><<<ctx->grid_slot[K], T, sm, st>>>(P, Q); \
            else if (mode == kSlotLast) k_slot_step<T, I, C, MB, kSlotLast><<<ctx->grid_slot[K], T, sm, st>>>(P, Q); \
            else k_slot_step<T, I, C, MB, kSlotMiddle><<<ctx->grid_slot[K], T, sm, st>>>(P, Q);  \
            LAUNCHED();                                                                          \
            if (serial) prof_mark(ctx, G_COLLIDE0 + K);                                          \
            else { CU(cudaEventRecord(ctx->ev_join[K], st)); CU(cudaStreamWaitEvent(main, ctx->ev_join[K], 0)); } \
        }
        CUBA_FOR_EACH_CLASS(CUBA_LAUNCH)
#undef CUBA_LAUNCH
        return CUBA_OK;
    };

    prof_mark(ctx, -1);
    k_slot_init_counts<<<(ncells * kDirs + 255u) / 256u, 256, 0, main>>>(ncells, cell_start, ctx->slot_geom, ctx->slot_st[0].cnt);
    LAUNCHED();
    int par = 0;
    for (int pass = 0; pass <= nsteps; ++pass) {
        const int mode = pass == 0 ? kSlotFirst : (pass == nsteps ? kSlotLast : kSlotMiddle);
        if (pass > 0) prof_mark(ctx, -1);
        CU(cudaMemsetAsync(zero, 0, kZeroWords * 4, main));
        k_slot_classify<<<(unsigned)lay.nblocks_cells, 256, 0, main>>>(ctx->g, ctx->slot_st[par].cnt, ctx->slot_st[1 - par].cnt, ct, zero, lists,
                                                                         ctx->at<unsigned long long>(lay.max_occ), zero + kStepMaxWord, flags,
                                                                         mode == kSlotFirst ? cell_start : nullptr);
        LAUNCHED();
        if (mode == kSlotLast) {
            // collisions move nobody: the compact layout of the result is known before the last pass
            k_slot_count<<<(unsigned)lay.nblocks_cells, 256, 0, main>>>(ncells, ctx->slot_st[par].cnt, ctx->at<uint32_t>(lay.count_new),
                                                                          ctx->at<uint32_t>(lay.block_sum));
            LAUNCHED();
            k_scan_blocks<<<1, 1024, 0, main>>>(ctx->at<uint32_t>(lay.block_sum), (int)lay.nblocks_cells, zero, kZeroWords);
            LAUNCHED();
            k_cell_start<<<(unsigned)lay.nblocks_cells, 256, 0, main>>>(ncells, ctx->at<uint32_t>(lay.count_new), ctx->at<uint32_t>(lay.block_sum),
                                                                          cell_start, ct, zero, lists,
                                                                          ctx->at<unsigned long long>(lay.max_occ), zero + kStepMaxWord);
            LAUNCHED();
        }
        prof_mark(ctx, G_SLOT_CLASSIFY);
        P.t = ctx->t + (uint32_t)(pass > 0 ? pass - 1 : 0);
        Q.in = mode == kSlotFirst ? compact_in : ctx->slot_st[par];
        Q.out = mode == kSlotLast ? compact_out : ctx->slot_st[1 - par];
        rc = launch_pass(mode);
        if (rc != CUBA_OK) return rc;
        if (!serial) prof_mark(ctx, mode == kSlotFirst ? G_SLOT_UNPACK : (mode == kSlotLast ? G_SLOT_PACK : G_SLOT_STEP));
        par = 1 - par;
    }
    ctx->cur = 1 - ctx->cur;
    ctx->t += (uint32_t)nsteps; ctx->steps += (uint64_t)nsteps; ctx->nmax_valid = false;
    return CUBA_OK;
}

static int step_fixed(cuba_ctx *ctx, int nsteps, double dt, double sigma, double etas);
static int read_step_max(cuba_ctx *ctx);

// Verify a pending slotted run (see above).  Called at the start of every entry point that reads or
// advances the state.  Synchronises only when a run is pending.
static int settle(cuba_ctx *ctx)
{
    if (!ctx->pend) return CUBA_OK;
    const Layout &lay = ctx->lay;
    uint32_t *h = ctx->h_u32;
    CU(cudaMemcpyAsync(h, ctx->at<uint32_t>(lay.flags), 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaMemcpyAsync(h + 1, ctx->at<uint32_t>(lay.zero) + kStepMaxWord, 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->pend = false;
    if (!(h[0] & kFlagSlots)) {
        ctx->nmax_cur = h[1]; ctx->nmax_valid = true;    // k_cell_start of the conversion recorded it
        return CUBA_OK;
    }
    // a segment (or a cell) outgrew the layout: restore the starting point and redo the run on the compact path
    ctx->slot_replays += 1;
    ctx->slot_boost *= 1.5;
    CU(cudaMemcpyAsync(ctx->at<void>(lay.counters), ctx->slot_backup, 64, cudaMemcpyDeviceToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->at<void>(lay.max_occ), ctx->slot_backup + 64, 8, cudaMemcpyDeviceToDevice, ctx->stream));
    CU(cudaMemcpyAsync(ctx->at<void>(lay.flags), ctx->slot_backup + 72, 4, cudaMemcpyDeviceToDevice, ctx->stream));
    ctx->cur = ctx->pend_cur; ctx->t = ctx->pend_t; ctx->steps = ctx->pend_steps;
    ctx->pre_dt = 0.0; ctx->nmax_valid = false;
    const int mode = ctx->slot_mode;
    ctx->slot_mode = 0;
    const int rc = step_fixed(ctx, ctx->pend_n, ctx->pend_dt, ctx->pend_sigma, 0.0);
    ctx->slot_mode = mode;
    return rc;
}

// fixed time step; etas > 0 selects the local cross section (sigma is then unused)
static int step_fixed(cuba_ctx *ctx, int nsteps, double dt, double sigma, double etas)
{
    if (!ctx) return CUBA_ERR_NULL;
    if (nsteps < 0) return CUBA_ERR_SIZE;
    if (ctx->slab && nsteps > 1) return CUBA_ERR_VALUE;     // a halo exchange belongs between two steps of a slab
    double base;
    int rc = check_step_args(ctx, dt, sigma, &base);
    if (rc != CUBA_OK) return rc;
    rc = settle(ctx);
    if (rc != CUBA_OK) return rc;
    ctx->own_valid = false;
    int s = 0;
    auto plain = [&]() -> int {
        const int r = step_once(ctx, dt, base, etas);
        if (r != CUBA_OK) return r;
        ctx->t += 1; ctx->steps += 1; ctx->nmax_valid = false; ++s;
        return CUBA_OK;
    };
    // the legacy default stream (0, cudaStreamLegacy) and cudaStreamPerThread cannot be captured
    const bool graphable = ctx->use_graph && ctx->fuse_hist && !ctx->prof_on && etas == 0.0 && ctx->n <= kGraphMaxParticles &&
                           reinterpret_cast<uintptr_t>(ctx->stream) > 2;
    // Slotted schedule: one kernel per step (slots.cuh).  Small problems are launch-bound and keep the graph.
    if (etas == 0.0 && ctx->slot_mode != 0 && !ctx->capturing && nsteps >= (ctx->slot_mode == 2 ? 1 : kSlotMinSteps) &&
        (ctx->slot_mode == 2 || !(graphable && nsteps >= 4))) {
        if (!ctx->nmax_valid) { rc = read_step_max(ctx); if (rc != CUBA_OK) return rc; }
        uint32_t cap_max = 0;
#define CUBA_CAPMAX(K, T, I, C, MB) cap_max = cap_max > (uint32_t)C ? cap_max : (uint32_t)C;
        CUBA_FOR_EACH_CLASS(CUBA_CAPMAX)
#undef CUBA_CAPMAX
        if (ctx->nmax_cur >= 1u && ctx->nmax_cur + ctx->nmax_cur / 8u <= cap_max && slot_prepare(ctx, ctx->nmax_cur, dt))
            return slot_run(ctx, nsteps, dt, sigma, base);
    }
    if (graphable && nsteps >= 4) {
        // reach the steady state the graph was captured in: histogram prepared for this dt, store in copy 0
        while (s < nsteps && !(ctx->pre_dt == dt && ctx->cur == 0)) { rc = plain(); if (rc != CUBA_OK) return rc; }
        if (nsteps - s >= 2) {
            if (!ctx->graph_exec || ctx->graph_dt != dt || ctx->graph_sigma != sigma) {
                // a stream that is already being captured by the caller cannot host a second capture
                cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
                if (cudaStreamIsCapturing(ctx->stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone ||
                    graph_capture(ctx, dt, sigma, base) != CUBA_OK) {
                    cudaGetLastError();          // not an error of the step: fall back to plain launches for good
                    graph_drop(ctx);
                    ctx->use_graph = false;
                }
            }
            if (ctx->graph_exec) {
                k_set_t<<<1, 1, 0, ctx->stream>>>(ctx->at<uint32_t>(ctx->lay.tdev), ctx->t);
                LAUNCHED();
                for (; nsteps - s >= 2; s += 2) {
                    CU(cudaGraphLaunch(ctx->graph_exec, ctx->stream));
                    g_launches.fetch_add(ctx->graph_kernels, std::memory_order_relaxed);
                    ctx->t += 2; ctx->steps += 2;
                }
                ctx->nmax_valid = false;
            }
        }
    }
    while (s < nsteps) { rc = plain(); if (rc != CUBA_OK) return rc; }
    return CUBA_OK;
}

int cuba_step(cuba_ctx *ctx, int nsteps, double dt, double sigma)
{
    return step_fixed(ctx, nsteps, dt, sigma, 0.0);
}

int cuba_step_local_sigma(cuba_ctx *ctx, int nsteps, double dt, double eta_over_s)
{
    if (!(eta_over_s > 0.0) || !std::isfinite(eta_over_s)) return ctx ? CUBA_ERR_VALUE : CUBA_ERR_NULL;
    return step_fixed(ctx, nsteps, dt, 0.0, eta_over_s);
}

// Variable time step, reading A23: the same fp64 expression, in the same order, as the oracle's.
static double adaptive_dt(const cuba_ctx *ctx, uint32_t nmax, double dt_max, double sigma)
{
    if (nmax < 2u || !(sigma > 0.0)) return dt_max;
    const double dx = ctx->box[0] / (double)ctx->g.nc[0];
    const double dy = ctx->box[1] / (double)ctx->g.nc[1];
    const double dz = ctx->box[2] / (double)ctx->g.nc[2];
    const double V = (dx * dy) * dz;
    const double cn = (nmax & 1u) ? (double)nmax : (double)(nmax - 1u);
    const double g = sigma / (ctx->n_test * V);
    const double lim = 0.9990234375 / ((2.0 * cn) * g);   // 1 - 2^-10
    return lim < dt_max ? lim : dt_max;
}

static int read_step_max(cuba_ctx *ctx)
{
    CU(cudaMemcpyAsync(ctx->h_u32, ctx->at<uint32_t>(ctx->lay.zero) + kStepMaxWord, 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->nmax_cur = *ctx->h_u32;
    ctx->nmax_valid = true;
    return CUBA_OK;
}

int cuba_step_adaptive(cuba_ctx *ctx, int nsteps, double dt_max, double sigma, double *dt_used, double *elapsed)
{
    if (!ctx) return CUBA_ERR_NULL;
    if (nsteps < 0) return CUBA_ERR_SIZE;
    if (ctx->slab) return CUBA_ERR_VALUE;      // the rule needs the fullest cell of ALL slabs: not built
    if (!(dt_max > 0.0) || !std::isfinite(dt_max) || !(sigma >= 0.0) || !std::isfinite(sigma)) return CUBA_ERR_VALUE;
    double sum = 0.0;
    int rc = settle(ctx);
    if (rc != CUBA_OK) { if (elapsed) *elapsed = 0.0; return rc; }
    if (nsteps > 0 && !ctx->nmax_valid) {      // the last binning's value is still on the device
        rc = read_step_max(ctx);
        if (rc != CUBA_OK) return rc;
    }
    // *elapsed is written on every return path: the time covered by the steps that completed
    auto done = [&](int code) { if (elapsed) *elapsed = sum; return code; };
    for (int s = 0; s < nsteps; ++s) {
        const double dt = adaptive_dt(ctx, ctx->nmax_cur, dt_max, sigma);
        double base;
        rc = check_step_args(ctx, dt, sigma, &base);
        if (rc != CUBA_OK) return done(rc);
        rc = enqueue_bin(ctx, dt, nullptr);
        if (rc != CUBA_OK) return done(rc);
        // the fullest cell of the new binning fixes the NEXT step, whose histogram this step's
        // collision kernel prepares: one 4-byte read-back per step between scatter and collide
        const int rm = read_step_max(ctx);
        double next_dt = (ctx->fuse_hist && rm == CUBA_OK) ? adaptive_dt(ctx, ctx->nmax_cur, dt_max, sigma) : 0.0;
        double nbase;
        if (next_dt > 0.0 && check_step_args(ctx, next_dt, sigma, &nbase) != CUBA_OK) next_dt = 0.0;   // the next call reports it
        rc = launch_collide<false>(ctx, base, nullptr, next_dt);   // the store is binned: always finish the step
        if (rc != CUBA_OK) return done(rc);
        ctx->pre_dt = next_dt;
        ctx->t += 1;
        ctx->steps += 1;
        if (dt_used) dt_used[s] = dt;
        sum = sum + dt;
        if (rm != CUBA_OK) return done(rm);
    }
    return done(CUBA_OK);
}

int cuba_step_traced(cuba_ctx *ctx, double dt, double sigma, cuba_trace *out)
{
    if (!ctx || !out || !out->cell_of_pid) return CUBA_ERR_NULL;
    if (ctx->slab) return CUBA_ERR_VALUE;      // pids are global in a slab: the per-pid trace arrays do not apply
    if (out->pair_capacity > 0 && (!out->pair_cell || !out->pair_round || !out->pid_a || !out->pid_b || !out->P ||
                                   !out->u || !out->decided)) return CUBA_ERR_NULL;
    double base;
    int rc = check_step_args(ctx, dt, sigma, &base);
    if (rc != CUBA_OK) return rc;
    rc = settle(ctx);
    if (rc != CUBA_OK) return rc;
    const int64_t n = ctx->n;
    const uint32_t ncells = ctx->g.ncells;
    TraceDev td;
    auto release = [&]() {
        cudaFree(td.off); cudaFree(td.cell); cudaFree(td.round); cudaFree(td.pa); cudaFree(td.pb);
        cudaFree(td.cell_of_pid); cudaFree(td.P); cudaFree(td.u); cudaFree(td.dec);
    };
    // After enqueue_bin the store has been streamed and re-sorted: from there on the step is always
    // completed (untraced if the records cannot be taken), so that an error never leaves the context
    // half-stepped -- a retry with a larger capacity would otherwise stream a second time.
    bool binned = false, collided = false;
    auto body = [&]() -> int {
        CU(cudaMalloc(&td.cell_of_pid, (size_t)n * 4));
        int r = enqueue_bin(ctx, dt, td.cell_of_pid);
        if (r != CUBA_OK) return r;
        binned = true;
        r = sync_and_check(ctx);
        if (r != CUBA_OK) return r;
        // per-cell record offsets: R(n) * floor(n/2), the same fp64 expressions as the kernel
        std::vector<uint32_t> start((size_t)ncells + 1);
        CU(cudaMemcpy(start.data(), ctx->at<uint32_t>(ctx->lay.cell_start), ((size_t)ncells + 1) * 4, cudaMemcpyDeviceToHost));
        std::vector<unsigned long long> off((size_t)ncells + 1);
        unsigned long long run = 0;
        for (uint32_t c = 0; c < ncells; ++c) {
            off[c] = run;
            const uint32_t nn = start[c + 1] - start[c];
            if (nn >= 2) {
                const double cn = (nn & 1u) ? (double)nn : (double)(nn - 1u);
                const double pmax = (2.0 * cn) * base;
                int R = !(pmax <= 64.0) ? 64 : ((pmax <= 1.0) ? 1 : (int)std::ceil(pmax));
                run += (unsigned long long)R * (nn >> 1);
            }
        }
        off[ncells] = run;
        out->n_pairs = (int64_t)run;
        CU(cudaMemcpy(out->cell_of_pid, td.cell_of_pid, (size_t)n * 4, cudaMemcpyDeviceToHost));
        if ((int64_t)run > out->pair_capacity) return CUBA_ERR_TRACE;
        const size_t m = run ? (size_t)run : 1;
        CU(cudaMalloc(&td.off, ((size_t)ncells + 1) * 8));
        CU(cudaMalloc(&td.cell, m * 4)); CU(cudaMalloc(&td.round, m * 4));
        CU(cudaMalloc(&td.pa, m * 4)); CU(cudaMalloc(&td.pb, m * 4));
        CU(cudaMalloc(&td.P, m * 8)); CU(cudaMalloc(&td.u, m * 8)); CU(cudaMalloc(&td.dec, m));
        CU(cudaMemcpy(td.off, off.data(), ((size_t)ncells + 1) * 8, cudaMemcpyHostToDevice));
        collided = true;
        r = launch_collide<true>(ctx, base, &td, 0.0);
        if (r != CUBA_OK) return r;
        ctx->t += 1;
        ctx->steps += 1;
        ctx->nmax_valid = false;
        r = sync_and_check(ctx);
        if (r != CUBA_OK) return r;
        if (run) {
            CU(cudaMemcpy(out->pair_cell, td.cell, m * 4, cudaMemcpyDeviceToHost));
            CU(cudaMemcpy(out->pair_round, td.round, m * 4, cudaMemcpyDeviceToHost));
            CU(cudaMemcpy(out->pid_a, td.pa, m * 4, cudaMemcpyDeviceToHost));
            CU(cudaMemcpy(out->pid_b, td.pb, m * 4, cudaMemcpyDeviceToHost));
            CU(cudaMemcpy(out->P, td.P, m * 8, cudaMemcpyDeviceToHost));
            CU(cudaMemcpy(out->u, td.u, m * 8, cudaMemcpyDeviceToHost));
            CU(cudaMemcpy(out->decided, td.dec, m, cudaMemcpyDeviceToHost));
        }
        return CUBA_OK;
    };
    rc = body();
    if (rc != CUBA_OK && binned && !collided) {
        // finish the step without records (a short capacity, a failed allocation)
        cudaGetLastError();
        if (launch_collide<false>(ctx, base, nullptr, 0.0) == CUBA_OK) {
            ctx->t += 1; ctx->steps += 1; ctx->nmax_valid = false;
            cudaStreamSynchronize(ctx->stream);
        }
    }
    release();
    return rc;

}

int cuba_set_option(cuba_ctx *ctx, int option, int value)
{
    if (!ctx) return CUBA_ERR_NULL;
    // a slab context steps on the plain compact schedule only (cuba_slab_init): the slotted store and the graph
    // would collide the ghost cells too, a fused histogram would cover the owned cells only -- switching one
    // on is refused, switching it off (what it already is) is accepted
    if (ctx->slab && value != 0 && (option == CUBA_OPT_SLOTS || option == CUBA_OPT_FUSE_HIST || option == CUBA_OPT_GRAPH))
        return CUBA_ERR_VALUE;
    if (option == CUBA_OPT_SLOTS) {
        if (value < 0 || value > 2) return CUBA_ERR_VALUE;
        ctx->slot_mode = value;
        return CUBA_OK;
    }
    if (option == CUBA_OPT_SLOT_MARGIN) {
        if (value < 1 || value > 1000) return CUBA_ERR_VALUE;
        ctx->slot_margin = (double)value / 100.0;
        ctx->slot_boost = 1.0;
        const int rs = settle(ctx);
        slot_release(ctx);
        return rs;
    }
    if ((option != CUBA_OPT_FUSE_HIST && option != CUBA_OPT_GRAPH) || (value != 0 && value != 1)) return CUBA_ERR_VALUE;
    if (option == CUBA_OPT_GRAPH) { ctx->use_graph = value != 0; return CUBA_OK; }
    ctx->fuse_hist = value != 0;
    if (!ctx->fuse_hist) ctx->pre_dt = 0.0;
    return CUBA_OK;
}

// ---- x-slab decomposition ---------------------------------------------------------
// Collisions are cell-local and dt < cell edge, so the path shards by layers of
// cells along x.  A rank owns the layers [layer_lo, layer_hi) and keeps, in the SAME global grid and
// coordinates (no offset: every operation rounds as on one GPU), a copy of the two adjacent boundary layers
// of its neighbours (ghosts).  One step = cuba_step(1) on the local store (S1-S4 on owned + ghost particles,
// S5 on the owned cells only: ClassTable range) -- the particles that enter an owned cell from a ghost cell
// are placed by the same stable sort as on one GPU, because the ghost cells hold exactly what the neighbour
// holds, in the same order -- then the halo exchange: every rank packs its two owned boundary layers after
// the collisions (contiguous ranges of the cell-sorted store: cuba_slab_pack), the neighbours rebuild their
// store as [ghost from below][owned cells][ghost from above] (cuba_slab_unpack).  What a rank streamed out of
// its owned layers is dropped there and reappears at the neighbour, which streamed its ghost copy of the same
// particles.  The concatenation of the ranks' owned ranges is the one-GPU store bit for bit.
static int slab_read_owned(cuba_ctx *ctx)
{
    if (ctx->own_valid) return CUBA_OK;
    const uint32_t *cs = ctx->at<uint32_t>(ctx->lay.cell_start);
    const uint32_t nyz = (uint32_t)(ctx->g.nc[1] * ctx->g.nc[2]);
    const uint32_t at[4] = {ctx->own_lo, ctx->own_lo + nyz, ctx->own_hi - nyz, ctx->own_hi};
    for (int k = 0; k < 4; ++k)
        CU(cudaMemcpyAsync(ctx->h_u32 + k, cs + at[k], 4, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    for (int k = 0; k < 4; ++k) ctx->own_cs[k] = ctx->h_u32[k];
    ctx->own_valid = true;
    return CUBA_OK;
}

__global__ void __launch_bounds__(256)
k_slab_pack_counts(const uint32_t *__restrict__ cell_start, uint32_t c0, uint32_t nyz, unsigned long long count,
                   unsigned long long *__restrict__ header, uint32_t *__restrict__ counts)
{
    const uint32_t i = blockIdx.x * 256u + threadIdx.x;
    if (i == 0) { header[0] = count; header[1] = nyz; }
    if (i < nyz) counts[i] = cell_start[c0 + i + 1] - cell_start[c0 + i];
}

// Copies up to three runs of particles (seven arrays each) into dst[0 .. n0 + n1 + n2): one launch instead of 21
// copies.  A run is (source arrays, first slot, count); a halo buffer is a source whose arrays are its sections.
struct SlabRun { const double *a[6]; const uint32_t *pid; uint32_t first, count; };

__global__ void __launch_bounds__(256)
k_slab_gather(SlabRun r0, SlabRun r1, SlabRun r2, Soa dst, uint32_t dst_first)
{
    const uint32_t total = r0.count + r1.count + r2.count;
    for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < total; i += gridDim.x * 256u) {
        const SlabRun &r = i < r0.count ? r0 : (i < r0.count + r1.count ? r1 : r2);
        const uint32_t k = r.first + (i < r0.count ? i : (i < r0.count + r1.count ? i - r0.count : i - r0.count - r1.count));
        const uint32_t o = dst_first + i;
        dst.x[o] = r.a[0][k]; dst.y[o] = r.a[1][k]; dst.z[o] = r.a[2][k];
        dst.px[o] = r.a[3][k]; dst.py[o] = r.a[4][k]; dst.pz[o] = r.a[5][k];
        dst.pid[o] = r.pid[k];
    }
}

static SlabRun slab_run_of_store(const Soa &s, uint32_t first, uint32_t count)
{
    SlabRun r{};
    r.a[0] = s.x; r.a[1] = s.y; r.a[2] = s.z; r.a[3] = s.px; r.a[4] = s.py; r.a[5] = s.pz;
    r.pid = s.pid; r.first = first; r.count = count;
    return r;
}

static SlabRun slab_run_of_buffer(const unsigned char *b, uint32_t count)
{
    SlabRun r{};
    if (b)
        for (int k = 0; k < 6; ++k) r.a[k] = reinterpret_cast<const double *>(b + 16 + (size_t)k * count * 8);
    r.pid = b ? reinterpret_cast<const uint32_t *>(b + 16 + (size_t)count * 48) : nullptr;
    r.first = 0; r.count = b ? count : 0u;
    return r;
}

// population of every cell of the rebuilt store + per-block sums for the scan
__global__ void __launch_bounds__(256)
k_slab_counts(uint32_t ncells, const uint32_t *__restrict__ cell_start_old, uint32_t own_lo, uint32_t own_hi, uint32_t nyz,
              const uint32_t *__restrict__ lo_counts, const uint32_t *__restrict__ hi_counts,
              uint32_t *__restrict__ count_new, uint32_t *__restrict__ block_sum,
              const unsigned long long *__restrict__ lo_header, unsigned long long lo_count,
              const unsigned long long *__restrict__ hi_header, unsigned long long hi_count, uint32_t *__restrict__ flags)
{
    __shared__ uint32_t s_warp[8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const uint32_t c = blockIdx.x * 256u + threadIdx.x;
    // the header {particles, cells per layer} that cuba_slab_pack wrote must be the count the caller passed on:
    // the sections of the buffer were addressed with that count
    if (c == 0 && ((lo_header && (lo_header[0] != lo_count || lo_header[1] != nyz)) ||
                   (hi_header && (hi_header[0] != hi_count || hi_header[1] != nyz))))
        atomicOr(flags, kFlagHalo);
    uint32_t v = 0;
    if (c < ncells) {
        if (c >= own_lo && c < own_hi) v = cell_start_old[c + 1] - cell_start_old[c];
        else if (lo_counts && c + nyz >= own_lo && c < own_lo) v = lo_counts[c + nyz - own_lo];
        else if (hi_counts && c >= own_hi && c < own_hi + nyz) v = hi_counts[c - own_hi];
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

int cuba_slab_layer_index(double box_x, int nx, int64_t n, const double *x, int32_t *layer)
{
    if (!x || !layer) return CUBA_ERR_NULL;
    if (n < 0 || nx < 1) return CUBA_ERR_SIZE;
    if (!(box_x > 0.0) || !std::isfinite(box_x)) return CUBA_ERR_VALUE;
    const double inv_d = 1.0 / (box_x / (double)nx);       // as Geom::inv_d in init_impl
    for (int64_t i = 0; i < n; ++i) layer[i] = axis_index(x[i], inv_d, nx);
    return CUBA_OK;
}

size_t cuba_slab_buffer_bytes(int64_t count, const int ncell[3])
{
    if (!ncell || count < 0) return 0;
    return 16 + (size_t)count * 52 + (size_t)ncell[1] * ncell[2] * 4;
}

int cuba_slab_owned(cuba_ctx *ctx, int64_t out[4])
{
    if (!ctx || !out) return CUBA_ERR_NULL;
    if (!ctx->slab) return CUBA_ERR_VALUE;
    const int rc = slab_read_owned(ctx);
    if (rc != CUBA_OK) return rc;
    out[0] = ctx->own_cs[0]; out[1] = (int64_t)ctx->own_cs[3] - ctx->own_cs[0]; out[2] = ctx->n; out[3] = ctx->cap;
    return CUBA_OK;
}

int cuba_slab_count(cuba_ctx *ctx, int side, int64_t *count)
{
    if (!ctx || !count) return CUBA_ERR_NULL;
    if (!ctx->slab || (side != 0 && side != 1)) return CUBA_ERR_VALUE;
    const int rc = slab_read_owned(ctx);
    if (rc != CUBA_OK) return rc;
    *count = side == 0 ? (int64_t)ctx->own_cs[1] - ctx->own_cs[0] : (int64_t)ctx->own_cs[3] - ctx->own_cs[2];
    return CUBA_OK;
}

int cuba_slab_pack(cuba_ctx *ctx, int side, void *buffer, size_t buffer_bytes)
{
    if (!ctx || !buffer) return CUBA_ERR_NULL;
    if (!ctx->slab || (side != 0 && side != 1)) return CUBA_ERR_VALUE;
    if (reinterpret_cast<uintptr_t>(buffer) & 15u) return CUBA_ERR_WORKSPACE;
    int rc = slab_read_owned(ctx);
    if (rc != CUBA_OK) return rc;
    const uint32_t nyz = (uint32_t)(ctx->g.nc[1] * ctx->g.nc[2]);
    const uint32_t first = side == 0 ? ctx->own_cs[0] : ctx->own_cs[2];
    const uint32_t count = (side == 0 ? ctx->own_cs[1] : ctx->own_cs[3]) - first;
    const uint32_t c0 = side == 0 ? ctx->own_lo : ctx->own_hi - nyz;
    if (buffer_bytes < cuba_slab_buffer_bytes(count, ctx->g.nc)) return CUBA_ERR_SIZE;
    unsigned char *b = static_cast<unsigned char *>(buffer);
    cudaStream_t st = ctx->stream;
    if (count) {
        Soa dst{};
        double **d6[6] = {&dst.x, &dst.y, &dst.z, &dst.px, &dst.py, &dst.pz};
        for (int k = 0; k < 6; ++k) *d6[k] = reinterpret_cast<double *>(b + 16 + (size_t)k * count * 8);
        dst.pid = reinterpret_cast<uint32_t *>(b + 16 + (size_t)count * 48);
        const SlabRun none{};
        k_slab_gather<<<std::min<unsigned>((count + 255u) / 256u, 148u * 8u), 256, 0, st>>>(slab_run_of_store(ctx->set[ctx->cur], first, count), none, none, dst, 0u);
        LAUNCHED();
    }
    k_slab_pack_counts<<<(nyz + 255u) / 256u, 256, 0, st>>>(ctx->at<uint32_t>(ctx->lay.cell_start), c0, nyz, count,
                                                            reinterpret_cast<unsigned long long *>(b),
                                                            reinterpret_cast<uint32_t *>(b + 16 + (size_t)count * 52));
    LAUNCHED();
    return CUBA_OK;
}

int cuba_slab_unpack(cuba_ctx *ctx, const void *lo_buffer, int64_t lo_count, const void *hi_buffer, int64_t hi_count)
{
    if (!ctx) return CUBA_ERR_NULL;
    if (!ctx->slab || lo_count < 0 || hi_count < 0) return CUBA_ERR_VALUE;
    if ((lo_buffer == nullptr) != (ctx->layer_lo == 0) || (hi_buffer == nullptr) != (ctx->layer_hi == ctx->g.nc[0])) return CUBA_ERR_VALUE;
    if (!lo_buffer) lo_count = 0;
    if (!hi_buffer) hi_count = 0;
    int rc = slab_read_owned(ctx);
    if (rc != CUBA_OK) return rc;
    const Layout &lay = ctx->lay;
    const uint32_t own_first = ctx->own_cs[0];
    const int64_t own_count = (int64_t)ctx->own_cs[3] - own_first;
    const int64_t n_new = lo_count + own_count + hi_count;
    if (n_new < 1 || n_new > ctx->cap) return CUBA_ERR_SIZE;
    cudaStream_t st = ctx->stream;
    const Soa &from = ctx->set[ctx->cur], &to = ctx->set[1 - ctx->cur];
    const unsigned char *lb = static_cast<const unsigned char *>(lo_buffer), *hb = static_cast<const unsigned char *>(hi_buffer);
    k_slab_gather<<<std::min<unsigned>((unsigned)((n_new + 255) / 256), 148u * 8u), 256, 0, st>>>(
        slab_run_of_buffer(lb, (uint32_t)lo_count), slab_run_of_store(from, own_first, (uint32_t)own_count),
        slab_run_of_buffer(hb, (uint32_t)hi_count), to, 0u);
    LAUNCHED();
    // cell table of the rebuilt store
    const uint32_t ncells = ctx->g.ncells, nyz = (uint32_t)(ctx->g.nc[1] * ctx->g.nc[2]);
    uint32_t *zero = ctx->at<uint32_t>(lay.zero);
    // the old table is read while the new one is written by a later kernel: counts first, into count_new
    k_slab_counts<<<(unsigned)lay.nblocks_cells, 256, 0, st>>>(ncells, ctx->at<uint32_t>(lay.cell_start), ctx->own_lo, ctx->own_hi, nyz,
                                                               lb ? reinterpret_cast<const uint32_t *>(lb + 16 + (size_t)lo_count * 52) : nullptr,
                                                               hb ? reinterpret_cast<const uint32_t *>(hb + 16 + (size_t)hi_count * 52) : nullptr,
                                                               ctx->at<uint32_t>(lay.count_new), ctx->at<uint32_t>(lay.block_sum),
                                                               reinterpret_cast<const unsigned long long *>(lb), (unsigned long long)lo_count,
                                                               reinterpret_cast<const unsigned long long *>(hb), (unsigned long long)hi_count,
                                                               ctx->at<uint32_t>(lay.flags));
    LAUNCHED();
    k_scan_blocks<<<1, 1024, 0, st>>>(ctx->at<uint32_t>(lay.block_sum), (int)lay.nblocks_cells, zero, kZeroWords);
    LAUNCHED();
    ClassTable ct{};
#define CUBA_CAP(K, T, I, C, MB) ct.max_n[K] = C;
    CUBA_FOR_EACH_CLASS(CUBA_CAP)
#undef CUBA_CAP
    ct.max_n[kSmemClasses] = 0xFFFFFFFFu;
    ct.c_lo = ctx->own_lo; ct.c_hi = ctx->own_hi;
    k_cell_start<<<(unsigned)lay.nblocks_cells, 256, 0, st>>>(ncells, ctx->at<uint32_t>(lay.count_new), ctx->at<uint32_t>(lay.block_sum),
                                                              ctx->at<uint32_t>(lay.cell_start), ct, zero, ctx->at<uint4>(lay.class_list),
                                                              ctx->at<unsigned long long>(lay.max_occ), zero + kStepMaxWord);
    LAUNCHED();
    ctx->cur = 1 - ctx->cur;
    ctx->n = n_new;
    ctx->pre_dt = 0.0; ctx->nmax_valid = false; ctx->own_valid = false;
    return CUBA_OK;
}

#ifdef CUBA_PHASE_CLOCKS
extern "C" int cuba_debug_phase(unsigned long long out[16], int reset)
{
    if (cudaDeviceSynchronize() != cudaSuccess) return CUBA_ERR_CUDA;
    if (cudaMemcpyFromSymbol(out, g_phase, sizeof(unsigned long long) * 16) != cudaSuccess) return CUBA_ERR_CUDA;
    if (reset) { unsigned long long z[16] = {}; cudaMemcpyToSymbol(g_phase, z, sizeof(z)); }
    return CUBA_OK;
}
#endif

int cuba_slot_stats(cuba_ctx *ctx, uint64_t out[2])
{
    if (!ctx || !out) return CUBA_ERR_NULL;
    const int rc = settle(ctx);      // a pending run is verified (and redone if it outgrew a segment) first
    out[0] = ctx->slot_runs; out[1] = ctx->slot_replays;
    return rc;
}

int cuba_observables(cuba_ctx *ctx, double total[4], int nslab, double *edens)
{
    if (!ctx || !total || !edens) return CUBA_ERR_NULL;
    if (nslab < 1 || nslab > kObsMaxSlabs) return CUBA_ERR_SIZE;
    { const int rs = settle(ctx); if (rs != CUBA_OK) return rs; }
    const Layout &lay = ctx->lay;
    Soa cur = ctx->set[ctx->cur];
    int64_t n_obs = ctx->n;
    if (ctx->slab) {           // a slab reports its owned particles only (the caller adds the slabs up)
        const int ro = slab_read_owned(ctx);
        if (ro != CUBA_OK) return ro;
        const size_t f = ctx->own_cs[0];
        cur.x += f; cur.px += f; cur.py += f; cur.pz += f;
        n_obs = (int64_t)ctx->own_cs[3] - ctx->own_cs[0];
    }
    cudaStream_t st = ctx->stream;
    const double inv_w = (double)nslab / ctx->box[0];
    const double vol = ((ctx->n_test * (ctx->box[0] / (double)nslab)) * ctx->box[1]) * ctx->box[2];
    double *partial = ctx->at<double>(lay.obs_partial), *result = ctx->at<double>(lay.obs_result);
    // slabs a layer of cells can touch; more than two: running sums in shared memory (observe.cuh, WIDE)
    const int per_layer = (nslab + ctx->g.nc[0] - 1) / ctx->g.nc[0] + 1;
    if (nslab > 2 * ctx->g.nc[0]) {
        const int window = per_layer < kObsWindowMax ? per_layer : kObsWindowMax;
        k_observe_partial<false, true><<<kObsGrid, kObsThreads, (size_t)kObsWarps * (nslab + window * 32) * 8, st>>>(
            n_obs, cur.x, cur.px, cur.py, cur.pz, inv_w, nslab, window, partial);
    } else {
        k_observe_partial<false, false><<<kObsGrid, kObsThreads, (size_t)kObsWarps * nslab * 8, st>>>(n_obs, cur.x, cur.px, cur.py, cur.pz,
                                                                                                 inv_w, nslab, 2, partial);
    }
    LAUNCHED();
    k_observe_final<<<(4 + nslab + 7) / 8, 256, 0, st>>>(kObsGrid, nslab, partial, vol, result);
    LAUNCHED();
    CU(cudaMemcpyAsync(ctx->h_obs, result, (size_t)(4 + nslab) * 8, cudaMemcpyDeviceToHost, st));
    int rc = sync_and_check(ctx);
    if (rc != CUBA_OK) return rc;
    memcpy(total, ctx->h_obs, 4 * sizeof(double));
    memcpy(edens, ctx->h_obs + 4, (size_t)nslab * sizeof(double));
    return CUBA_OK;
}

int cuba_observables_lrf(cuba_ctx *ctx, int nslab, double *T, double *lrf)
{
    if (!ctx || !T || !lrf) return CUBA_ERR_NULL;
    if (nslab < 1 || nslab > kLrfMaxSlabs) return CUBA_ERR_SIZE;
    { const int rs = settle(ctx); if (rs != CUBA_OK) return rs; }
    const Layout &lay = ctx->lay;
    Soa cur = ctx->set[ctx->cur];
    int64_t n_obs = ctx->n;
    if (ctx->slab) {           // a slab reports its owned particles only (the caller adds the slabs up)
        const int ro = slab_read_owned(ctx);
        if (ro != CUBA_OK) return ro;
        const size_t f = ctx->own_cs[0];
        cur.x += f; cur.px += f; cur.py += f; cur.pz += f;
        n_obs = (int64_t)ctx->own_cs[3] - ctx->own_cs[0];
    }
    cudaStream_t st = ctx->stream;
    const double inv_w = (double)nslab / ctx->box[0];
    const double vol = ((ctx->n_test * (ctx->box[0] / (double)nslab)) * ctx->box[1]) * ctx->box[2];
    double *partial = ctx->at<double>(lay.obs_partial), *result = ctx->at<double>(lay.obs_result);
    const int grid = 148 * 3;           // 3 CTAs per SM (2 when nslab needs more than 75 KB of shared memory each)
    static_assert(148 * 3 <= kObsGrid, "partial buffer is sized for kObsGrid blocks");
    const int per_layer = (nslab + ctx->g.nc[0] - 1) / ctx->g.nc[0] + 1;
    if (nslab > 2 * ctx->g.nc[0]) {
        const int window = per_layer < kLrfWindowMax ? per_layer : kLrfWindowMax;
        k_observe_partial<true, true><<<grid, kObsThreads, (size_t)kObsWarps * kLrfComp * (nslab + window * 32) * 8, st>>>(
            n_obs, cur.x, cur.px, cur.py, cur.pz, inv_w, nslab, window, partial);
    } else {
        k_observe_partial<true, false><<<grid, kObsThreads, (size_t)kObsWarps * kLrfComp * nslab * 8, st>>>(n_obs, cur.x, cur.px, cur.py, cur.pz,
                                                                                                         inv_w, nslab, 2, partial);
    }
    LAUNCHED();
    k_observe_lrf_final<<<(nslab + 7) / 8, 256, 0, st>>>(grid, nslab, partial, vol, result);
    LAUNCHED();
    CU(cudaMemcpyAsync(ctx->h_obs, result, (size_t)9 * nslab * 8, cudaMemcpyDeviceToHost, st));
    int rc = sync_and_check(ctx);
    if (rc != CUBA_OK) return rc;
    memcpy(T, ctx->h_obs, (size_t)kLrfComp * nslab * sizeof(double));
    memcpy(lrf, ctx->h_obs + (size_t)kLrfComp * nslab, (size_t)4 * nslab * sizeof(double));
    return CUBA_OK;
}

// ---- cuba_observables_noalloc: the observables pass for callers that must not allocate -------------------
// The per-CTA partial sums that cuba_observables keeps in the caller's workspace live here in a
// fixed array that is part of the loaded library image instead: kObsGrid rows of 4 totals +
// CUBA_NOALLOC_MAX_SLABS slab energies (592 x 132 doubles = 625,152 bytes on every GPU that loads
// the library, until the process exits).
static __device__ __align__(256) double g_noalloc_partial[(size_t)kObsGrid * (4 + CUBA_NOALLOC_MAX_SLABS)];

namespace {
constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mutex;
double *g_noalloc_ptr[kNoallocMaxDevices] = {};   // device address of g_noalloc_partial on each device, once looked up
}  // namespace

// In host code the name g_noalloc_partial is only a handle for the runtime, not a device address: the
// address a kernel can use has to be asked for, per device, with that device current.  Done on the first
// call on each device and remembered; later calls on that device touch no CUDA API but the launches.
static int noalloc_scratch(double **out)
{
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoallocMaxDevices) return CUBA_ERR_VALUE;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void *p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_noalloc_partial));
        if (!p) return CUBA_ERR_CUDA;
        g_noalloc_ptr[dev] = static_cast<double *>(p);
    }
    *out = g_noalloc_ptr[dev];
    return CUBA_OK;
}

int cuba_observables_noalloc(int64_t n, const double *x, const double *px, const double *py, const double *pz,
                             const double box[3], double n_test, int nslab, double *result, void *cuda_stream)
{
    if (!x || !px || !py || !pz || !box || !result) return CUBA_ERR_NULL;
    if (n < 1 || n >= ((int64_t)1 << 32)) return CUBA_ERR_SIZE;
    if (nslab < 1 || nslab > CUBA_NOALLOC_MAX_SLABS) return CUBA_ERR_SIZE;   // the fixed array has no room for more
    for (int k = 0; k < 3; ++k) if (!(box[k] > 0.0) || !std::isfinite(box[k])) return CUBA_ERR_VALUE;
    if (!(n_test > 0.0) || !std::isfinite(n_test)) return CUBA_ERR_VALUE;
    for (const double *a : {x, px, py, pz, (const double *)result})
        if (reinterpret_cast<uintptr_t>(a) & 7u) return CUBA_ERR_WORKSPACE;
    double *partial = nullptr;
    const int rc = noalloc_scratch(&partial);
    if (rc != CUBA_OK) return rc;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    // the same two kernels, grid, operation order and constants as cuba_observables with nslab <= 2 nx, so
    // the sums come out with the same bits; every CTA writes its whole row of `partial` before the second
    // kernel reads it, so what the previous call left in the array is never read and nothing needs clearing
    const double inv_w = (double)nslab / box[0];
    const double vol = ((n_test * (box[0] / (double)nslab)) * box[1]) * box[2];
    k_observe_partial<false, false><<<kObsGrid, kObsThreads, (size_t)kObsWarps * nslab * 8, st>>>(n, x, px, py, pz, inv_w, nslab, 2,
                                                                                             partial);
    LAUNCHED();
    k_observe_final<<<(4 + nslab + 7) / 8, 256, 0, st>>>(kObsGrid, nslab, partial, vol, result);
    LAUNCHED();
    return CUBA_OK;
}

int cuba_state(cuba_ctx *ctx, cuba_soa *out)
{
    if (!ctx || !out) return CUBA_ERR_NULL;
    { const int rs = settle(ctx); if (rs != CUBA_OK) return rs; }
    const Soa &c = ctx->set[ctx->cur];
    out->x = c.x; out->y = c.y; out->z = c.z; out->px = c.px; out->py = c.py; out->pz = c.pz;
    out->pid = c.pid;
    out->cell_start = ctx->at<uint32_t>(ctx->lay.cell_start);
    return CUBA_OK;
}

int cuba_get_particles(cuba_ctx *ctx, uint32_t *pid, double *x, double *y, double *z,
                       double *px, double *py, double *pz)
{
    if (!ctx) return CUBA_ERR_NULL;
    int rc = settle(ctx);
    if (rc != CUBA_OK) return rc;
    rc = sync_and_check(ctx);
    if (rc != CUBA_OK) return rc;
    const Soa &c = ctx->set[ctx->cur];
    const size_t b = (size_t)ctx->n * 8;
    if (pid) CU(cudaMemcpy(pid, c.pid, (size_t)ctx->n * 4, cudaMemcpyDeviceToHost));
    if (x) CU(cudaMemcpy(x, c.x, b, cudaMemcpyDeviceToHost));
    if (y) CU(cudaMemcpy(y, c.y, b, cudaMemcpyDeviceToHost));
    if (z) CU(cudaMemcpy(z, c.z, b, cudaMemcpyDeviceToHost));
    if (px) CU(cudaMemcpy(px, c.px, b, cudaMemcpyDeviceToHost));
    if (py) CU(cudaMemcpy(py, c.py, b, cudaMemcpyDeviceToHost));
    if (pz) CU(cudaMemcpy(pz, c.pz, b, cudaMemcpyDeviceToHost));
    return CUBA_OK;
}

const char *cuba_profile_name(int group)
{
    static const char *names[CUBA_PROFILE_GROUPS] = {
        "memset_cnt", "k_stream_hist", "k_gather", "k_scan_blocks", "k_cell_start", "k_carry", "k_dest_base", "k_scatter",
        "k_collide (all classes, concurrent)"};
#define CUBA_STR2(x) #x
#define CUBA_STR(x) CUBA_STR2(x)
#define CUBA_NAME(K, T, I, C, MB) names[G_COLLIDE0 + K] = "k_collide<T=" CUBA_STR(T) ",cap=" CUBA_STR(C) ">";
    CUBA_FOR_EACH_CLASS(CUBA_NAME)
#undef CUBA_NAME
    names[G_COLLIDE0 + kSmemClasses] = "k_collide_overflow";
    names[G_SLOT_UNPACK] = "k_slot_step<first> (stream from the compact store)";
    names[G_SLOT_CLASSIFY] = "k_slot_classify";
    names[G_SLOT_STEP] = "k_slot_step (all classes, concurrent)";
    names[G_SLOT_PACK] = "k_slot_step<last> (collide into the compact store)";
    return (group >= 0 && group < CUBA_PROFILE_GROUPS) ? names[group] : "?";
}

int cuba_profile_enable(cuba_ctx *ctx, int on)
{
    if (!ctx) return CUBA_ERR_NULL;
    CU(cudaStreamSynchronize(ctx->stream));
    for (auto &pe : ctx->prof_log) ctx->prof_pool.push_back(pe.first);
    ctx->prof_log.clear();
    ctx->prof_on = on != 0;
    ctx->prof_mode = on;
    return CUBA_OK;
}

int cuba_profile_read(cuba_ctx *ctx, double *ms_sum, uint64_t *launches)
{
    if (!ctx || !ms_sum || !launches) return CUBA_ERR_NULL;
    CU(cudaStreamSynchronize(ctx->stream));
    for (int g = 0; g < CUBA_PROFILE_GROUPS; ++g) { ms_sum[g] = 0.0; launches[g] = 0; }
    for (size_t i = 1; i < ctx->prof_log.size(); ++i) {
        const int g = ctx->prof_log[i].second;
        if (g < 0) continue;                          // a step-start marker closes nothing
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, ctx->prof_log[i - 1].first, ctx->prof_log[i].first));
        ms_sum[g] += (double)ms;
        launches[g] += 1;
    }
    for (auto &pe : ctx->prof_log) ctx->prof_pool.push_back(pe.first);
    ctx->prof_log.clear();
    return CUBA_OK;
}

// fp64 FMA micro-benchmark (probe.cuh): thread-level DFMA instructions per second of the whole device
int cuba_probe_fp64(void *cuda_stream, int repeats, double *dfma_per_s)
{
    if (!dfma_per_s) return CUBA_ERR_NULL;
    if (repeats < 1 || repeats > 64) return CUBA_ERR_SIZE;
    *dfma_per_s = 0.0;
    cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int grid = sms * 8, iters = 1 << 14;
    double *out = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    CU(cudaMalloc(&out, (size_t)grid * kProbeThreads * sizeof(double)));
    auto done = [&](int code) { if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); cudaFree(out); return code; };
    if (!cuda_ok(cudaEventCreate(&e0), "cudaEventCreate") || !cuda_ok(cudaEventCreate(&e1), "cudaEventCreate")) return done(CUBA_ERR_CUDA);
    double best = 0.0;
    for (int r = 0; r <= repeats; ++r) {       // the first launch warms up
        cudaEventRecord(e0, st);
        k_probe_fp64<<<grid, kProbeThreads, 0, st>>>(iters, 0.999999, 1e-6, out);
        LAUNCHED();
        cudaEventRecord(e1, st);
        if (!cuda_ok(cudaEventSynchronize(e1), "cudaEventSynchronize")) return done(CUBA_ERR_CUDA);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double rate = (double)grid * kProbeThreads * kProbeChains * (double)iters / ((double)ms * 1e-3);
        if (r > 0 && rate > best) best = rate;
    }
    *dfma_per_s = best;
    return done(CUBA_OK);
}

int cuba_get_cells(cuba_ctx *ctx, uint32_t *cell_start)
{
    if (!ctx || !cell_start) return CUBA_ERR_NULL;
    int rc = settle(ctx);
    if (rc != CUBA_OK) return rc;
    rc = sync_and_check(ctx);
    if (rc != CUBA_OK) return rc;
    CU(cudaMemcpy(cell_start, ctx->at<uint32_t>(ctx->lay.cell_start), ((size_t)ctx->g.ncells + 1) * 4, cudaMemcpyDeviceToHost));
    return CUBA_OK;
}

int cuba_counters(cuba_ctx *ctx, cuba_counters_t *out)
{
    if (!ctx || !out) return CUBA_ERR_NULL;
    unsigned long long c[8] = {0};
    unsigned long long mo = 0;
    uint32_t f = 0;
    { const int rs = settle(ctx); if (rs != CUBA_OK) return rs; }
    CU(cudaStreamSynchronize(ctx->stream));
    CU(cudaMemcpy(c, ctx->at<void>(ctx->lay.counters), 64, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(&mo, ctx->at<void>(ctx->lay.max_occ), 8, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(&f, ctx->at<void>(ctx->lay.flags), 4, cudaMemcpyDeviceToHost));
    out->steps = ctx->steps; out->pairs = c[0]; out->collisions = c[1]; out->rounds = c[2];
    out->near_threshold = c[3]; out->max_occupancy = mo; out->overflow_cells = c[4]; out->device_flags = f;
    return CUBA_OK;
}

// Memory pool of cuba_run_host, one per device, created on first use and kept for the life of the
// process (release threshold: keep everything).
static int run_host_pool(int dev_id, cudaMemPool_t *out)
{
    static std::mutex mu;
    static cudaMemPool_t pools[64] = {};
    if (dev_id < 0 || dev_id >= 64) return CUBA_ERR_CUDA;
    std::lock_guard<std::mutex> lock(mu);
    if (!pools[dev_id]) {
        cudaMemPoolProps props{};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev_id;
        CU(cudaMemPoolCreate(&pools[dev_id], &props));
        uint64_t keep = UINT64_MAX;
        CU(cudaMemPoolSetAttribute(pools[dev_id], cudaMemPoolAttrReleaseThreshold, &keep));
    }
    *out = pools[dev_id];
    return CUBA_OK;
}

int cuba_run_host(const double box[3], const int ncell[3], int64_t n,
                  double *x, double *y, double *z, double *px, double *py, double *pz,
                  double n_test, uint64_t seed, int nsteps, double dt, double sigma,
                  double total[4], int nslab, double *edens, uint32_t *pid_out, int download)
{
    if (!box || !ncell || !x || !y || !z || !px || !py || !pz || !total || !edens) return CUBA_ERR_NULL;
    const size_t wsb = cuba_workspace_bytes(n, ncell);
    if (wsb == 0) return CUBA_ERR_SIZE;
    double *host[6] = {x, y, z, px, py, pz};
    double *dev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    void *ws = nullptr;
    cuba_ctx *ctx = nullptr;
    cudaStream_t st = nullptr, st2 = nullptr;
    cudaEvent_t ev_alloc = nullptr, ev_mom = nullptr;
    auto body = [&]() -> int {
        CU(cudaStreamCreate(&st));
        // stream-ordered allocations from a pool owned by the library, which keeps what it has been
        // given: a second call of the same size maps no new memory (cudaMalloc / cudaFree of 3.3 GB
        // cost ~10 ms per call at 24.9M particles).  The process-wide default pool is left alone.
        int dev_id = 0;
        CU(cudaGetDevice(&dev_id));
        cudaMemPool_t pool = nullptr;
        int rp = run_host_pool(dev_id, &pool);
        if (rp != CUBA_OK) return rp;
        for (int k = 0; k < 6; ++k) CU(cudaMallocFromPoolAsync(reinterpret_cast<void **>(&dev[k]), (size_t)n * 8, pool, st));
        CU(cudaMallocFromPoolAsync(&ws, wsb, pool, st));
        // positions on the main stream, momenta on a second one: the binning of the initial state needs the
        // positions only until it gathers the sorted store, so the sort of the keys overlaps the second half of the upload
        CU(cudaStreamCreateWithFlags(&st2, cudaStreamNonBlocking));
        CU(cudaEventCreateWithFlags(&ev_alloc, cudaEventDisableTiming));
        CU(cudaEventCreateWithFlags(&ev_mom, cudaEventDisableTiming));
        CU(cudaEventRecord(ev_alloc, st));
        CU(cudaStreamWaitEvent(st2, ev_alloc, 0));
        for (int k = 0; k < 3; ++k) CU(cudaMemcpyAsync(dev[k], host[k], (size_t)n * 8, cudaMemcpyHostToDevice, st));
        for (int k = 3; k < 6; ++k) CU(cudaMemcpyAsync(dev[k], host[k], (size_t)n * 8, cudaMemcpyHostToDevice, st2));
        CU(cudaEventRecord(ev_mom, st2));
        if (!ncell) return CUBA_ERR_NULL;
        int r = init_impl(&ctx, box, ncell, n, n, dev[0], dev[1], dev[2], dev[3], dev[4], dev[5], n_test, seed, ws, wsb, st,
                          nullptr, 0, ncell[0] > 0 ? ncell[0] : 1, false, ev_mom);
        if (r != CUBA_OK) return r;
        r = cuba_step(ctx, nsteps, dt, sigma);
        if (r != CUBA_OK) return r;
        r = cuba_observables(ctx, total, nslab, edens);
        if (r != CUBA_OK) return r;
        if (download) {
            const Soa &c = ctx->set[ctx->cur];
            const double *from[6] = {c.x, c.y, c.z, c.px, c.py, c.pz};
            for (int k = 0; k < 6; ++k) CU(cudaMemcpyAsync(host[k], from[k], (size_t)n * 8, cudaMemcpyDeviceToHost, st));
            if (pid_out) CU(cudaMemcpyAsync(pid_out, c.pid, (size_t)n * 4, cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
        }
        return CUBA_OK;
    };
    const int rc = body();
    if (ctx) cuba_destroy(ctx);
    if (st2) { cudaStreamSynchronize(st2); cudaStreamDestroy(st2); }     // (an early error may have left the copy running)
    if (st) {
        for (int k = 0; k < 6; ++k) if (dev[k]) cudaFreeAsync(dev[k], st);
        if (ws) cudaFreeAsync(ws, st);
        cudaStreamSynchronize(st);
        cudaStreamDestroy(st);
    }
    if (ev_alloc) cudaEventDestroy(ev_alloc);
    if (ev_mom) cudaEventDestroy(ev_mom);
    return rc;
}

