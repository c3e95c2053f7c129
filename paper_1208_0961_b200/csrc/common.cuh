// common.cuh -- shared device helpers of the CuBA B200 library: geometry, Eq. 2 streaming,
// wall reflection, cell index, Philox4x32-10.  Compiled with -fmad=false: every written
// fp64 operation rounds once (A2).  Citations: /root/reference/PAPER.md lines.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cuba {

constexpr int kDirs = 27;           // (dix+1)*9 + (diy+1)*3 + (diz+1), each di in {-1,0,1}
constexpr int kTileThreads = 256;
#ifndef CUBA_TILE_ITEMS
#define CUBA_TILE_ITEMS 2
#endif
constexpr int kTileItems = CUBA_TILE_ITEMS;
constexpr int kTile = kTileThreads * kTileItems;   // particles per tile in the flat passes
constexpr int kTileRows = kTile / 32;
constexpr int kTileRec = 32;        // u32 words per tile record: 27 counts, cf, cl, pad

// device error bits (sticky)
constexpr uint32_t kFlagMoved = 1u;    // a particle crossed more than one cell in a step
constexpr uint32_t kFlagRounds = 2u;   // a cell needed more than CUBA_MAX_ROUNDS rounds
constexpr uint32_t kFlagState = 4u;    // invalid particle at init
constexpr uint32_t kFlagTrace = 8u;    // trace capacity exceeded
constexpr uint32_t kFlagHalo = 32u;    // cuba_slab_unpack: a halo buffer's header disagrees with the count it was given (16 = kFlagSlots)

constexpr uint32_t kTagShuf = 0u, kTagDec = 1u, kTagDir = 2u;

struct Geom {
    double L[3];       // box edges, walls at 0 and L
    double inv_d[3];   // 1/(L/ncell) per axis
    int nc[3];         // cells per axis
    uint32_t ncells;
};

struct Soa {
    double *x, *y, *z, *px, *py, *pz;
    uint32_t *pid;
};

// ---- Philox4x32-10 (Salmon et al., SC'11): ten rounds of two 32x32->64 multiplies -------
struct U4 { uint32_t x, y, z, w; };

__device__ __forceinline__ U4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                            uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return U4{c0, c1, c2, c3};
}

// counter = {particle id, global step t, round rho, tag<<16 | sub}; key = seed (DESIGN.md RNG)
__device__ __forceinline__ U4 draw(uint64_t seed, uint32_t id, uint32_t t, uint32_t rho,
                                   uint32_t tag, uint32_t sub)
{
    return philox4x32_10(id, t, rho, (tag << 16) | sub, (uint32_t)seed, (uint32_t)(seed >> 32));
}

// ---- S1-S3 ---------------------------------------------------------------------------
__device__ __forceinline__ double energy(double px, double py, double pz)
{
    return sqrt((px * px + py * py) + pz * pz);      // massless: E = |p|
}

__device__ __forceinline__ void reflect_axis(double &x, double &p, double L)
{
    if (x < 0.0) { x = -x; p = -p; }                 // PAPER.md:44, walls at 0 and L (A12)
    else if (x > L) { x = 2.0 * L - x; p = -p; }
}

__device__ __forceinline__ void stream_reflect(const Geom &g, double dt, double &x, double &y,
                                               double &z, double &px, double &py, double &pz)
{
    const double E = energy(px, py, pz);
    const double w = dt / E;                         // PAPER.md:34 Eq. 2 with c = 1
    x = x + px * w;
    y = y + py * w;
    z = z + pz * w;
    reflect_axis(x, px, g.L[0]);
    reflect_axis(y, py, g.L[1]);
    reflect_axis(z, pz, g.L[2]);
}

// Also compiled for the host (cuba_slab_layer_index): there the conversion spells out what cvt.rzi.s32.f64 does
// (truncation, saturation, NaN -> 0); the product rounds the same (IEEE fp64, no contraction on either side).
__host__ __device__ __forceinline__ int axis_index(double x, double inv_d, int nc)
{
#ifdef __CUDA_ARCH__
    int i = __double2int_rz(x * inv_d);
#else
    const double v = x * inv_d;
    int i = (v != v) ? 0 : (v >= 2147483647.0 ? 2147483647 : (v <= -2147483648.0 ? (-2147483647 - 1) : (int)v));
    using std::min; using std::max;
#endif
    i = min(i, nc - 1);                              // x == L lands in the last cell (A12)
    return max(i, 0);
}

__device__ __forceinline__ uint32_t cell_linear(const Geom &g, int ix, int iy, int iz)
{
    return ((uint32_t)ix * (uint32_t)g.nc[1] + (uint32_t)iy) * (uint32_t)g.nc[2] + (uint32_t)iz;
}

__device__ __forceinline__ uint32_t lanemask_lt()
{
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

__device__ __forceinline__ uint32_t lanemask_le()
{
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_le;" : "=r"(m));
    return m;
}

// ---- TMA-style bulk staging: cp.async.bulk global -> shared, completion on an mbarrier ---
__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}

__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra.uni WAIT_DONE;\n"
        "bra.uni WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// bytes must be a multiple of 16 and both addresses 16-byte aligned.
// (Measured and rejected: an L2 evict-first cache hint on these copies, meant to leave the L2 to the
// partially written output sectors of the scatter: k_scatter 0.52 -> 0.63 ms at configs[2].)
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

}  // namespace cuba
