// Test-only helper: exposes cuRAND's own Philox4x32-10 block function (the library routine
// in <curand_philox4x32_x.h>) to the host so the oracle's Philox can be pinned against it
// on all four counter words and both key words.  Not part of the product or the oracle.
#define QUALIFIERS static inline __host__ __device__
#include <cuda_runtime.h>
#include <curand_philox4x32_x.h>
#include <stdint.h>

extern "C" void curand_ref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint4 c = make_uint4(ctr[0], ctr[1], ctr[2], ctr[3]);
    uint2 k = make_uint2(key[0], key[1]);
    uint4 r = curand_Philox4x32_10(c, k);
    out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
