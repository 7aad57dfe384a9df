// Test-only shim: exposes NVIDIA cuRAND's own curand_Philox4x32_10(uint4, uint2)
// (header /usr/local/cuda/include/curand_philox4x32_x.h, host code path) to the
// CPU tests as an independent implementation to pin the oracle's Philox against.
// Holds no arithmetic of its own.
#include <cuda_runtime.h>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>
#include <stdint.h>

extern "C" void shim_curand_philox4x32_10(const uint32_t c[4], const uint32_t k[2], uint32_t out[4])
{
    uint4 ctr = make_uint4(c[0], c[1], c[2], c[3]);
    uint2 key = make_uint2(k[0], k[1]);
    uint4 r = curand_Philox4x32_10(ctr, key);
    out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
