// Test-only helper: exposes the CUDA toolkit's own Philox4x32-10 (curand_philox4x32_x.h, which has
// a host code path) through a C symbol so the oracle's generator can be pinned to a library
// routine on the CPU.  Not part of the product; built by tests/test_oracle_sampling.py.
#include <cuda_runtime.h>
#define QUALIFIERS static inline __host__ __device__
#include <curand_philox4x32_x.h>
#include <stdint.h>

extern "C" void curand_philox_host(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
    uint4 c = make_uint4(ctr[0], ctr[1], ctr[2], ctr[3]);
    uint2 k = make_uint2(key[0], key[1]);
    uint4 r = curand_Philox4x32_10(c, k);
    out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
