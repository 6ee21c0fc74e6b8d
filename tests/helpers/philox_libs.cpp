// Test helper: exposes two *library* Philox4x32-10 implementations present on this box so
// the oracle's block function can be pinned against something other than itself:
//   (1) ATen's CPU philox_engine (torch/include/ATen/core/PhiloxRNGEngine.h)
//   (2) cuRAND's curand_Philox4x32_10 host path (/usr/local/cuda/include/curand_philox4x32_x.h)
// Contains no code of ours beyond argument marshalling.
#include <cstdint>
#include <ATen/core/PhiloxRNGEngine.h>

extern "C" void aten_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint64_t seed = (uint64_t)key[0] | ((uint64_t)key[1] << 32);
    const uint64_t subseq = (uint64_t)ctr[2] | ((uint64_t)ctr[3] << 32);
    const uint64_t offset = (uint64_t)ctr[0] | ((uint64_t)ctr[1] << 32);
    at::philox_engine eng(seed, subseq, 0);
    eng.set_offset(offset);
    for (int i = 0; i < 4; ++i) out[i] = eng();
}

#ifdef WITH_CURAND_HOST
#include <vector_types.h>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>
extern "C" void curand_host_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint4 c; c.x = ctr[0]; c.y = ctr[1]; c.z = ctr[2]; c.w = ctr[3];
    uint2 k; k.x = key[0]; k.y = key[1];
    uint4 r = curand_Philox4x32_10(c, k);
    out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
#endif
