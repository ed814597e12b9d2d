// Independent Philox4x32-10 for the oracle's pin: NVIDIA cuRAND's own header
// (curand_philox4x32_x.h from the CUDA toolkit on this image), compiled for the host with g++.
// Exposes curand_Philox4x32_10(counter, key) through a C symbol.  Test helper only.
#include <cstdint>
#include <vector_types.h>
#include <nv/target>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>

extern "C" void curand_ref_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint4 c; c.x = ctr[0]; c.y = ctr[1]; c.z = ctr[2]; c.w = ctr[3];
    uint2 k; k.x = key[0]; k.y = key[1];
    uint4 r = curand_Philox4x32_10(c, k);
    out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
