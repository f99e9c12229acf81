// Test helper: the CUDA toolkit's own Philox4x32-10 block function (curand_philox4x32_x.h),
// compiled for the HOST (the header has a host branch), exported with a C ABI so that the
// CPU tests can pin oracle/ and the CUDA path's generator against a library routine.
#include <cstdint>
#include <vector_types.h>
#define QUALIFIERS static inline __host__ __device__
#include <curand_philox4x32_x.h>

extern "C" void ref_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  uint4 c = {ctr[0], ctr[1], ctr[2], ctr[3]};
  uint2 k = {key[0], key[1]};
  uint4 r = curand_Philox4x32_10(c, k);
  out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
