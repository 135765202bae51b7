// Test-only: exposes the CUDA toolkit's own curand_Philox4x32_10 (header
// /usr/local/cuda/include/curand_philox4x32_x.h, compiled for the host) so that the oracle's
// Philox can be pinned against an implementation it shares no code with.
#include <vector_types.h>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>

extern "C" void toolkit_philox4x32_10(const unsigned int *ctr, const unsigned int *key,
                                      unsigned int *out) {
  uint4 c = {ctr[0], ctr[1], ctr[2], ctr[3]};
  uint2 k = {key[0], key[1]};
  uint4 r = curand_Philox4x32_10(c, k);
  out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
