// Test helper: thin wrappers around two LIBRARY implementations of Philox4x32-10
// that are on the box (pin P1): cuRAND's host-callable curand_Philox4x32_10 and
// torch's at::philox_engine.  No Philox arithmetic is written here.
#include <cstdint>
#include <vector_types.h>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>
#ifdef WITH_TORCH
#include <ATen/core/PhiloxRNGEngine.h>
#endif

extern "C" void ref_curand_philox(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4])
{
  uint4 c = {ctr[0], ctr[1], ctr[2], ctr[3]};
  uint2 k = {key[0], key[1]};
  uint4 r = curand_Philox4x32_10(c, k);
  out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}

#ifdef WITH_TORCH
// seed -> key, offset -> counter words 0,1, subsequence -> counter words 2,3
extern "C" void ref_torch_philox(uint64_t seed, uint64_t subsequence, uint64_t offset, uint32_t out[4])
{
  at::philox_engine e(seed, subsequence, offset);
  for (int i = 0; i < 4; ++i) out[i] = e();
}
#endif
