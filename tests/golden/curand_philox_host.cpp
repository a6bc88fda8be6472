// Host-side call of cuRAND's own Philox4x32-10 routine: an independent LIBRARY implementation
// used by tests/test_oracle_pins.py to pin the oracle's Philox on random counters/keys.
// (Test helper; compiled to a temp dir by the test.  Not part of the oracle or the product.)
#include <cstdint>
#include <vector_types.h>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>
extern "C" void curand_philox_host(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  uint4 c = {ctr[0], ctr[1], ctr[2], ctr[3]};
  uint2 k = {key[0], key[1]};
  uint4 r = curand_Philox4x32_10(c, k);
  out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
