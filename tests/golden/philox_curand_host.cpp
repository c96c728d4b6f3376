// Test-only shim: compiles cuRAND's own Philox4x32-10 round function for the host so the oracle's
// generator can be pinned to it word for word.  /usr/local/cuda/include/
// curand_philox4x32_x.h lets QUALIFIERS be overridden (its lines 84-85).
#define QUALIFIERS static inline
#include <vector_types.h>
#include <curand_philox4x32_x.h>
extern "C" void curand_philox_host(const unsigned* c, const unsigned* k, unsigned* out) {
  uint4 cc; cc.x = c[0]; cc.y = c[1]; cc.z = c[2]; cc.w = c[3];
  uint2 kk; kk.x = k[0]; kk.y = k[1];
  uint4 r = curand_Philox4x32_10(cc, kk);
  out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
