// Test-only translation unit: exposes cuRAND's own library routine
// curand_Philox4x32_10 (/usr/local/cuda/include/curand_philox4x32_x.h) to the host
// so that the oracle's and the kernel library's Philox can be pinned against it.
// Neither oracle/ nor paper_2410_05985_b200/csrc/ includes that header.
#include <vector_types.h>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>

extern "C" void curand_philox_host(const unsigned *ctr, const unsigned *key, unsigned *out, long n) {
  for (long i = 0; i < n; ++i) {
    uint4 c = {ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]};
    uint2 k = {key[2 * i], key[2 * i + 1]};
    uint4 r = curand_Philox4x32_10(c, k);
    out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
  }
}
