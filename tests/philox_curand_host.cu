// Test helper (tests/test_oracle_generators.py): evaluates the CUDA toolkit's own Philox-4x32-10
// round function (curand_philox4x32_x.h, host-callable once QUALIFIERS is redefined) on
// "k0 k1 c0 c1 c2 c3" lines from stdin.  Library code, used as an independent pin of the oracle's
// restatement of the published algorithm; no GPU is needed.
#define QUALIFIERS static __forceinline__ __host__ __device__
#include <cuda_runtime.h>
#include <curand_philox4x32_x.h>
#include <cstdio>
int main() {
  unsigned k0, k1, c0, c1, c2, c3;
  while (scanf("%u %u %u %u %u %u", &k0, &k1, &c0, &c1, &c2, &c3) == 6) {
    uint4 c; uint2 k;
    k.x = k0; k.y = k1; c.x = c0; c.y = c1; c.z = c2; c.w = c3;
    const uint4 r = curand_Philox4x32_10(c, k);
    printf("%u %u %u %u\n", r.x, r.y, r.z, r.w);
  }
  return 0;
}
