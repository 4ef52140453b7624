// Host-side driver around the CUDA toolkit's own Philox4x32-10 round function
// (curand_philox4x32_x.h has a host branch).  Used only by tests/test_oracle_philox.py as an
// INDEPENDENT implementation to pin the oracle's generator; prints "c0 c1 c2 c3 k0 k1 -> x0 x1 x2 x3".
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>
#define QUALIFIERS static inline __host__ __device__
#include <curand_philox4x32_x.h>

int main(int argc, char **argv) {
  unsigned long long s = 0x9E3779B97F4A7C15ull;
  int n = argc > 1 ? atoi(argv[1]) : 64;
  for (int i = 0; i < n; ++i) {
    unsigned int v[6];
    for (int j = 0; j < 6; ++j) {  // splitmix64 to make arbitrary counters / keys
      s += 0x9E3779B97F4A7C15ull;
      unsigned long long z = s;
      z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
      z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
      z = z ^ (z >> 31);
      v[j] = (unsigned int)(z >> 16);
    }
    uint4 c = make_uint4(v[0], v[1], v[2], v[3]);
    uint2 k = make_uint2(v[4], v[5]);
    uint4 x = curand_Philox4x32_10(c, k);
    printf("%08x %08x %08x %08x %08x %08x -> %08x %08x %08x %08x\n", c.x, c.y, c.z, c.w, k.x, k.y, x.x, x.y, x.z, x.w);
  }
  return 0;
}
