// Test helper: the CUDA toolkit's own Philox4x32-10 (curand_philox4x32_x.h), compiled for the
// host with g++, as a LIBRARY cross-check of the oracle's C1 (tests/test_oracle_philox.py).
// Reads "c0 c1 c2 c3 k0 k1" (hex) per line on stdin, writes "o0 o1 o2 o3" (hex) per line.
#include <cuda_runtime.h>
#define QUALIFIERS static inline
#include <curand_philox4x32_x.h>
#include <cstdio>
int main() {
    unsigned c0, c1, c2, c3, k0, k1;
    while (scanf("%x %x %x %x %x %x", &c0, &c1, &c2, &c3, &k0, &k1) == 6) {
        uint4 o = curand_Philox4x32_10(make_uint4(c0, c1, c2, c3), make_uint2(k0, k1));
        printf("%08x %08x %08x %08x\n", o.x, o.y, o.z, o.w);
    }
    return 0;
}
