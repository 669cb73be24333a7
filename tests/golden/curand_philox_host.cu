// Independent known-answer source for Philox4x32-10: NVIDIA's own implementation in the
// CUDA toolkit header curand_philox4x32_x.h, compiled for the HOST (the header carries a
// host branch).  Reads "c0 c1 c2 c3 k0 k1" lines (hex) on stdin, prints the four output
// words.  Used by tests/test_oracle_elementary.py; holds none of our code.
#include <cstdio>
#include <cuda_runtime.h>
#define QUALIFIERS static inline __host__ __device__
#include <curand_philox4x32_x.h>

int main() {
    unsigned c0, c1, c2, c3, k0, k1;
    while (std::scanf("%x %x %x %x %x %x", &c0, &c1, &c2, &c3, &k0, &k1) == 6) {
        uint4 c = make_uint4(c0, c1, c2, c3);
        uint2 k = make_uint2(k0, k1);
        uint4 r = curand_Philox4x32_10(c, k);
        std::printf("%08x %08x %08x %08x\n", r.x, r.y, r.z, r.w);
    }
    return 0;
}
