// Pin P1(i): NVIDIA's own Philox4x32-10 (CUDA toolkit header curand_philox4x32_x.h, host
// path of mulhilo32) used as an independent implementation to check oracle/ising_oracle.c.
// Reads "c0 c1 c2 c3 k0 k1" (hex) per line on stdin, prints the four output words.
// Host-only program: launches no kernel and needs no GPU.
#include <cstdio>
#include <cuda_runtime.h>
#define QUALIFIERS static inline __host__ __device__
#include <curand_philox4x32_x.h>

int main()
{
    unsigned c0, c1, c2, c3, k0, k1;
    while (scanf("%x %x %x %x %x %x", &c0, &c1, &c2, &c3, &k0, &k1) == 6) {
        uint4 r = curand_Philox4x32_10(make_uint4(c0, c1, c2, c3), make_uint2(k0, k1));
        printf("%08x %08x %08x %08x\n", r.x, r.y, r.z, r.w);
    }
    return 0;
}
