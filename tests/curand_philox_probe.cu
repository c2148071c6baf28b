// Test infrastructure (tests/test_gpu_curand_crosscheck.py): prints the four 32-bit words cuRAND's Philox4x32-10 device
// generator returns for (seed, subsequence, offset) triples given on the command line -- a third, independent
// implementation to check the oracle's Philox against (pin P1).
#include <cstdio>
#include <cstdlib>
#include <curand_kernel.h>

__global__ void probe(unsigned long long seed, unsigned long long subsequence, unsigned long long offset, unsigned int *out)
{
    curandStatePhilox4_32_10_t st;
    curand_init(seed, subsequence, offset, &st);
    const uint4 r = curand4(&st);
    out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}

int main(int argc, char **argv)
{
    unsigned int *d, h[4];
    if (cudaMalloc(&d, 16) != cudaSuccess) return 2;
    for (int a = 1; a + 2 < argc; a += 3) {
        const unsigned long long seed = strtoull(argv[a], nullptr, 0), sub = strtoull(argv[a + 1], nullptr, 0),
                                 off = strtoull(argv[a + 2], nullptr, 0);
        probe<<<1, 1>>>(seed, sub, off, d);
        if (cudaMemcpy(h, d, 16, cudaMemcpyDeviceToHost) != cudaSuccess) return 3;
        printf("%llu %llu %llu %08x %08x %08x %08x\n", seed, sub, off, h[0], h[1], h[2], h[3]);
    }
    return 0;
}
