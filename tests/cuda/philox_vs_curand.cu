// Test program (not product): the product's Philox4x32-10 (rms_internal.cuh) beside cuRAND's Philox4_32_10 on the same
// (key, counter).  cuRAND: curand_init(seed, subsequence, offset) sets key = (seed_lo, seed_hi) and counter =
// (offset / 4 lo, offset / 4 hi, subsequence lo, subsequence hi); curand4() returns the block of that counter.
// Prints n lines "a0 a1 a2 a3 b0 b1 b2 b3" (ours, cuRAND's) in hex.
#include <cstdio>
#include <curand_kernel.h>

#include "../../paper_2012_06478_b200/csrc/rms_internal.cuh"

__global__ void both(rms_philox_keys rk, unsigned long long seed, int n, uint32_t* out)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    // a spread of counters: offset / 4 = 7919 t + 1 (crosses 2^32 for large t * stride), subsequence = 104729 t * 2^20 + 3
    const unsigned long long c01 = 7919ull * t * 1000003ull + 1ull, c23 = (104729ull * t << 20) + 3ull;
    uint32_t a0, a1, a2, a3;
    rms_philox(rk, (uint32_t)c01, (uint32_t)(c01 >> 32), (uint32_t)c23, (uint32_t)(c23 >> 32), a0, a1, a2, a3);
    curandStatePhilox4_32_10_t st;
    curand_init(seed, c23, 4ull * c01, &st);
    const uint4 b = curand4(&st);
    uint32_t* o = out + 8 * t;
    o[0] = a0; o[1] = a1; o[2] = a2; o[3] = a3; o[4] = b.x; o[5] = b.y; o[6] = b.z; o[7] = b.w;
}

int main()
{
    const int n = 4096;
    const unsigned long long seed = 0x123456789ABCDEF1ull;
    uint32_t* d = nullptr;
    if (cudaMalloc(&d, n * 8 * sizeof(uint32_t)) != cudaSuccess) return 2;
    both<<<(n + 127) / 128, 128>>>(rms_make_keys(seed), seed, n, d);
    static uint32_t h[4096 * 8];
    if (cudaMemcpy(h, d, sizeof h, cudaMemcpyDeviceToHost) != cudaSuccess) return 3;
    for (int t = 0; t < n; ++t)
        printf("%08x %08x %08x %08x %08x %08x %08x %08x\n", h[8 * t], h[8 * t + 1], h[8 * t + 2], h[8 * t + 3], h[8 * t + 4],
               h[8 * t + 5], h[8 * t + 6], h[8 * t + 7]);
    return 0;
}
