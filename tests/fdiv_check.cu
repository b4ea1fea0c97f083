// fdiv_check.cu -- is the seeded division of csrc/vs_div.cuh (k_raster_direct's depth key) the IEEE division?
// For EVERY integer divisor a small triangle can have (A2 = 1 .. 2^24) and 64 numerators each -- random mantissas at
// exponents spread over what f_i q_i can produce, plus the numerators next to exact multiples of the divisor (quotients next to
// a rounding boundary) -- the bits must equal __fdiv_rn's.  Prints "fdiv_check ok" or the first mismatches.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#include "../paper_2409_02482_b200/csrc/vs_div.cuh"

__device__ __forceinline__ uint32_t mix(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
    return x;
}

__global__ void k_check(unsigned long long* bad, float* first)
{
    const uint32_t a2 = blockIdx.x * blockDim.x + threadIdx.x + 1u;   // 1 .. 2^24
    const float b = (float)a2;
    const float r = vs_rcp_seed(b);
    for (uint32_t i = 0; i < 64; ++i) {
        float a;
        const uint32_t h = mix(a2 * 64u + i);
        if (i < 48) {
            // exponent in [2^-24, 2^36): q_i in [2^-24, 2^12] times f_i in [1, 2^24]
            const uint32_t e = 127u - 24u + (mix(h) % 60u);
            a = __uint_as_float((e << 23) | (h & 0x7FFFFFu));
        } else {
            // next to k * b for a random quotient k: the remainder is a few ulps, the hard case for the correction step
            const float k = __uint_as_float(((127u - 6u + (h % 12u)) << 23) | (mix(h) & 0x7FFFFFu));
            const float p = __fmul_rn(k, b);
            a = __uint_as_float(__float_as_uint(p) + (int)(i - 56));
        }
        const float want = __fdiv_rn(a, b);
        const float got = vs_div_seeded(a, b, r);
        if (__float_as_uint(want) != __float_as_uint(got)) {
            if (atomicAdd(bad, 1ull) == 0ull) { first[0] = a; first[1] = b; first[2] = want; first[3] = got; }
        }
    }
}

int main()
{
    unsigned long long* bad; float* first;
    if (cudaMalloc(&bad, 8) != cudaSuccess || cudaMalloc(&first, 16) != cudaSuccess) { printf("no device\n"); return 2; }
    cudaMemset(bad, 0, 8); cudaMemset(first, 0, 16);
    k_check<<<(1u << 24) / 256, 256>>>(bad, first);
    unsigned long long h = 0; float f[4];
    if (cudaMemcpy(&h, bad, 8, cudaMemcpyDeviceToHost) != cudaSuccess) { printf("kernel failed: %s\n", cudaGetErrorString(cudaGetLastError())); return 2; }
    cudaMemcpy(f, first, 16, cudaMemcpyDeviceToHost);
    if (h) { printf("fdiv_check FAILED: %llu mismatches, first %.9g / %.9g: __fdiv_rn %.9g, seeded %.9g\n", h, f[0], f[1], f[2], f[3]); return 1; }
    printf("fdiv_check ok: 2^24 divisors x 64 numerators, seeded division == __fdiv_rn bit for bit\n");
    return 0;
}
