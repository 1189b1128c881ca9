// pn_philox.cuh -- Philox4x64-10 (Salmon et al., SC'11) as a device function, in the stream layout of
// numpy.random.Philox: raw word e of a keyed stream is word (e & 3) of Philox(counter = (e >> 2) + 1, key), and a
// double in [0, 1) is (word >> 11) * 2^-53.  Used by pn_gen.cu (initial data) and pn_check.cu (subset selection).
// Shares nothing with oracle/ (which writes the same generator out in plain C with 128-bit products).
#pragma once
#include <cuda_runtime.h>

#define PHILOX_M0 0xD2E7470EE14C6C93ULL
#define PHILOX_M1 0xCA5A826395121157ULL
#define PHILOX_W0 0x9E3779B97F4A7C15ULL
#define PHILOX_W1 0xBB67AE8584CAA73BULL

// all four words of Philox4x64-10(counter = blk + 1, key): raw words 4 blk ... 4 blk + 3 of the stream
__device__ __forceinline__ void gen_block(unsigned long long k0, unsigned long long k1, unsigned long long blk,
                                          unsigned long long (&w)[4])
{
    unsigned long long c0 = blk + 1ull, c1 = 0ull, c2 = 0ull, c3 = 0ull;
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += PHILOX_W0; k1 += PHILOX_W1; }
        const unsigned long long hi0 = __umul64hi(PHILOX_M0, c0), lo0 = PHILOX_M0 * c0;
        const unsigned long long hi1 = __umul64hi(PHILOX_M1, c2), lo1 = PHILOX_M1 * c2;
        const unsigned long long n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
}

// word (e & 3) of Philox4x64-10(counter = (e >> 2) + 1, key)
__device__ __forceinline__ unsigned long long gen_raw(unsigned long long k0, unsigned long long k1, unsigned long long e)
{
    unsigned long long c0 = (e >> 2) + 1ull, c1 = 0ull, c2 = 0ull, c3 = 0ull;
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += PHILOX_W0; k1 += PHILOX_W1; }
        const unsigned long long hi0 = __umul64hi(PHILOX_M0, c0), lo0 = PHILOX_M0 * c0;
        const unsigned long long hi1 = __umul64hi(PHILOX_M1, c2), lo1 = PHILOX_M1 * c2;
        const unsigned long long n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    }
    const unsigned w = (unsigned)(e & 3ull);
    return w == 0 ? c0 : (w == 1 ? c1 : (w == 2 ? c2 : c3));
}
__device__ __forceinline__ double gen_uniform(unsigned long long k0, unsigned long long k1, unsigned long long e)
{
    return (double)(gen_raw(k0, k1, e) >> 11) * (1.0 / 9007199254740992.0);
}
