// pn_gen.cu -- on-device initial data for sm_100a: random spin orientations uniform on the sphere, random
// mass ratios and spin magnitudes, L^ = (0,0,1), M = 1.
//
// Counter-based, so a system's initial state is a pure function of (key, ensemble size, system index):
// seven uniform variates per system, variate column k = the k-th length-n_total block of ONE Philox4x64-10
// stream laid out like numpy.random.Philox (counter incremented before every block of four 64-bit words,
// double = (word >> 11) * 2^-53), so that pn_generate reproduces paper_0908_3889_b200/workloads.generate
// to the last bits that do not depend on sin/cos.  Any chunk [first, first+count) of an ensemble can be
// generated on its own (chunked 10^8-system runs, multi-GPU shards).
//
// HBM-bound: 96 B written per system, nothing read.  One thread per system writes its AoS row into a
// shared-memory tile; the tile leaves with one TMA bulk store (cp.async.bulk.global.shared::cta) per
// array, so global writes are full 16-byte-aligned bursts.
// This file shares nothing with oracle/.
#include <cstdint>
#include "pn_internal.h"

#define GEN_TILE 256

#include "pn_gen.cuh"

template <bool SHARE>
__global__ void __launch_bounds__(GEN_TILE) pn_generate_kernel(const GenSpec* __restrict__ specs, long long n_total,
                                                               long long first, long long count, int tiles_per_ens,
                                                               double* __restrict__ init_states, double* __restrict__ masses)
{
    __shared__ __align__(128) double tile_y[GEN_TILE * 10];
    __shared__ __align__(128) double tile_m[GEN_TILE * 2];
    const int ens = blockIdx.x / tiles_per_ens;
    const long long j0 = (long long)(blockIdx.x - ens * tiles_per_ens) * GEN_TILE;      // first row of this tile within the chunk
    const int cnt = (int)min((long long)GEN_TILE, count - j0);
    const GenSpec sp = specs[ens];
    const int t = threadIdx.x;
    // SHARE (n_total and first multiples of 4): the four systems 4q .. 4q+3 read the four words of the SAME Philox
    // block in every variate column, so thread r of a quad evaluates only the blocks of columns r and r + 4 and the
    // quad exchanges words through shared memory: 7 blocks per quad instead of 28.
    __shared__ unsigned long long words[SHARE ? GEN_TILE / 4 * 7 * 4 : 1];
    if (SHARE) {
        const unsigned long long N = (unsigned long long)n_total;
        const unsigned long long blk0 = (unsigned long long)(first + j0 + t) >> 2;     // block of this quad in column 0
        const int q = t >> 2, r = t & 3;
#pragma unroll
        for (int kk = 0; kk < 2; ++kk) {
            const int k = r + 4 * kk;
            if (k < 7) {
                unsigned long long w[4];
                gen_block(sp.key0, sp.key1, (unsigned long long)k * (N >> 2) + blk0, w);
#pragma unroll
                for (int x = 0; x < 4; ++x) words[(q * 7 + k) * 4 + x] = w[x];
            }
        }
        __syncthreads();
    }
    if (t < cnt) {
        const unsigned long long i = (unsigned long long)(first + j0 + t), N = (unsigned long long)n_total;
        double u[7];
#pragma unroll
        for (int k = 0; k < 7; ++k) {
            if (SHARE) u[k] = (double)(words[((t >> 2) * 7 + k) * 4 + (t & 3)] >> 11) * (1.0 / 9007199254740992.0);
            else u[k] = gen_uniform(sp.key0, sp.key1, (unsigned long long)k * N + i);
        }
        double yy[10], m1, m2;
        gen_system(sp, u, yy, m1, m2);
        double* y = tile_y + t * 10;
#pragma unroll
        for (int c = 0; c < 10; ++c) y[c] = yy[c];
        tile_m[2 * t] = m1; tile_m[2 * t + 1] = m2;
    }
    // generic-proxy writes -> visible to the async proxy, then one bulk store per array by one thread
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    if (t == 0) {
        const long long row = (long long)ens * count + j0;
        const uint32_t sy = (uint32_t)__cvta_generic_to_shared(tile_y), sm = (uint32_t)__cvta_generic_to_shared(tile_m);
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(init_states + row * 10), "r"(sy),
                     "r"((uint32_t)cnt * 80u)
                     : "memory");
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(masses + row * 2), "r"(sm),
                     "r"((uint32_t)cnt * 16u)
                     : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");     // the block may exit only after the stores have left smem
    }
}

cudaError_t pn_launch_generate(const void* specs_dev, int n_ens, long long n_total, long long first, long long count,
                               double* init_states, double* masses, cudaStream_t s)
{
    if (count <= 0 || n_ens <= 0) return cudaSuccess;
    const long long tiles = (count + GEN_TILE - 1) / GEN_TILE;
    if (tiles * n_ens > 0x7fffffffLL) return cudaErrorInvalidValue;
    if ((n_total & 3) == 0 && (first & 3) == 0)
        pn_generate_kernel<true><<<(unsigned)(tiles * n_ens), GEN_TILE, 0, s>>>((const GenSpec*)specs_dev, n_total, first, count,
                                                                                (int)tiles, init_states, masses);
    else
        pn_generate_kernel<false><<<(unsigned)(tiles * n_ens), GEN_TILE, 0, s>>>((const GenSpec*)specs_dev, n_total, first, count,
                                                                                 (int)tiles, init_states, masses);
    ++g_pn_launches;
    return cudaGetLastError();
}
