// pn_check.cu -- the paper's cross-check on the device: a pseudo-random subset of a
// batch is re-integrated in FP64 and the final unit dot products are compared with the results under test.
// This file holds the three small kernels around the re-integration (which is pn_integrate_ex itself):
//   selection  system i is in the subset iff u_i < fraction, u_i = element i of the keyed Philox4x64-10 stream
//              (pn_philox.cuh); an ordered stream compaction (count, scan, scatter), so the index list is sorted;
//   gather     the selected rows of init_states / masses into dense AoS arrays;
//   compare    per dot product the largest |d(checked) - d(reference)| and the lowest index where it occurs,
//              the largest relative deviation of the final time, the number of failed reference systems;
//              one block, fixed reduction order: deterministic.
// Shares nothing with oracle/.
#include <cstdint>
#include "pn_internal.h"
#include "pn_philox.cuh"
#include "pn_dots.cuh"

// ---- selection: ordered stream compaction of {i : u_i < fraction}, three small kernels --------------------------
//   count    every thread tests 8 consecutive indices (two Philox blocks give their 8 words), block totals;
//   scan     exclusive scan of the block totals (one block, running carry), grand total -> n_selected;
//   scatter  the flags are recomputed, ranked inside the block (warp shuffles + shared memory) and the selected
//            indices written at block offset + rank: ascending order, no atomics, deterministic.
#define CHK_SEL_THREADS 256
#define CHK_SEL_PER 8
#define CHK_SEL_TILE (CHK_SEL_THREADS * CHK_SEL_PER)

// bit j of the result: index i0 + j is selected (i0 a multiple of 8)
__device__ __forceinline__ unsigned chk_flags8(unsigned long long k0, unsigned long long k1, long long i0, long long n, double fraction)
{
    unsigned f = 0u;
    if (i0 >= n) return f;
    unsigned long long w[4];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        gen_block(k0, k1, ((unsigned long long)i0 >> 2) + h, w);
#pragma unroll
        for (int x = 0; x < 4; ++x) {
            const double u = (double)(w[x] >> 11) * (1.0 / 9007199254740992.0);
            if (i0 + 4 * h + x < n && u < fraction) f |= 1u << (4 * h + x);
        }
    }
    return f;
}

// exclusive prefix of v over the block's threads; total in *tot (all threads)
__device__ __forceinline__ unsigned chk_block_exscan(unsigned v, unsigned* smem /*[33]*/, unsigned* tot)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) smem[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        const unsigned w = lane < CHK_SEL_THREADS / 32 ? smem[lane] : 0u;
        unsigned wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, wi, o); if (lane >= o) wi += t; }
        if (lane < CHK_SEL_THREADS / 32) smem[lane] = wi - w;
        if (lane == 31) smem[32] = wi;
    }
    __syncthreads();
    *tot = smem[32];
    return smem[warp] + inc - v;
}

__global__ void __launch_bounds__(CHK_SEL_THREADS) pn_check_count_kernel(long long n, double fraction, unsigned long long k0,
                                                                         unsigned long long k1, long long* __restrict__ block_counts)
{
    __shared__ unsigned sm[33];
    const long long i0 = (long long)blockIdx.x * CHK_SEL_TILE + (long long)threadIdx.x * CHK_SEL_PER;
    unsigned tot;
    chk_block_exscan((unsigned)__popc(chk_flags8(k0, k1, i0, n, fraction)), sm, &tot);
    if (threadIdx.x == 0) block_counts[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(1024) pn_check_scan_kernel(long long* __restrict__ block_counts, int n_blocks, long long* __restrict__ n_selected)
{
    __shared__ long long warp_tot[32];
    __shared__ long long carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int base = 0; base < n_blocks; base += 1024) {
        const int b = base + threadIdx.x;
        const long long v = b < n_blocks ? block_counts[b] : 0;
        long long inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const long long t = __shfl_up_sync(0xffffffffu, inc, o); if ((threadIdx.x & 31) >= o) inc += t; }
        if ((threadIdx.x & 31) == 31) warp_tot[threadIdx.x >> 5] = inc;
        __syncthreads();
        if (threadIdx.x < 32) {
            const long long w = warp_tot[threadIdx.x];
            long long wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const long long t = __shfl_up_sync(0xffffffffu, wi, o); if (threadIdx.x >= o) wi += t; }
            warp_tot[threadIdx.x] = wi - w;
        }
        __syncthreads();
        const long long carry = carry_s;
        if (b < n_blocks) block_counts[b] = carry + warp_tot[threadIdx.x >> 5] + inc - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry_s = carry + warp_tot[31] + inc;
        __syncthreads();
    }
    if (threadIdx.x == 0) *n_selected = carry_s;
}

__global__ void __launch_bounds__(CHK_SEL_THREADS) pn_check_scatter_kernel(long long n, double fraction, unsigned long long k0,
                                                                           unsigned long long k1, const long long* __restrict__ block_offsets,
                                                                           long long* __restrict__ indices)
{
    __shared__ unsigned sm[33];
    const long long i0 = (long long)blockIdx.x * CHK_SEL_TILE + (long long)threadIdx.x * CHK_SEL_PER;
    unsigned f = chk_flags8(k0, k1, i0, n, fraction), tot;
    long long pos = block_offsets[blockIdx.x] + chk_block_exscan((unsigned)__popc(f), sm, &tot);
    while (f) {
        const int j = __ffs(f) - 1;
        f &= f - 1u;
        indices[pos++] = i0 + j;
    }
}

size_t pn_check_select_temp_bytes(long long n)
{
    return sizeof(long long) * (size_t)((n + CHK_SEL_TILE - 1) / CHK_SEL_TILE + 1);
}

cudaError_t pn_launch_check_select(long long n, double fraction, unsigned long long k0, unsigned long long k1,
                                   long long* indices, long long* n_selected, void* temp, cudaStream_t s)
{
    const long long nb = (n + CHK_SEL_TILE - 1) / CHK_SEL_TILE;
    if (nb > 0x7fffffffLL) return cudaErrorInvalidValue;
    long long* block_counts = (long long*)temp;
    if (nb == 0) return cudaMemsetAsync(n_selected, 0, sizeof(long long), s);
    pn_check_count_kernel<<<(unsigned)nb, CHK_SEL_THREADS, 0, s>>>(n, fraction, k0, k1, block_counts);
    pn_check_scan_kernel<<<1, 1024, 0, s>>>(block_counts, (int)nb, n_selected);
    pn_check_scatter_kernel<<<(unsigned)nb, CHK_SEL_THREADS, 0, s>>>(n, fraction, k0, k1, block_counts, indices);
    g_pn_launches += 3;
    return cudaGetLastError();
}

__global__ void pn_check_gather_kernel(const long long* __restrict__ indices, long long m, const double* __restrict__ init,
                                       const double* __restrict__ masses, double* __restrict__ sub_init,
                                       double* __restrict__ sub_masses)
{
    // one thread per (subset row, column): 12 doubles per row
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= m * 12) return;
    const long long j = e / 12;
    const int c = (int)(e - j * 12);
    const long long i = indices[j];
    if (c < 10) sub_init[j * 10 + c] = init[i * 10 + c];
    else sub_masses[j * 2 + (c - 10)] = masses[i * 2 + (c - 10)];
}

cudaError_t pn_launch_check_gather(const long long* indices, long long m, const double* init, const double* masses,
                                   double* sub_init, double* sub_masses, cudaStream_t s)
{
    if (m <= 0) return cudaSuccess;
    pn_check_gather_kernel<<<(unsigned)((m * 12 + 255) / 256), 256, 0, s>>>(indices, m, init, masses, sub_init, sub_masses);
    ++g_pn_launches;
    return cudaGetLastError();
}

__device__ __forceinline__ void chk_unit_dots(const double* __restrict__ row, double (&d)[3])
{
    const double v[9] = {row[1], row[2], row[3], row[4], row[5], row[6], row[7], row[8], row[9]};
    bool ok[3];
    pn_unit_dots(v, d, ok);
#pragma unroll
    for (int k = 0; k < 3; ++k) d[k] = ok[k] ? d[k] : nan("");
}

// result record (device and host): [0..2] max deviation per dot product, [3] max relative time deviation,
// then as long long: [4..6] index of the worst system per dot product (-1: none), [7] failed reference systems
#define CHK_THREADS 512
__global__ void __launch_bounds__(CHK_THREADS) pn_check_compare_kernel(const long long* __restrict__ indices, long long m,
                                                                       const double* __restrict__ fin, const double* __restrict__ times,
                                                                       const double* __restrict__ ref_fin, const double* __restrict__ ref_times,
                                                                       const int* __restrict__ ref_steps, double* __restrict__ out)
{
    __shared__ double s_dev[4][CHK_THREADS];
    __shared__ long long s_idx[3][CHK_THREADS];
    __shared__ unsigned s_failed;
    if (threadIdx.x == 0) s_failed = 0u;
    __syncthreads();
    double dev[4] = {-1.0, -1.0, -1.0, 0.0};
    long long widx[3] = {-1, -1, -1};
    unsigned failed = 0;
    // thread t looks at subset rows t, t + 512, ...: ascending indices, so ">" keeps the lowest index of a tie
    for (long long j = threadIdx.x; j < m; j += CHK_THREADS) {
        if (ref_steps[j] <= 0) { ++failed; continue; }
        const long long i = indices[j];
        double dc[3], dr[3];
        chk_unit_dots(fin + i * 10, dc);
        chk_unit_dots(ref_fin + j * 10, dr);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double e = fabs(dc[k] - dr[k]);
            if (e > dev[k]) { dev[k] = e; widx[k] = i; }          // false for NaN
        }
        if (times) {
            const double e = fabs(times[i] / ref_times[j] - 1.0);
            if (e > dev[3]) dev[3] = e;
        }
    }
    if (failed) atomicAdd(&s_failed, failed);
#pragma unroll
    for (int k = 0; k < 4; ++k) s_dev[k][threadIdx.x] = dev[k];
#pragma unroll
    for (int k = 0; k < 3; ++k) s_idx[k][threadIdx.x] = widx[k];
    __syncthreads();
    for (int o = CHK_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double a = s_dev[k][threadIdx.x], b = s_dev[k][threadIdx.x + o];
                const long long ia = s_idx[k][threadIdx.x], ib = s_idx[k][threadIdx.x + o];
                // larger deviation wins; on a tie the lower system index
                if (b > a || (b == a && ib >= 0 && (ia < 0 || ib < ia))) { s_dev[k][threadIdx.x] = b; s_idx[k][threadIdx.x] = ib; }
            }
            s_dev[3][threadIdx.x] = fmax(s_dev[3][threadIdx.x], s_dev[3][threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        long long* oi = reinterpret_cast<long long*>(out);
        for (int k = 0; k < 3; ++k) { out[k] = s_idx[k][0] >= 0 ? s_dev[k][0] : 0.0; oi[4 + k] = s_idx[k][0]; }
        out[3] = s_dev[3][0];
        oi[7] = (long long)s_failed;
    }
}

cudaError_t pn_launch_check_compare(const long long* indices, long long m, const double* fin, const double* times,
                                    const double* ref_fin, const double* ref_times, const int* ref_steps, double* out,
                                    cudaStream_t s)
{
    pn_check_compare_kernel<<<1, CHK_THREADS, 0, s>>>(indices, m, fin, times, ref_fin, ref_times, ref_steps, out);
    ++g_pn_launches;
    return cudaGetLastError();
}
