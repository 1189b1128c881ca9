// pn_check.cu -- the paper's cross-check on the device: a pseudo-random subset of a
// batch is re-integrated in FP64 and the final unit dot products are compared with the results under test.
// This file holds the three small kernels around the re-integration (which is pn_integrate_ex itself):
//   selection  system i is in the subset iff u_i < fraction, u_i = element i of the keyed Philox4x64-10 stream
//              (pn_philox.cuh); cub::DeviceSelect::If over a counting iterator, so the index list is sorted;
//   gather     the selected rows of init_states / masses into dense AoS arrays;
//   compare    per dot product the largest |d(checked) - d(reference)| and the lowest index where it occurs,
//              the largest relative deviation of the final time, the number of failed reference systems;
//              one block, fixed reduction order: deterministic.
// Shares nothing with oracle/.
#include <cstdint>
#include <cub/device/device_select.cuh>
#include <thrust/iterator/counting_iterator.h>
#include "pn_internal.h"
#include "pn_philox.cuh"

struct CheckSelectOp {
    unsigned long long k0, k1;
    double fraction;
    __device__ __forceinline__ bool operator()(const long long& i) const
    {
        return gen_uniform(k0, k1, (unsigned long long)i) < fraction;
    }
};

size_t pn_check_select_temp_bytes(long long n)
{
    size_t bytes = 0;
    thrust::counting_iterator<long long> it(0);
    CheckSelectOp op{0ull, 0ull, 0.0};
    cub::DeviceSelect::If(nullptr, bytes, it, (long long*)nullptr, (long long*)nullptr, n, op);
    return bytes;
}

cudaError_t pn_launch_check_select(long long n, double fraction, unsigned long long k0, unsigned long long k1,
                                   long long* indices, long long* n_selected, void* temp, size_t temp_bytes, cudaStream_t s)
{
    thrust::counting_iterator<long long> it(0);
    CheckSelectOp op{k0, k1, fraction};
    g_pn_launches += 2;      // cub's select passes (library kernels, counted approximately)
    return cub::DeviceSelect::If(temp, temp_bytes, it, indices, n_selected, n, op, s);
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
    const double s1x = row[1], s1y = row[2], s1z = row[3], s2x = row[4], s2y = row[5], s2z = row[6];
    const double lx = row[7], ly = row[8], lz = row[9];
    const double n1 = sqrt(s1x * s1x + s1y * s1y + s1z * s1z), n2 = sqrt(s2x * s2x + s2y * s2y + s2z * s2z);
    const double nl = sqrt(lx * lx + ly * ly + lz * lz);
    d[0] = (n1 > 0 && n2 > 0) ? (s1x * s2x + s1y * s2y + s1z * s2z) / (n1 * n2) : nan("");
    d[1] = (n1 > 0 && nl > 0) ? (s1x * lx + s1y * ly + s1z * lz) / (n1 * nl) : nan("");
    d[2] = (n2 > 0 && nl > 0) ? (s2x * lx + s2y * ly + s2z * lz) / (n2 * nl) : nan("");
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
