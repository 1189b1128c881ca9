// pn_aux.cu -- staging (AoS <-> SoA), dot-product histogram and FMA-peak kernels of libpn_b200.
#include <cstdint>
#include <cub/device/device_radix_sort.cuh>
#include "pn_internal.h"

// ------------------------------------------------------------------------------------------------
// AoS [n][W]  <->  SoA [W][n], coalesced on both sides through a shared-memory tile (stage-in /
// stage-out; the paper transfers state only at start and end).
// ------------------------------------------------------------------------------------------------
#define PN_TILE 256
template <int W, bool TO_SOA>
__global__ void __launch_bounds__(PN_TILE) pn_transpose_kernel(const double* __restrict__ in, double* __restrict__ out, int n)
{
    __shared__ double tile[PN_TILE * W];
    const int base = blockIdx.x * PN_TILE;
    const int cnt = min(PN_TILE, n - base);
    if (TO_SOA) {
        for (int e = threadIdx.x; e < cnt * W; e += PN_TILE) tile[e] = in[(size_t)base * W + e];
        __syncthreads();
        if (threadIdx.x < cnt)
#pragma unroll
            for (int c = 0; c < W; ++c) out[(size_t)c * n + base + threadIdx.x] = tile[threadIdx.x * W + c];
    } else {
        if (threadIdx.x < cnt)
#pragma unroll
            for (int c = 0; c < W; ++c) tile[threadIdx.x * W + c] = in[(size_t)c * n + base + threadIdx.x];
        __syncthreads();
        for (int e = threadIdx.x; e < cnt * W; e += PN_TILE) out[(size_t)base * W + e] = tile[e];
    }
}

template <bool TO_SOA>
static cudaError_t launch_transpose(const double* in, double* out, int n, int width, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    const int grid = (n + PN_TILE - 1) / PN_TILE;
    if (width == 10) pn_transpose_kernel<10, TO_SOA><<<grid, PN_TILE, 0, s>>>(in, out, n);
    else if (width == 2) pn_transpose_kernel<2, TO_SOA><<<grid, PN_TILE, 0, s>>>(in, out, n);
    else return cudaErrorInvalidValue;
    ++g_pn_launches;
    return cudaGetLastError();
}
cudaError_t pn_launch_aos_to_soa(const double* aos, double* soa, int n, int width, cudaStream_t s) { return launch_transpose<true>(aos, soa, n, width, s); }
cudaError_t pn_launch_soa_to_aos(const double* soa, double* aos, int n, int width, cudaStream_t s) { return launch_transpose<false>(soa, aos, n, width, s); }

// ------------------------------------------------------------------------------------------------
// Histograms of S1^.S2^, S1^.L^, S2^.L^ (R14).
// One system per thread; AoS input is read through a shared tile so global loads stay coalesced.
// Counting: lanes that hit the same bin are merged with __match_any_sync and the leader adds the
// population count to a per-block shared-memory histogram; blocks flush with one 64-bit global atomic
// per non-empty bin.  HBM-bound: 80 B read per system.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int pn_bin_of(double d, int bins)
{
    int b = (int)floor((d + 1.0) * (double)bins * 0.5);
    return max(0, min(bins - 1, b));
}

template <bool SOA, bool SMEM_HIST>
__global__ void __launch_bounds__(PN_TILE) pn_histogram_kernel(const double* __restrict__ st, long long n, int bins,
                                                               unsigned long long* __restrict__ counts,
                                                               unsigned long long* __restrict__ skipped)
{
    extern __shared__ unsigned char smem_raw[];
    double* tile = reinterpret_cast<double*>(smem_raw);                       // AoS only: PN_TILE*10 doubles
    unsigned* hist = reinterpret_cast<unsigned*>(smem_raw + (SOA ? 0 : PN_TILE * 10 * sizeof(double)));
    __shared__ unsigned skip_s[3];
    if (SMEM_HIST) for (int b = threadIdx.x; b < 3 * bins; b += PN_TILE) hist[b] = 0u;
    if (threadIdx.x < 3) skip_s[threadIdx.x] = 0u;
    __syncthreads();

    const long long ntiles = (n + PN_TILE - 1) / PN_TILE;
    for (long long tIdx = blockIdx.x; tIdx < ntiles; tIdx += gridDim.x) {
        const long long base = tIdx * PN_TILE;
        const int cnt = (int)min((long long)PN_TILE, n - base);
        double v[9];
        const bool have = threadIdx.x < cnt;
        if (SOA) {
            if (have)
#pragma unroll
                for (int c = 0; c < 9; ++c) v[c] = st[(size_t)(c + 1) * n + base + threadIdx.x];
        } else {
            for (int e = threadIdx.x; e < cnt * 10; e += PN_TILE) tile[e] = st[(size_t)base * 10 + e];
            __syncthreads();
            if (have)
#pragma unroll
                for (int c = 0; c < 9; ++c) v[c] = tile[threadIdx.x * 10 + 1 + c];
            __syncthreads();
        }
        int bin[3] = {-1, -1, -1};
        if (have) {
            const double n1 = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
            const double n2 = sqrt(v[3] * v[3] + v[4] * v[4] + v[5] * v[5]);
            const double nl = sqrt(v[6] * v[6] + v[7] * v[7] + v[8] * v[8]);
            const double d[3] = {(v[0] * v[3] + v[1] * v[4] + v[2] * v[5]) / (n1 * n2),
                                 (v[0] * v[6] + v[1] * v[7] + v[2] * v[8]) / (n1 * nl),
                                 (v[3] * v[6] + v[4] * v[7] + v[5] * v[8]) / (n2 * nl)};
            const bool ok[3] = {n1 > 0 && n2 > 0, n1 > 0 && nl > 0, n2 > 0 && nl > 0};
#pragma unroll
            for (int hh = 0; hh < 3; ++hh) {
                if (ok[hh] && isfinite(d[hh])) bin[hh] = pn_bin_of(d[hh], bins);
                else bin[hh] = -2;   // skipped
            }
        }
#pragma unroll
        for (int hh = 0; hh < 3; ++hh) {
            const int b = bin[hh];
            const unsigned peers = __match_any_sync(0xffffffffu, b);
            const bool leader = ((int)(__ffs(peers) - 1) == (int)(threadIdx.x & 31));
            if (leader && b != -1) {
                const unsigned cntp = (unsigned)__popc(peers);
                if (b == -2) atomicAdd(&skip_s[hh], cntp);
                else if (SMEM_HIST) atomicAdd(&hist[hh * bins + b], cntp);
                else atomicAdd(&counts[(size_t)hh * bins + b], (unsigned long long)cntp);
            }
        }
    }
    __syncthreads();
    if (SMEM_HIST)
        for (int b = threadIdx.x; b < 3 * bins; b += PN_TILE)
            if (hist[b]) atomicAdd(&counts[b], (unsigned long long)hist[b]);
    if (threadIdx.x < 3 && skipped && skip_s[threadIdx.x]) atomicAdd(&skipped[threadIdx.x], (unsigned long long)skip_s[threadIdx.x]);
}

cudaError_t pn_launch_histogram(const double* states, int layout_soa, long long n, int bins,
                                unsigned long long* counts, unsigned long long* skipped, cudaStream_t s)
{
    cudaError_t e;
    if ((e = cudaMemsetAsync(counts, 0, sizeof(unsigned long long) * 3 * (size_t)bins, s)) != cudaSuccess) return e;
    if (skipped && (e = cudaMemsetAsync(skipped, 0, sizeof(unsigned long long) * 3, s)) != cudaSuccess) return e;
    if (n <= 0) return cudaSuccess;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long long ntiles = (n + PN_TILE - 1) / PN_TILE;
    const int grid = (int)((ntiles < (long long)sms * 8) ? ntiles : (long long)sms * 8);
    const size_t tile_b = layout_soa ? 0 : PN_TILE * 10 * sizeof(double);
    const size_t hist_b = (size_t)3 * bins * sizeof(unsigned);
    const bool smem_hist = tile_b + hist_b <= 160 * 1024;
    const size_t shm = tile_b + (smem_hist ? hist_b : 0);
#define PN_HIST_LAUNCH(SOA, SH)                                                                                     \
    do {                                                                                                            \
        if (shm > 48 * 1024 &&                                                                                      \
            (e = cudaFuncSetAttribute(pn_histogram_kernel<SOA, SH>, cudaFuncAttributeMaxDynamicSharedMemorySize,    \
                                      (int)shm)) != cudaSuccess)                                                    \
            return e;                                                                                               \
        pn_histogram_kernel<SOA, SH><<<grid, PN_TILE, shm, s>>>(states, n, bins, counts, skipped);                  \
    } while (0)
    if (layout_soa) { if (smem_hist) PN_HIST_LAUNCH(true, true); else PN_HIST_LAUNCH(true, false); }
    else { if (smem_hist) PN_HIST_LAUNCH(false, true); else PN_HIST_LAUNCH(false, false); }
#undef PN_HIST_LAUNCH
    ++g_pn_launches;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Queue ordering by expected cost (default; pn_options.input_order turns it off).  The number of trial steps of
// an inspiral follows the number of precession cycles of the faster-precessing body,
//     key = (4 + 3 m_big/m_small)/eta * (1/(M omega_0) - 1/(M omega_f))        (Eq. (4) over Eq. (1), leading order)
// (log-correlation 0.98 with the measured step counts on C3 and C5).  Issuing the queue longest-first
// (LPT) shortens the drain tail of the persistent grid; results do not depend on the order.
// ------------------------------------------------------------------------------------------------
__global__ void pn_cost_key_kernel(const double* __restrict__ y0, const double* __restrict__ masses, int n,
                                   double omegaf, float* __restrict__ keys, int* __restrict__ idx)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double m1 = masses[i], m2 = masses[(size_t)n + i], M = m1 + m2;
    const double eta = m1 * m2 / (M * M);
    const double big = fmax(m1, m2), small = fmin(m1, m2);
    double key = (4.0 + 3.0 * big / small) / eta * (1.0 / (M * y0[i]) - 1.0 / (M * omegaf));
    if (!(key > 0.0) || !isfinite(key)) key = 0.0;      // bad inputs go last; they are rejected at refill
    keys[i] = (float)key;
    idx[i] = i;
}

size_t pn_cost_order_temp_bytes(int n)
{
    size_t bytes = 0;
    cub::DeviceRadixSort::SortPairsDescending(nullptr, bytes, (const float*)nullptr, (float*)nullptr,
                                              (const int*)nullptr, (int*)nullptr, n);
    return bytes;
}

cudaError_t pn_launch_cost_order(const double* y0_soa, const double* m_soa, int n, double omegaf, float* keys_in,
                                 float* keys_out, int* idx_in, int* idx_out, void* temp, size_t temp_bytes,
                                 cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    pn_cost_key_kernel<<<(n + 255) / 256, 256, 0, s>>>(y0_soa, m_soa, n, omegaf, keys_in, idx_in);
    ++g_pn_launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    e = cub::DeviceRadixSort::SortPairsDescending(temp, temp_bytes, keys_in, keys_out, idx_in, idx_out, n, 0, 32, s);
    g_pn_launches += 3;   // cub's histogram + onesweep passes (library kernels, counted approximately)
    return e;
}

// ------------------------------------------------------------------------------------------------
// FMA peak and operand-port micro-benchmarks: CHAINS independent dependent-FMA chains per thread, no
// memory traffic.  MODE 0: a = a*U + U (one register source, two uniform operands): the denominator of
// the ALU roofline at the clocks the device actually holds.  MODE 1: a = a*x + U (two
// distinct register sources).  MODE 2: a = a*x + z (three distinct register sources).  On sm_100a a DFMA
// issues every 2 cycles per scheduler with <= 2 register sources and every 3 cycles with 3.
// ------------------------------------------------------------------------------------------------
template <typename real, int CHAINS, int MODE>
__global__ void __launch_bounds__(256) pn_fma_peak_kernel(real* out, int iters, long long* clocks, real m, real b)
{
    real a[CHAINS], x[CHAINS], z[CHAINS];
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) {
        a[i] = (real)(threadIdx.x + i) * (real)1e-3;
        x[i] = (real)1 - (real)1e-7 * (real)(threadIdx.x + i) + out[1];
        z[i] = (real)1e-7 * (real)(i + threadIdx.x) + out[2];
    }
    const long long c0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int i = 0; i < CHAINS; ++i) {
                if (MODE == 0) a[i] = a[i] * m + b;
                if (MODE == 1) a[i] = a[i] * x[i] + b;
                if (MODE == 2) a[i] = a[i] * x[i] + z[i];
            }
    }
    const long long c1 = clock64();
    real s = 0;
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) s += a[i];
    if (s == (real)123.456) out[0] = s;
    if (blockIdx.x == 0 && threadIdx.x == 0) clocks[0] = c1 - c0;
}

cudaError_t pn_run_fma_peak(int precision, int mode, double seconds, double* tflops, double* sm_mhz,
                            double* cycles_per_warp_inst)
{
    const int CH = 8;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    void* scratch = nullptr;
    long long* dclk = nullptr;
    cudaError_t e;
    if ((e = cudaMalloc(&scratch, 64)) != cudaSuccess) return e;
    if ((e = cudaMemset(scratch, 0, 64)) != cudaSuccess) { cudaFree(scratch); return e; }
    if ((e = cudaMalloc((void**)&dclk, sizeof(long long))) != cudaSuccess) { cudaFree(scratch); return e; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int block = 256, grid = sms * 4;      // 4 resident blocks per SM = 8 warps per scheduler, one wave
    auto run = [&](int iters, float* ms) {
        cudaEventRecord(e0);
#define PN_PEAK(T, M) pn_fma_peak_kernel<T, CH, M><<<grid, block>>>((T*)scratch, iters, dclk, (T)0.999999, (T)1e-7)
        if (precision == 0) { if (mode == 0) PN_PEAK(double, 0); else if (mode == 1) PN_PEAK(double, 1); else PN_PEAK(double, 2); }
        else { if (mode == 0) PN_PEAK(float, 0); else if (mode == 1) PN_PEAK(float, 1); else PN_PEAK(float, 2); }
#undef PN_PEAK
        ++g_pn_launches;
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        cudaEventElapsedTime(ms, e0, e1);
        return cudaGetLastError();
    };
    float ms = 0;
    int iters = 2000;
    if ((e = run(iters, &ms)) == cudaSuccess && (e = run(iters, &ms)) == cudaSuccess) {
        double want = seconds > 0 ? seconds : 0.25;
        double scale = want * 1e3 / (ms > 1e-3 ? ms : 1e-3);
        long long it2 = (long long)(iters * scale);
        if (it2 < iters) it2 = iters;
        if (it2 > 2000000000ll) it2 = 2000000000ll;
        iters = (int)it2;
        e = run(iters, &ms);
        if (e == cudaSuccess) {
            const double fl = 2.0 * 8.0 * CH * (double)iters * (double)grid * block;
            if (tflops) *tflops = fl / (ms * 1e-3) / 1e12;
            long long clk = 0;
            cudaMemcpy(&clk, dclk, sizeof clk, cudaMemcpyDeviceToHost);
            if (sm_mhz) *sm_mhz = (double)clk / (ms * 1e-3) / 1e6;
            // warp instructions per scheduler = iters*8*CH per warp x 8 warps per scheduler
            if (cycles_per_warp_inst) *cycles_per_warp_inst = (double)clk / ((double)iters * 8.0 * CH * 8.0);
        }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(scratch); cudaFree(dclk);
    return e;
}
