// pn_aux.cu -- staging (AoS <-> SoA), dot-product histogram and FMA-peak kernels of libpn_b200.
#include <cstdint>
#include "pn_internal.h"
#include "pn_dots.cuh"

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
            double d[3];
            bool ok[3];
            pn_unit_dots(v, d, ok);
#pragma unroll
            for (int hh = 0; hh < 3; ++hh) bin[hh] = ok[hh] ? pn_bin_of(d[hh], bins) : -2;      // -2: skipped
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
// Queue ordering by expected cost (default; pn_options.input_order turns it off).  The seed kernel
// writes key[i] (expected number of precession cycles, log-correlation 0.98 with the measured step counts on C3
// and C5) and the range of the keys; issuing the queue longest-first (LPT) shortens the drain tail of the
// persistent grid.  An LPT order only needs to be approximate, so it is a ONE-pass bucket sort on
// PN_ORDER_BUCKETS equal-width buckets of [kmin, kmax], bucket 0 holding the largest keys:
//   count (shared-memory histogram per block, one global add per non-empty bucket) ->
//   exclusive scan of the 2048 counts (one block) ->
//   scatter (rank inside the block from a shared-memory atomic, one global add per block and bucket reserves the
//   block's range, then order[base + rank] = i).
// Systems inside a bucket land in block-arrival order: the ORDER may differ from run to run, the results cannot
// (every system's result is independent of its queue position; tested bit for bit).
// ------------------------------------------------------------------------------------------------
#define PN_ORD_THREADS 256
#define PN_ORD_ITEMS 8       /* systems per thread */
__device__ __forceinline__ int pn_order_bucket(float key, float kmax, float scale)
{
    const int b = (int)((kmax - key) * scale);
    return max(0, min(PN_ORDER_BUCKETS - 1, b));
}
// flat: a batch with many systems per lane (n >= n_flat) whose keys span less than a factor 2 (equal masses: only the spin
// term differs) stays in input order: its
// drain tail is < 0.5 % of the run either way, and neighbouring systems finishing close in time keep the SoA result
// stores and the record reads sector-efficient (C4f: 8.71 -> 8.46 ms, DRAM traffic 3.9 -> 1.2 GB)
__device__ __forceinline__ void pn_order_range(const unsigned* scratch, int n, int n_flat, float& kmax, float& scale)
{
    const unsigned lo = scratch[PN_ORDER_BUCKETS], hi = scratch[PN_ORDER_BUCKETS + 1];
    const float kmin = lo == 0xffffffffu ? 0.0f : __uint_as_float(lo);
    kmax = __uint_as_float(hi);
    scale = kmax > kmin ? (float)(PN_ORDER_BUCKETS - 1) / (kmax - kmin) : 0.0f;     // all keys equal: one bucket
    if (n_flat > 0 && n >= n_flat && kmax < 2.0f * kmin) scale = -1.0f;      // flat: the callers write the identity order
}

__global__ void __launch_bounds__(PN_ORD_THREADS) pn_order_count_kernel(const float* __restrict__ keys, int n, int n_flat, unsigned* __restrict__ scratch)
{
    __shared__ unsigned cnt[PN_ORDER_BUCKETS];
    for (int b = threadIdx.x; b < PN_ORDER_BUCKETS; b += PN_ORD_THREADS) cnt[b] = 0u;
    float kmax, scale;
    pn_order_range(scratch, n, n_flat, kmax, scale);
    if (scale < 0.0f) return;                    // flat (uniform decision): nothing to count
    __syncthreads();
    const int base = blockIdx.x * (PN_ORD_THREADS * PN_ORD_ITEMS);
#pragma unroll
    for (int k = 0; k < PN_ORD_ITEMS; ++k) {
        const int i = base + k * PN_ORD_THREADS + threadIdx.x;
        if (i < n) atomicAdd(&cnt[pn_order_bucket(keys[i], kmax, scale)], 1u);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < PN_ORDER_BUCKETS; b += PN_ORD_THREADS)
        if (cnt[b]) atomicAdd(&scratch[b], cnt[b]);
}

// exclusive scan of the PN_ORDER_BUCKETS counts in place: scratch[b] becomes the first queue position of bucket b
__global__ void __launch_bounds__(1024) pn_order_scan_kernel(unsigned* __restrict__ scratch)
{
    __shared__ unsigned warp_tot[32];
    constexpr int PER = PN_ORDER_BUCKETS / 1024;
    unsigned v[PER], run = 0;
#pragma unroll
    for (int k = 0; k < PER; ++k) { v[k] = scratch[threadIdx.x * PER + k]; run += v[k]; }
    unsigned inc = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, inc, o); if ((threadIdx.x & 31) >= o) inc += t; }
    if ((threadIdx.x & 31) == 31) warp_tot[threadIdx.x >> 5] = inc;
    __syncthreads();
    if (threadIdx.x < 32) {
        unsigned w = warp_tot[threadIdx.x], wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const unsigned t = __shfl_up_sync(0xffffffffu, wi, o); if (threadIdx.x >= o) wi += t; }
        warp_tot[threadIdx.x] = wi - w;
    }
    __syncthreads();
    unsigned start = warp_tot[threadIdx.x >> 5] + inc - run;
#pragma unroll
    for (int k = 0; k < PER; ++k) { scratch[threadIdx.x * PER + k] = start; start += v[k]; }
}

__global__ void __launch_bounds__(PN_ORD_THREADS) pn_order_scatter_kernel(const float* __restrict__ keys, int n, int n_flat, unsigned* __restrict__ scratch,
                                                                          int* __restrict__ order)
{
    __shared__ unsigned cnt[PN_ORDER_BUCKETS];       // systems of this block per bucket, then the block's first position in it
    for (int b = threadIdx.x; b < PN_ORDER_BUCKETS; b += PN_ORD_THREADS) cnt[b] = 0u;
    float kmax, scale;
    pn_order_range(scratch, n, n_flat, kmax, scale);
    const int base = blockIdx.x * (PN_ORD_THREADS * PN_ORD_ITEMS);
    if (scale < 0.0f) {                          // flat: input order
#pragma unroll
        for (int k = 0; k < PN_ORD_ITEMS; ++k) {
            const int i = base + k * PN_ORD_THREADS + threadIdx.x;
            if (i < n) order[i] = i;
        }
        return;
    }
    __syncthreads();
    int bucket[PN_ORD_ITEMS];
    unsigned rank[PN_ORD_ITEMS];
#pragma unroll
    for (int k = 0; k < PN_ORD_ITEMS; ++k) {
        const int i = base + k * PN_ORD_THREADS + threadIdx.x;
        bucket[k] = i < n ? pn_order_bucket(keys[i], kmax, scale) : -1;
        rank[k] = bucket[k] >= 0 ? atomicAdd(&cnt[bucket[k]], 1u) : 0u;
    }
    __syncthreads();
    for (int b = threadIdx.x; b < PN_ORDER_BUCKETS; b += PN_ORD_THREADS)
        if (cnt[b]) cnt[b] = atomicAdd(&scratch[b], cnt[b]);
    __syncthreads();
#pragma unroll
    for (int k = 0; k < PN_ORD_ITEMS; ++k)
        if (bucket[k] >= 0) order[cnt[bucket[k]] + rank[k]] = base + k * PN_ORD_THREADS + threadIdx.x;
}

__global__ void pn_fold_status_kernel(const int* __restrict__ status, int* __restrict__ sticky) { if (*status > *sticky) *sticky = *status; }
cudaError_t pn_launch_fold_status(const int* status, int* sticky, cudaStream_t s)
{
    pn_fold_status_kernel<<<1, 1, 0, s>>>(status, sticky);
    ++g_pn_launches;
    return cudaGetLastError();
}

cudaError_t pn_launch_order_init(unsigned int* scratch, cudaStream_t s)
{
    cudaError_t e;
    if ((e = cudaMemsetAsync(scratch, 0, sizeof(unsigned) * (PN_ORDER_BUCKETS + 2), s)) != cudaSuccess) return e;
    return cudaMemsetAsync(scratch + PN_ORDER_BUCKETS, 0xff, sizeof(unsigned), s);      // running minimum starts at 0xffffffff
}

cudaError_t pn_launch_cost_order(const float* keys, int n, unsigned int* scratch, int* order, cudaStream_t s, int n_flat)
{
    if (n <= 0) return cudaSuccess;
    const int per = PN_ORD_THREADS * PN_ORD_ITEMS, grid = (n + per - 1) / per;
    pn_order_count_kernel<<<grid, PN_ORD_THREADS, 0, s>>>(keys, n, n_flat, scratch);
    pn_order_scan_kernel<<<1, 1024, 0, s>>>(scratch);
    pn_order_scatter_kernel<<<grid, PN_ORD_THREADS, 0, s>>>(keys, n, n_flat, scratch, order);
    g_pn_launches += 3;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// FMA peak and operand-port micro-benchmarks: CHAINS independent dependent-FMA chains per thread, no
// memory traffic.  MODE 0: a = a*U + U (one register source, two uniform operands): the denominator of
// the ALU roofline at the clocks the device actually holds.  MODE 1: a = a*x + U (two
// distinct register sources).  MODE 2: a = a*x + z (three distinct register sources).  On sm_100a a DFMA
// issues every 2 cycles per scheduler with <= 2 register sources and every 3 cycles with 3.
// MODE 3: MODE 1 plus TWO independent integer instructions (LOP3, IADD3) per FMA: do instructions of another pipe issue in
// the shadow of a 2-cycle DFMA?  Mostly not: 3.7 cycles per group, against 2 if hidden and 4 if fully additive.
// Clock: every block measures its own clock64() span and the LONGEST span is kept (atomicMax).  Co-resident
// blocks are not served evenly: the warp arbiter runs the blocks of an SM almost one after the other (measured:
// with 4 resident blocks the first finishes after 1/4 of the kernel's duration, the last spans all of it), so
// the span of one fixed block is not the duration of the kernel -- r1 read block 0's and got 1/4 of the SM clock.
// ------------------------------------------------------------------------------------------------
template <typename real, int CHAINS, int MODE>
__global__ void __launch_bounds__(256) pn_fma_peak_kernel(real* out, int iters, unsigned long long* clocks, real m, real b)
{
    real a[CHAINS], x[CHAINS], z[CHAINS];
    unsigned w[CHAINS];
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) {
        a[i] = (real)(threadIdx.x + i) * (real)1e-3;
        x[i] = (real)1 - (real)1e-7 * (real)(threadIdx.x + i) + out[1];
        z[i] = (real)1e-7 * (real)(i + threadIdx.x) + out[2];
        w[i] = threadIdx.x * 7u + i;
    }
    const long long c0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int i = 0; i < CHAINS; ++i) {
                if (MODE == 0) a[i] = a[i] * m + b;
                if (MODE == 1 || MODE == 3) a[i] = a[i] * x[i] + b;
                if (MODE == 2) a[i] = a[i] * x[i] + z[i];
                if (MODE == 3) w[i] = (w[i] ^ (unsigned)it) + (unsigned)i + 1u;      // one LOP3 + one IADD3
            }
    }
    const long long c1 = clock64();
    real s = 0;
#pragma unroll
    for (int i = 0; i < CHAINS; ++i) s += a[i] + (MODE == 3 ? (real)w[i] : (real)0);
    if (s == (real)123.456) out[0] = s;
    if (threadIdx.x == 0) atomicMax(clocks, (unsigned long long)(c1 - c0));
}

// packed FP32: a = a * m + b on register pairs (FFMA2), 8 chains per thread; 4 flops per instruction and lane
__global__ void __launch_bounds__(256) pn_ffma2_peak_kernel(float* out, int iters, unsigned long long* clocks, float m, float b)
{
    float2 a[8];
    const float2 mm = make_float2(m, m), bb = make_float2(b, b);
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = make_float2((threadIdx.x + i) * 1e-3f, (threadIdx.x + i) * 2e-3f);
    const long long c0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = __ffma2_rn(a[i], mm, bb);
    }
    const long long c1 = clock64();
    float s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i].x + a[i].y;
    if (s == 123.456f) out[0] = s;
    if (threadIdx.x == 0) atomicMax(clocks, (unsigned long long)(c1 - c0));
}

// precision 0 / 1: FP64 / FP32 scalar FMA; 3: FP32 packed (FFMA2, mode ignored)
cudaError_t pn_run_fma_peak(int precision, int mode, double seconds, double* tflops, double* sm_mhz,
                            double* cycles_per_warp_inst)
{
    const int CH = 8;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    void* scratch = nullptr;
    unsigned long long* dclk = nullptr;
    cudaError_t e;
    if ((e = cudaMalloc(&scratch, 64)) != cudaSuccess) return e;
    if ((e = cudaMemset(scratch, 0, 64)) != cudaSuccess) { cudaFree(scratch); return e; }
    if ((e = cudaMalloc((void**)&dclk, sizeof(unsigned long long))) != cudaSuccess) { cudaFree(scratch); return e; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    // 4 resident blocks of 8 warps per SM = 8 warps per scheduler, one wave; checked against the occupancy the
    // runtime reports for this instantiation (fewer resident blocks -> a smaller grid, still one wave)
    const int block = 256;
    int occ = 0;
#define PN_PEAK_OCC(T, M) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pn_fma_peak_kernel<T, CH, M>, block, 0)
    if (precision == 3) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pn_ffma2_peak_kernel, block, 0);
    else if (precision == 0) { if (mode == 0) PN_PEAK_OCC(double, 0); else if (mode == 1) PN_PEAK_OCC(double, 1); else if (mode == 2) PN_PEAK_OCC(double, 2); else PN_PEAK_OCC(double, 3); }
    else { if (mode == 0) PN_PEAK_OCC(float, 0); else if (mode == 1) PN_PEAK_OCC(float, 1); else if (mode == 2) PN_PEAK_OCC(float, 2); else PN_PEAK_OCC(float, 3); }
#undef PN_PEAK_OCC
    const int resident = occ >= 4 ? 4 : (occ >= 1 ? occ : 1);
    const int grid = sms * resident;
    const double warps_per_scheduler = resident * (block / 32) / 4.0;
    auto run = [&](int iters, float* ms) {
        cudaMemsetAsync(dclk, 0, sizeof(unsigned long long));
        cudaEventRecord(e0);
#define PN_PEAK(T, M) pn_fma_peak_kernel<T, CH, M><<<grid, block>>>((T*)scratch, iters, dclk, (T)0.999999, (T)1e-7)
        if (precision == 3) pn_ffma2_peak_kernel<<<grid, block>>>((float*)scratch, iters, dclk, 0.999999f, 1e-7f);
        else if (precision == 0) { if (mode == 0) PN_PEAK(double, 0); else if (mode == 1) PN_PEAK(double, 1); else if (mode == 2) PN_PEAK(double, 2); else PN_PEAK(double, 3); }
        else { if (mode == 0) PN_PEAK(float, 0); else if (mode == 1) PN_PEAK(float, 1); else if (mode == 2) PN_PEAK(float, 2); else PN_PEAK(float, 3); }
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
            const double fl = (precision == 3 ? 4.0 : 2.0) * 8.0 * CH * (double)iters * (double)grid * block;
            if (tflops) *tflops = fl / (ms * 1e-3) / 1e12;
            unsigned long long clk = 0;
            cudaMemcpy(&clk, dclk, sizeof clk, cudaMemcpyDeviceToHost);
            if (sm_mhz) *sm_mhz = (double)clk / (ms * 1e-3) / 1e6;
            // warp instructions per scheduler = iters*8*CH per warp x resident warps per scheduler
            if (cycles_per_warp_inst) *cycles_per_warp_inst = (double)clk / ((double)iters * 8.0 * CH * warps_per_scheduler);
        }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(scratch); cudaFree(dclk);
    return e;
}
