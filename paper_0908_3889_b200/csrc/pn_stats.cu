// pn_stats.cu -- one-pass ensemble statistics of (initial, final) states for sm_100a:
// Pearson r of the initial vs final unit dot products, their bivariate histograms
// and the 1-D histograms of the final ones, per ensemble ("group":
// a contiguous range of group_size systems, so a parameter sweep -- Figs. 6, 7 -- is one launch).
//
// HBM-bound: 160 B per system (two AoS rows) + 4 B (steps).  One persistent block (two consumer groups of 256
// threads) per SM streams tiles of
// 256 systems (2 x 20 KB, contiguous in the AoS arrays) through one shared-memory slot per group, filled by
// cp.async.bulk (TMA 1-D bulk copies, one elected thread, completion on an mbarrier), so up to 80 KB per SM
// are in flight.  Per-thread shifted sums -> (n, mean, M2, C) -> Chan's pairwise merge over the
// warp (xor butterfly), the block (shared memory) and the grid (one record per (block, group), merged in
// block order by the finish kernel): no floating-point atomics, results are bit-identical run to run.
// Histograms are privatised in shared memory (3 x bins1 + 3 x bins2^2 u32) and flushed with 64-bit global
// atomics when the block leaves a group.
// This file shares nothing with oracle/ (which evaluates the two-pass definitions in numpy).
#include <cstdint>
#include "../../include/pn.h"
#include "pn_internal.h"
#include "pn_dots.cuh"
#include "pn_moments.cuh"

#define ST_TILE 256
#define ST_STAGES 2      /* one ring slot per consumer group (see pn_stats_kernel) */
#define ST_ROW 10
#define ST_TILE_BYTES (ST_TILE * ST_ROW * 8)

// ---- mbarrier / bulk-copy PTX ---------------------------------------------------------------------------
__device__ __forceinline__ uint32_t st_smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void st_mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void st_mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void st_bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void st_mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    do {
        asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok)
                     : "r"(bar), "r"(parity)
                     : "memory");
    } while (!ok);
}

// per-thread running sums of (x - x0), (y - y0) about the thread's first sample of the group
struct StAcc {
    int n;
    double x0, y0, sx, sy, sxx, syy, sxy;
    __device__ __forceinline__ void reset() { n = 0; x0 = y0 = sx = sy = sxx = syy = sxy = 0.0; }
    __device__ __forceinline__ void add(double x, double y)
    {
        if (n == 0) { x0 = x; y0 = y; }
        const double dx = x - x0, dy = y - y0;
        ++n;
        sx += dx; sy += dy;
        sxx = fma(dx, dx, sxx); syy = fma(dy, dy, syy); sxy = fma(dx, dy, sxy);
    }
    __device__ __forceinline__ StMom moments() const
    {
        StMom m;
        m.n = (double)n;
        if (n == 0) { m.mx = m.my = m.m2x = m.m2y = m.cxy = 0.0; return m; }
        const double inv = 1.0 / m.n;
        m.mx = x0 + sx * inv; m.my = y0 + sy * inv;
        m.m2x = fmax(sxx - sx * sx * inv, 0.0);
        m.m2y = fmax(syy - sy * sy * inv, 0.0);
        m.cxy = sxy - sx * sy * inv;
        return m;
    }
};

// unit dot products of one AoS row (the shared routine of pn_dots.cuh); ok[k] false where undefined (R14)
__device__ __forceinline__ void st_unit_dots(const double* __restrict__ row, double (&d)[3], bool (&ok)[3])
{
    const double v[9] = {row[1], row[2], row[3], row[4], row[5], row[6], row[7], row[8], row[9]};
    pn_unit_dots(v, d, ok);
}
__device__ __forceinline__ int st_bin(double d, int bins) { return pn_bin_of(d, bins); }

struct StParams {
    const double* init;     // [N][10] or null (final-only mode: 1-D histograms and skipped counts only)
    const double* fin;      // [N][10]
    const int* steps;       // [N] or null
    long long n, group_size;
    int n_groups, tiles_per_group, items_per_block;
    long long n_items;
    int bins1, bins2, hist2_smem;
    double* records;                 // [(blocks + groups)][3][6]
    unsigned long long* rec_skipped; // [(blocks + groups)][3]
    unsigned long long* hist1;       // [G][3][bins1] or null
    unsigned long long* hist2;       // [G][3][bins2][bins2] or null
};

// ST_GROUPS consumer groups of ST_TILE threads, each with its own shared-memory slot and mbarrier: item k of the
// block (k = 0, 1, ...) is consumed by group k % ST_GROUPS.  A group copies its rows to registers, syncs on its own
// named barrier and its first thread immediately re-arms the slot for the group's next item, so each group's next
// tile (40 KB) is in flight while it does its FP64 work, and the groups run out of phase with one another
// (16 warps per SM hide the rsqrt / atomic latencies that 8 lock-stepped warps could not).  A slot is never
// shared between groups: a consumer that ran ahead of the re-arming group would see the PREVIOUS phase of the
// mbarrier as complete and read a stale tile.
#define ST_GROUPS 2
#define ST_THREADS (ST_GROUPS * ST_TILE)
template <bool HAVE_INIT>
__global__ void __launch_bounds__(ST_THREADS, 1) pn_stats_kernel(const StParams p)
{
    extern __shared__ __align__(128) unsigned char st_smem[];
    // layout: [stages][2 tiles] | mbarriers | warp scratch | hist1 | hist2
    constexpr int NT = HAVE_INIT ? 2 : 1;
    constexpr int NW = ST_THREADS / 32;
    double* tiles = reinterpret_cast<double*>(st_smem);
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(st_smem + (size_t)ST_STAGES * NT * ST_TILE_BYTES);
    double* wscr = reinterpret_cast<double*>(bars + 8);                        // [NW warps][3][6]
    unsigned* skip_s = reinterpret_cast<unsigned*>(wscr + NW * 18);            // [4]
    unsigned* hist1 = skip_s + 4;
    unsigned* hist2 = hist1 + 3 * p.bins1;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int grp = tid / ST_TILE, row = tid - grp * ST_TILE;
    const int nh1 = 3 * p.bins1, nh2 = p.hist2_smem ? 3 * p.bins2 * p.bins2 : 0;

    // item indices fit an int: n_items = N/256 < 2^31 for any N the ABI accepts
    const int w_begin = blockIdx.x * p.items_per_block;
    const int w_end = (int)min((long long)w_begin + p.items_per_block, p.n_items);
    if (w_begin >= w_end) return;

    for (int b = tid; b < nh1 + nh2; b += ST_THREADS) hist1[b] = 0u;
    if (tid < 4) skip_s[tid] = 0u;
    if (tid == 0) {
        for (int s = 0; s < ST_STAGES; ++s) st_mbar_init(st_smem_addr(&bars[s]), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    auto item_range = [&](int w, long long& start, int& cnt) {
        const int g = w / p.tiles_per_group;
        const long long t = w - g * p.tiles_per_group;
        start = (long long)g * p.group_size + t * ST_TILE;
        cnt = (int)min((long long)ST_TILE, p.group_size - t * ST_TILE);
    };
    auto issue = [&](int w, int stage) {       // one elected thread
        long long start; int cnt;
        item_range(w, start, cnt);
        const uint32_t bar = st_smem_addr(&bars[stage]);
        const uint32_t bytes = (uint32_t)cnt * ST_ROW * 8u;
        st_mbar_expect_tx(bar, bytes * NT);
        double* dst = tiles + (size_t)stage * NT * ST_TILE * ST_ROW;
        st_bulk_g2s(st_smem_addr(dst), p.fin + start * ST_ROW, bytes, bar);
        if (HAVE_INIT) st_bulk_g2s(st_smem_addr(dst + ST_TILE * ST_ROW), p.init + start * ST_ROW, bytes, bar);
    };
    if (tid == 0)
        for (int s = 0; s < ST_STAGES && w_begin + s < w_end; ++s) issue(w_begin + s, s);

    StAcc acc[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) acc[k].reset();

    int w = w_begin + grp;                    // this consumer group's next item
    const int g_first = w_begin / p.tiles_per_group, g_last = (w_end - 1) / p.tiles_per_group;
    for (int g = g_first; g <= g_last; ++g) {
        const int w_g_end = (int)min((long long)w_end, (long long)(g + 1) * p.tiles_per_group);
        for (; w < w_g_end; w += ST_GROUPS) {
            const int stage = grp;                                            // each group owns one slot
            const uint32_t parity = (uint32_t)(((w - w_begin) / ST_GROUPS) & 1);
            long long start; int cnt;
            item_range(w, start, cnt);
            st_mbar_wait(st_smem_addr(&bars[stage]), parity);
            // final-state rows first: their dot products are formed before the initial-state rows are read, so the
            // two 10-double rows are never live together (the kernel must fit 128 registers at 512 threads)
            double df[3], di[3];
            bool okf[3] = {false, false, false}, oki[3] = {true, true, true};
            const bool have = row < cnt;
            if (have) {
                // 16-byte shared loads: rows are 80 B apart, so a quarter-warp covers 8 distinct 16-byte bank groups
                const double2* src = reinterpret_cast<const double2*>(tiles + (size_t)stage * NT * ST_TILE * ST_ROW + row * ST_ROW);
                double rw[ST_ROW];
#pragma unroll
                for (int c = 0; c < ST_ROW / 2; ++c) { const double2 v = src[c]; rw[2 * c] = v.x; rw[2 * c + 1] = v.y; }
                st_unit_dots(rw, df, okf);
                if (HAVE_INIT) {
#pragma unroll
                    for (int c = 0; c < ST_ROW / 2; ++c) { const double2 v = src[ST_TILE * ST_ROW / 2 + c]; rw[2 * c] = v.x; rw[2 * c + 1] = v.y; }
                    st_unit_dots(rw, di, oki);
                }
            }
            const bool failed = have && p.steps && (p.steps[start + row] < 0);
            // only six doubles per thread are live across the barrier (the kernel must fit 128 registers at 512 threads)
            asm volatile("bar.sync %0, %1;" ::"r"(1 + grp), "r"(ST_TILE) : "memory");     // this group has read the slot
            if (row == 0 && w + ST_STAGES < w_end) issue(w + ST_STAGES, stage);

            if (have) {
#pragma unroll
                for (int kk = 0; kk < 3; ++kk) {
                    const bool ok = okf[kk] && oki[kk] && !failed;
                    if (!ok) { atomicAdd(&skip_s[kk], 1u); continue; }      // rare: straight to the block counter
                    if (HAVE_INIT) acc[kk].add(di[kk], df[kk]);
                    if (p.bins1) atomicAdd(&hist1[kk * p.bins1 + st_bin(df[kk], p.bins1)], 1u);
                    if (HAVE_INIT && p.bins2) {
                        const size_t cell = ((size_t)kk * p.bins2 + st_bin(di[kk], p.bins2)) * p.bins2 + st_bin(df[kk], p.bins2);
                        if (p.hist2_smem) atomicAdd(&hist2[cell], 1u);
                        else atomicAdd(&p.hist2[(size_t)g * 3 * p.bins2 * p.bins2 + cell], 1ull);
                    }
                }
            }
        }

        // ---- the block leaves ensemble g: merge (warp butterfly, then warps in order) and flush ----
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            StMom m = acc[k].moments();
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { StMom other = st_shfl_xor(m, o); st_merge(m, other); }
            // the butterfly leaves every lane with a (not bitwise identical) total; lane 0's is the result
            if (lane == 0) {
                double* q = wscr + (warp * 3 + k) * 6;
                q[0] = m.n; q[1] = m.mx; q[2] = m.my; q[3] = m.m2x; q[4] = m.m2y; q[5] = m.cxy;
            }
            acc[k].reset();
        }
        __syncthreads();
        const size_t slot = (size_t)blockIdx.x + (size_t)g;        // unique per (block, ensemble): both only grow
        if (tid < 3) {
            StMom m = {0, 0, 0, 0, 0, 0};
            for (int ww = 0; ww < NW; ++ww) {
                const double* q = wscr + (ww * 3 + tid) * 6;
                StMom o = {q[0], q[1], q[2], q[3], q[4], q[5]};
                st_merge(m, o);
            }
            double* r = p.records + (slot * 3 + tid) * 6;
            r[0] = m.n; r[1] = m.mx; r[2] = m.my; r[3] = m.m2x; r[4] = m.m2y; r[5] = m.cxy;
            p.rec_skipped[slot * 3 + tid] = skip_s[tid];
        }
        if (p.hist1)
            for (int b = tid; b < nh1; b += ST_THREADS)
                if (hist1[b]) { atomicAdd(&p.hist1[(size_t)g * nh1 + b], (unsigned long long)hist1[b]); hist1[b] = 0u; }
        if (nh2)
            for (int b = tid; b < nh2; b += ST_THREADS)
                if (hist2[b]) { atomicAdd(&p.hist2[(size_t)g * nh2 + b], (unsigned long long)hist2[b]); hist2[b] = 0u; }
        __syncthreads();
        if (tid < 4) skip_s[tid] = 0u;
        __syncthreads();
    }
}

// One warp per (ensemble, dot product): the per-block records of that ensemble are merged lane-strided in block
// order, then over the lanes with the same xor butterfly as in the main kernel (fixed order: deterministic).
__global__ void __launch_bounds__(128) pn_stats_finish_kernel(const StParams p, int n_blocks, double* __restrict__ r_out,
                                                              double* __restrict__ mom_out, unsigned long long* __restrict__ skipped_out)
{
    const int j = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (j >= p.n_groups * 3) return;
    const int g = j / 3, k = j % 3;
    const long long w_lo = (long long)g * p.tiles_per_group, w_hi = w_lo + p.tiles_per_group - 1;
    const int b_lo = (int)(w_lo / p.items_per_block), b_hi = min((int)(w_hi / p.items_per_block), n_blocks - 1);
    StMom m = {0, 0, 0, 0, 0, 0};
    unsigned long long sk = 0;
    for (int b = b_lo + lane; b <= b_hi; b += 32) {
        const size_t slot = (size_t)b + (size_t)g;
        const double* q = p.records + (slot * 3 + k) * 6;
        StMom o = {q[0], q[1], q[2], q[3], q[4], q[5]};
        st_merge(m, o);
        sk += p.rec_skipped[slot * 3 + k];
    }
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        StMom other = st_shfl_xor(m, o);
        st_merge(m, other);
        sk += __shfl_xor_sync(0xffffffffu, sk, o);
    }
    if (lane != 0) return;
    if (mom_out) {
        double* q = mom_out + (size_t)j * 6;
        q[0] = m.n; q[1] = m.n > 0 ? m.mx : nan(""); q[2] = m.n > 0 ? m.my : nan(""); q[3] = m.m2x; q[4] = m.m2y; q[5] = m.cxy;
    }
    // PAPER.md:138 with sample standard deviations (R18): r = Cxy / sqrt(M2x M2y); undefined for n < 2 or zero variance
    if (r_out) r_out[j] = (m.n >= 2.0 && m.m2x > 0.0 && m.m2y > 0.0) ? m.cxy / sqrt(m.m2x * m.m2y) : nan("");
    if (skipped_out) skipped_out[j] = sk;
}

// One block per (group, dot product): maximum count of the bivariate histogram and counts / max.
__global__ void __launch_bounds__(256) pn_stats_norm_kernel(const unsigned long long* __restrict__ hist2, int cells,
                                                            unsigned long long* __restrict__ max_out, double* __restrict__ norm_out)
{
    __shared__ unsigned long long red[256];
    const unsigned long long* h = hist2 + (size_t)blockIdx.x * cells;
    unsigned long long mx = 0;
    for (int c = threadIdx.x; c < cells; c += 256) mx = max(mx, h[c]);
    red[threadIdx.x] = mx;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] = max(red[threadIdx.x], red[threadIdx.x + o]);
        __syncthreads();
    }
    mx = red[0];
    if (threadIdx.x == 0 && max_out) max_out[blockIdx.x] = mx;
    if (norm_out) {
        for (int c = threadIdx.x; c < cells; c += 256)
            norm_out[(size_t)blockIdx.x * cells + c] = mx ? (double)h[c] / (double)mx : 0.0;    // correctly rounded quotient
    }
}

cudaError_t pn_launch_stats_norm(const unsigned long long* hist2, long long n_hists, int cells, unsigned long long* max_out,
                                 double* norm_out, cudaStream_t s)
{
    if (n_hists <= 0) return cudaSuccess;
    pn_stats_norm_kernel<<<(unsigned)n_hists, 256, 0, s>>>(hist2, cells, max_out, norm_out);
    ++g_pn_launches;
    return cudaGetLastError();
}

// Multi-GPU exchange step of the statistics: the moment records of R parts of the same ensembles
// (one part per rank, gathered with one all-gather of R x G x 3 x 6 doubles) are merged in part order with the same
// pairwise update as inside a launch.  One thread per (group, dot product).
__global__ void pn_stats_merge_kernel(const double* __restrict__ parts, int n_parts, int n_groups,
                                      double* __restrict__ mom_out, double* __restrict__ r_out)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_groups * 3) return;
    StMom m = {0, 0, 0, 0, 0, 0};
    for (int part = 0; part < n_parts; ++part) {
        const double* q = parts + ((size_t)part * n_groups * 3 + j) * 6;
        StMom o = {q[0], q[0] > 0 ? q[1] : 0.0, q[0] > 0 ? q[2] : 0.0, q[3], q[4], q[5]};      // empty parts carry NaN means
        st_merge(m, o);
    }
    if (mom_out) {
        double* q = mom_out + (size_t)j * 6;
        q[0] = m.n; q[1] = m.n > 0 ? m.mx : nan(""); q[2] = m.n > 0 ? m.my : nan(""); q[3] = m.m2x; q[4] = m.m2y; q[5] = m.cxy;
    }
    if (r_out) r_out[j] = (m.n >= 2.0 && m.m2x > 0.0 && m.m2y > 0.0) ? m.cxy / sqrt(m.m2x * m.m2y) : nan("");
}

cudaError_t pn_launch_stats_merge(const double* parts, int n_parts, int n_groups, double* mom_out, double* r_out, cudaStream_t s)
{
    if (n_groups <= 0) return cudaSuccess;
    pn_stats_merge_kernel<<<(n_groups * 3 + 127) / 128, 128, 0, s>>>(parts, n_parts, n_groups, mom_out, r_out);
    ++g_pn_launches;
    return cudaGetLastError();
}

size_t pn_stats_scratch_bytes(long long n, long long group_size, int* n_blocks_out)
{
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long long gs = group_size > 0 ? group_size : n;
    const long long G = gs > 0 ? n / gs : 0;
    const long long tpg = (gs + ST_TILE - 1) / ST_TILE;
    const long long items = G * tpg;
    const long long blocks = items < sms ? items : sms;
    if (n_blocks_out) *n_blocks_out = (int)blocks;
    return (size_t)(blocks + G + 1) * 3 * (6 * sizeof(double) + sizeof(unsigned long long));
}

cudaError_t pn_launch_stats(const double* init, const double* fin, const int* steps, long long n, long long group_size,
                            int bins1, int bins2, void* scratch, double* r_out, double* mom_out,
                            unsigned long long* skipped_out, unsigned long long* hist1, unsigned long long* hist2,
                            unsigned long long* hist2_max, double* hist2_norm, cudaStream_t s)
{
    const long long gs = group_size > 0 ? group_size : n;
    const long long G = gs > 0 ? n / gs : 0;
    cudaError_t e;
    if (hist1 && (e = cudaMemsetAsync(hist1, 0, sizeof(unsigned long long) * 3 * (size_t)bins1 * G, s)) != cudaSuccess) return e;
    if (hist2 && (e = cudaMemsetAsync(hist2, 0, sizeof(unsigned long long) * 3 * (size_t)bins2 * bins2 * G, s)) != cudaSuccess) return e;
    if (n <= 0 || G <= 0) return cudaSuccess;
    int n_blocks = 0;
    const size_t scr = pn_stats_scratch_bytes(n, group_size, &n_blocks);
    if ((e = cudaMemsetAsync(scratch, 0, scr, s)) != cudaSuccess) return e;
    StParams p;
    p.init = init; p.fin = fin; p.steps = steps; p.n = n; p.group_size = gs; p.n_groups = (int)G;
    p.tiles_per_group = (int)((gs + ST_TILE - 1) / ST_TILE);
    p.n_items = G * p.tiles_per_group;
    if (p.n_items > 0x7fffffffLL) return cudaErrorInvalidValue;
    p.items_per_block = (int)((p.n_items + n_blocks - 1) / n_blocks);
    n_blocks = (int)((p.n_items + p.items_per_block - 1) / p.items_per_block);
    p.bins1 = hist1 ? bins1 : 0;
    p.bins2 = (hist2 && init) ? bins2 : 0;
    p.records = (double*)scratch;
    p.rec_skipped = (unsigned long long*)((char*)scratch + (size_t)(n_blocks + G + 1) * 3 * 6 * sizeof(double));
    p.hist1 = hist1; p.hist2 = hist2;
    const int nt = init ? 2 : 1;
    const size_t fixed = (size_t)ST_STAGES * nt * ST_TILE_BYTES + 64 + (ST_THREADS / 32) * 18 * sizeof(double) + 16 + 3 * (size_t)p.bins1 * 4;
    const size_t h2 = 3 * (size_t)p.bins2 * p.bins2 * 4;
    const size_t cap = 220 * 1024;
    if (fixed > cap) return cudaErrorInvalidValue;
    p.hist2_smem = (p.bins2 > 0 && fixed + h2 <= cap) ? 1 : 0;
    const size_t shm = fixed + (p.hist2_smem ? h2 : 0);
    // opt in to large dynamic shared memory once per process (a host-side call per launch leaves the GPU idle)
    static bool attr_done_dev[64] = {false};          // the attribute is per device
    int dev_id = 0;
    if ((e = cudaGetDevice(&dev_id)) != cudaSuccess) return e;
    bool& attr_done = attr_done_dev[dev_id & 63];
    if (!attr_done) {
        if ((e = cudaFuncSetAttribute(pn_stats_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cap)) != cudaSuccess) return e;
        if ((e = cudaFuncSetAttribute(pn_stats_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cap)) != cudaSuccess) return e;
        attr_done = true;
    }
    if (init) pn_stats_kernel<true><<<n_blocks, ST_THREADS, shm, s>>>(p);
    else pn_stats_kernel<false><<<n_blocks, ST_THREADS, shm, s>>>(p);
    ++g_pn_launches;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    pn_stats_finish_kernel<<<(int)((G * 3 + 3) / 4), 128, 0, s>>>(p, n_blocks, r_out, mom_out, skipped_out);
    ++g_pn_launches;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if (p.bins2 && (hist2_max || hist2_norm)) {
        pn_stats_norm_kernel<<<(int)(G * 3), 256, 0, s>>>(hist2, bins2 * bins2, hist2_max, hist2_norm);
        ++g_pn_launches;
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

// ---- pn_statistics_static: the statistics pass without any allocation (include/pn.h) ---------------------------------
// For embedders that cannot call cudaMalloc when they want the statistics: the whole HBM already belongs to their
// framework's caching allocator (a library cudaMalloc then fails with out-of-memory), or other streams are running and
// must not be stalled by the device-wide synchronisation that cudaMalloc / cudaFree imply, or the process has a fixed
// memory budget.  The per-(block, ensemble) moment records and skipped counters that pn_launch_stats needs live in this
// array instead of a cudaMalloc'ed buffer.  It is part of the module image: each GPU that loads the library holds these
// 336 KB until the process exits.  One array per device serves every call, so it always holds what the last call left:
// pn_launch_stats zeroes the part it is about to use on the stream, ahead of the kernels, and calls that may overlap on
// the GPU (unordered streams) race on it; see the header.
static __device__ __align__(256) unsigned char pn_static_scratch[PN_STATIC_SCRATCH_BYTES];

// Device address of the array, per device.  In host code the identifier pn_static_scratch is only the handle the runtime
// uses to find the symbol: handing it to a kernel would make the kernel dereference a host address.  The real address
// differs from device to device, so it is looked up once per device with that device current.
#define PN_STATIC_MAX_DEVICES 64
static void* g_static_addr[PN_STATIC_MAX_DEVICES] = {nullptr};

extern "C" int pn_statistics_static(const double* init_states, const double* final_states, const int* steps, long long N,
                                    long long group_size, int bins1, int bins2, const pn_stats_out* out_in, void* stream, int async)
{
    // the argument rules of pn_statistics for device buffers
    if (!out_in || out_in->size != (int)sizeof(pn_stats_out)) return PN_EINVAL;
    pn_stats_out out = *out_in;
    if (N < 0 || N > 0x7fffffffLL * 8) return PN_EINVAL;
    if (N > 0 && !final_states) return PN_EINVAL;
    if (bins1 > 8192 || bins2 > 4096) return PN_EINVAL;
    if (bins1 < 1) { bins1 = 0; out.hist1 = nullptr; }
    if (bins2 < 1 || !init_states) { bins2 = 0; out.hist2 = nullptr; }
    if (!out.hist2 && (out.hist2_max || out.hist2_norm)) return PN_EINVAL;
    const long long gs = group_size > 0 ? group_size : N;
    if (N > 0 && N % gs != 0) return PN_EINVAL;
    if (N == 0) return PN_OK;
    if (((uintptr_t)final_states & 15u) || ((uintptr_t)init_states & 15u)) return PN_EINVAL;
    // capacity: refuse, with its own status, before anything is enqueued
    if (N / gs > PN_STATIC_MAX_GROUPS) return PN_ETOOLARGE;
    if (pn_stats_scratch_bytes(N, group_size, nullptr) > (size_t)PN_STATIC_SCRATCH_BYTES) return PN_ETOOLARGE;

    // set-up, first call on this device: where the array lives in this device's memory
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { pn_note_cuda_error("pn_statistics_static: cudaGetDevice", e); return PN_ECUDA; }
    if (dev < 0 || dev >= PN_STATIC_MAX_DEVICES) return PN_EINVAL;
    if (!g_static_addr[dev]) {
        void* addr = nullptr;
        e = cudaGetSymbolAddress((void**)&addr, pn_static_scratch);
        if (e != cudaSuccess || !addr) {
            pn_note_cuda_error("pn_statistics_static: cudaGetSymbolAddress(pn_static_scratch)", e);
            return PN_ECUDA;
        }
        g_static_addr[dev] = addr;
    }
    cudaStream_t s = (cudaStream_t)stream;
    // the unchanged launcher of pn_statistics (memset of the records it uses, main kernel, finish kernel, optional
    // normalisation), pointed at the static array: no allocation anywhere below
    e = pn_launch_stats(init_states, final_states, steps, N, group_size, bins1, bins2, g_static_addr[dev], out.pearson_r,
                        out.moments, out.n_skipped, out.hist1, out.hist2, out.hist2_max, out.hist2_norm, s);
    if (e != cudaSuccess) { pn_note_cuda_error("pn_statistics_static: launch", e); return PN_ECUDA; }
    if (async) return PN_OK;
    e = cudaStreamSynchronize(s);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) { pn_note_cuda_error("pn_statistics_static: synchronize", e); return PN_ECUDA; }
    return PN_OK;
}
