// pn_api.cu -- the C ABI of libpn_b200 (include/pn.h): argument checks, scratch management, staging,
// launches, status collection.  Every CUDA call is checked.
#include <cstdint>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <string>
#include <vector>
#include "../../include/pn.h"
#include "pn_internal.h"

#define PN_VERSION 100

static std::string g_last_err;
#define CK(call)                                                                                     \
    do {                                                                                             \
        cudaError_t _e = (call);                                                                     \
        if (_e != cudaSuccess) {                                                                     \
            char _b[512];                                                                            \
            snprintf(_b, sizeof _b, "%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(_e)); \
            g_last_err = _b;                                                                         \
            return PN_ECUDA;                                                                         \
        }                                                                                            \
    } while (0)

void pn_note_cuda_error(const char* where, cudaError_t e)
{
    g_last_err = std::string(where) + " -> " + cudaGetErrorString(e);
}

// ---- cached device scratch ------------------------------------------------------------------------
struct Buf {
    void* p = nullptr;
    size_t cap = 0;
    int ensure(size_t bytes)
    {
        if (bytes <= cap) return PN_OK;
        if (p) { CK(cudaFree(p)); p = nullptr; cap = 0; }
        CK(cudaMalloc(&p, bytes));
        cap = bytes;
        return PN_OK;
    }
    int release()
    {
        if (p) { cudaError_t e = cudaFree(p); p = nullptr; cap = 0; if (e != cudaSuccess) return PN_ECUDA; }
        return PN_OK;
    }
};
// One scratch context per stream: two calls in flight on different streams never share a buffer, a work counter or
// a status word (the single global set was aliased by concurrent async calls).  Calls on ONE stream are
// ordered by the stream, so they may share their context's buffers; what they must not share is the status word:
// every call owns the status in its (re-zeroed) Small block and async calls fold it into the context's sticky word
// with a one-thread kernel at the end, which only pn_stream_status reads and clears.
struct Ctx {
    Buf soa_in, soa_m, soa_out, small, sticky, redo, seed, keys, order, ord_scr, h_init, h_m, h_final, h_steps, h_time, h_rej,
        h_counts, st_scratch, st_in, st_out, gen_specs, gen_y, gen_m, ck_idx, ck_tmp, ck_sub, ck_out, ck_in, fu_scr;
    cudaEvent_t ev[5];
    bool ev_ok = false;
    bool async_pending = false;
    int slot = -1;              // row of the __constant__ table of the uniform-mass kernel; -1: none left (generic kernel only)
    Buf* all[29] = {&soa_in, &soa_m, &soa_out, &small, &sticky, &redo, &seed, &keys, &order, &ord_scr, &h_init, &h_m, &h_final,
                    &h_steps, &h_time, &h_rej, &h_counts, &st_scratch, &st_in, &st_out, &gen_specs, &gen_y, &gen_m, &ck_idx,
                    &ck_tmp, &ck_sub, &ck_out, &ck_in, &fu_scr};
};
// Contexts are keyed by (device, stream): the NULL stream (and any handle value) of two devices are different streams, and
// the buffers, events and the __constant__ table row of a context belong to the device it was created on.
typedef std::pair<int, void*> CtxKey;
static std::map<CtxKey, Ctx*> g_ctx;
#define PN_MAX_DEVICES 64
static bool g_slot_used[PN_MAX_DEVICES][PN_UNI_SLOTS];     // rows of each device's uniform-mass table in use by a context
static float g_ms[4] = {0, 0, 0, 0};
static unsigned long long g_counters[4] = {0, 0, 0, 0};
static unsigned g_redo_count = 0;   // systems that went through the redo pass in the last synchronous call

static int current_device()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); dev = 0; }
    return dev;
}

static Ctx* ctx_for(void* stream)
{
    const int dev = current_device();
    auto it = g_ctx.find(CtxKey(dev, stream));
    if (it != g_ctx.end()) return it->second;
    Ctx* c = new Ctx();
    // a row of this device's table, if one is free (pn_stream_release returns rows); none left: the generic kernel only
    if (dev >= 0 && dev < PN_MAX_DEVICES)
        for (int k = 0; k < PN_UNI_SLOTS && c->slot < 0; ++k)
            if (!g_slot_used[dev][k]) { g_slot_used[dev][k] = true; c->slot = k; }
    g_ctx[CtxKey(dev, stream)] = c;
    return c;
}

static int free_ctx(Ctx* c)
{
    int rc = PN_OK;
    for (Buf* b : c->all) if (b->release() != PN_OK) rc = PN_ECUDA;
    if (c->ev_ok) for (int i = 0; i < 5; ++i) cudaEventDestroy(c->ev[i]);
    delete c;
    return rc;
}

// layout of g_small: [0..3] counters (u64), then queue (u32), status (i32)
struct Small { unsigned long long counters[4]; unsigned int queue; int status; unsigned int queue2; unsigned int redo_count; unsigned long long skipped[3]; int nonuniform; int pad; double uni_row[PN_UNI_ROW]; };

static int ensure_events(Ctx& c)
{
    if (!c.ev_ok) {
        for (int i = 0; i < 5; ++i) CK(cudaEventCreate(&c.ev[i]));
        c.ev_ok = true;
    }
    return PN_OK;
}

static void default_options(pn_options* o)
{
    memset(o, 0, sizeof *o);
    o->size = (int)sizeof *o;
}

extern "C" int pn_integrate_ex(const double* init_states, const double* masses, long long N, double omega0,
                               double omegaf, double rtol, double atol, int precision, double* out_final,
                               int* out_steps, const pn_options* opt_in)
{
    pn_options o;
    default_options(&o);
    if (opt_in) {
        if (opt_in->size != (int)sizeof(pn_options)) return PN_EINVAL;
        o = *opt_in;
    }
    if (N < 0 || N > 0x7fffffffLL / 16) return PN_EINVAL;
    if (o.hist_counts && (o.hist_bins < 1 || o.hist_bins > (1 << 24))) return PN_EINVAL;
    if (N == 0) {
        if (o.hist_counts) {              // the histogram of nothing: zero counts, as pn_histogram writes them
            const size_t hb = sizeof(unsigned long long) * 3 * (size_t)o.hist_bins, sb = sizeof(unsigned long long) * 3;
            if (o.host_buffers) { memset(o.hist_counts, 0, hb); if (o.hist_skipped) memset(o.hist_skipped, 0, sb); }
            else {
                CK(cudaMemsetAsync(o.hist_counts, 0, hb, (cudaStream_t)o.stream));
                if (o.hist_skipped) CK(cudaMemsetAsync(o.hist_skipped, 0, sb, (cudaStream_t)o.stream));
                if (!o.async) CK(cudaStreamSynchronize((cudaStream_t)o.stream));
            }
        }
        return PN_OK;
    }
    if (!init_states || !masses || !out_final || !out_steps) return PN_EINVAL;
    if (precision != PN_FP64 && precision != PN_FP32 && precision != PN_MIXED) return PN_EINVAL;
    const bool fixed = o.fixed_steps > 0;
    if (!fixed) {
        if (!(rtol > 0.0) || !(atol >= 0.0) || !(omegaf > 0.0)) return PN_EINVAL;
        if (omega0 > 0.0 && !(omega0 < omegaf)) return PN_EINVAL;
    }
    if (o.async && o.host_buffers) return PN_EINVAL;
    if (o.block_threads != 0 && o.block_threads != 128 && o.block_threads != 256) return PN_EINVAL;
    cudaStream_t s = (cudaStream_t)o.stream;
    Ctx& c = *ctx_for(o.stream);
    const int n = (int)N;
    int rc;
    if ((rc = ensure_events(c)) != PN_OK) return rc;

    // ---- host buffers: stage through device scratch ----
    const double* d_init = init_states;
    const double* d_m = masses;
    double* d_final = out_final;
    int* d_steps = out_steps;
    double* d_time = o.out_time;
    int* d_rej = o.out_rejected;
    if (o.host_buffers) {
        if ((rc = c.h_init.ensure(sizeof(double) * 10 * (size_t)n)) != PN_OK) return rc;
        if ((rc = c.h_m.ensure(sizeof(double) * 2 * (size_t)n)) != PN_OK) return rc;
        if ((rc = c.h_final.ensure(sizeof(double) * 10 * (size_t)n)) != PN_OK) return rc;
        if ((rc = c.h_steps.ensure(sizeof(int) * (size_t)n)) != PN_OK) return rc;
        if (o.out_time && (rc = c.h_time.ensure(sizeof(double) * (size_t)n)) != PN_OK) return rc;
        if (o.out_rejected && (rc = c.h_rej.ensure(sizeof(int) * (size_t)n)) != PN_OK) return rc;
        CK(cudaMemcpyAsync(c.h_init.p, init_states, sizeof(double) * 10 * (size_t)n, cudaMemcpyHostToDevice, s));
        CK(cudaMemcpyAsync(c.h_m.p, masses, sizeof(double) * 2 * (size_t)n, cudaMemcpyHostToDevice, s));
        d_init = (const double*)c.h_init.p; d_m = (const double*)c.h_m.p;
        d_final = (double*)c.h_final.p; d_steps = (int*)c.h_steps.p;
        d_time = o.out_time ? (double*)c.h_time.p : nullptr;
        d_rej = o.out_rejected ? (int*)c.h_rej.p : nullptr;
    }

    // ---- per-call work counters and status (stream-ordered: an earlier call on this stream has finished with them) ----
    if ((rc = c.small.ensure(sizeof(Small))) != PN_OK) return rc;
    Small* small = (Small*)c.small.p;
    CK(cudaMemsetAsync(small, 0, sizeof(Small), s));
    PnKernelParams p;
    memset(&p, 0, sizeof p);
    CK(cudaEventRecord(c.ev[0], s));
    // ---- SoA staging ----
    if (o.layout == 0) {
        if ((rc = c.soa_in.ensure(sizeof(double) * 10 * (size_t)n)) != PN_OK) return rc;
        if ((rc = c.soa_m.ensure(sizeof(double) * 2 * (size_t)n)) != PN_OK) return rc;
        if ((rc = c.soa_out.ensure(sizeof(double) * 10 * (size_t)n)) != PN_OK) return rc;
        CK(pn_launch_aos_to_soa(d_init, (double*)c.soa_in.p, n, 10, s));
        CK(pn_launch_aos_to_soa(d_m, (double*)c.soa_m.p, n, 2, s));
        p.y0 = (const double*)c.soa_in.p; p.masses = (const double*)c.soa_m.p; p.yf = (double*)c.soa_out.p;
    } else {
        p.y0 = d_init; p.masses = d_m; p.yf = d_final;
    }
    if (!o.input_order && !fixed && n > 1024) {
        // longest-expected-first queue order: keys from the seed kernel, then a bucket sort
        if ((rc = c.keys.ensure(sizeof(float) * (size_t)n)) != PN_OK) return rc;
        if ((rc = c.order.ensure(sizeof(int) * (size_t)n)) != PN_OK) return rc;
        if ((rc = c.ord_scr.ensure(sizeof(unsigned) * (PN_ORDER_BUCKETS + 2))) != PN_OK) return rc;
        p.keys = (float*)c.keys.p; p.order_out = (int*)c.order.p; p.order = p.order_out;
        p.order_scratch = (unsigned*)c.ord_scr.p;
    }
    CK(cudaEventRecord(c.ev[1], s));
    p.steps = d_steps; p.time = d_time; p.rejected = d_rej;
    p.n = n;
    p.omega0 = omega0; p.omegaf = omegaf; p.rtol = rtol; p.atol = atol; p.h0 = o.h0;
    p.tau = o.tau_land > 0.0 ? o.tau_land : (precision == PN_FP64 ? 1e-13 : (precision == PN_MIXED ? 1e-8 : 3e-7));
    // range of the series for (M omega)^{1/3} and ln(M omega) in the FP64 fast kernel (pn_rhs.cuh): |1 - x/x0| <= emax.
    // 0.03 up to rtol 1e-10 and in fixed-step mode (truncation s10 emax^9 = 6e-17 relative); at looser tolerances the
    // largest range whose truncation stays below 1e-3 rtol, at most 0.2: a run at rtol 1e-7 need not evaluate f to 1e-16.
    // A system with an ACCEPTED step beyond the range goes to the wide-range redo pass.
    p.emax = 0.03;
    if (!fixed && rtol > 1e-10) { p.emax = pow(1e-3 * rtol / 0.0852, 1.0 / 9.0); if (p.emax > 0.2) p.emax = 0.2; }
    pn_host_series(o.term_mask, p.qc);
    p.max_steps = o.max_steps > 0 ? o.max_steps : 10000000;
    p.fixed_steps = fixed ? o.fixed_steps : 0;
    p.mask = o.term_mask;
    if ((rc = c.redo.ensure(sizeof(int) * (size_t)n)) != PN_OK) return rc;
    if (!fixed) {
        if ((rc = c.seed.ensure((precision == PN_FP64 ? sizeof(double) : sizeof(float)) * 40 * (size_t)n)) != PN_OK) return rc;
        p.seed = c.seed.p;
    }
    p.queue = &small->queue; p.counters = small->counters; p.status = &small->status;
    p.queue2 = &small->queue2; p.redo_count = &small->redo_count; p.redo_list = (int*)c.redo.p;
    p.nonuniform = &small->nonuniform; p.uni_row = small->uni_row;
    p.uni_slot = c.slot;
    CK(pn_launch_integrate(p, precision, o.block_threads, o.grid_blocks, s, o.variant));
    CK(cudaEventRecord(c.ev[2], s));
    if (o.layout == 0) CK(pn_launch_soa_to_aos((const double*)c.soa_out.p, d_final, n, 10, s));
    CK(cudaEventRecord(c.ev[3], s));
    // optional: the histograms of the final states while they are on the device (pn_options.hist_counts)
    unsigned long long* d_hc = o.hist_counts;
    unsigned long long* d_hs = o.hist_skipped;
    if (o.hist_counts) {
        if (o.host_buffers) {
            if ((rc = c.h_counts.ensure(sizeof(unsigned long long) * (3 * (size_t)o.hist_bins + 3))) != PN_OK) return rc;
            d_hc = (unsigned long long*)c.h_counts.p;
            d_hs = d_hc + 3 * (size_t)o.hist_bins;
        }
        CK(pn_launch_histogram(d_final, o.layout, N, o.hist_bins, d_hc, d_hs, s));
        CK(cudaEventRecord(c.ev[4], s));
    }

    if (o.async) {
        // the call's status is folded into the stream's sticky word, which pn_stream_status() reads and clears
        if ((rc = c.sticky.ensure(sizeof(int))) != PN_OK) return rc;
        if (!c.async_pending) CK(cudaMemsetAsync(c.sticky.p, 0, sizeof(int), s));
        CK(pn_launch_fold_status(&small->status, (int*)c.sticky.p, s));
        c.async_pending = true;
        return PN_OK;
    }
    if (o.host_buffers) {
        CK(cudaMemcpyAsync(out_final, d_final, sizeof(double) * 10 * (size_t)n, cudaMemcpyDeviceToHost, s));
        CK(cudaMemcpyAsync(out_steps, d_steps, sizeof(int) * (size_t)n, cudaMemcpyDeviceToHost, s));
        if (o.out_time) CK(cudaMemcpyAsync(o.out_time, d_time, sizeof(double) * (size_t)n, cudaMemcpyDeviceToHost, s));
        if (o.out_rejected) CK(cudaMemcpyAsync(o.out_rejected, d_rej, sizeof(int) * (size_t)n, cudaMemcpyDeviceToHost, s));
        if (o.hist_counts) CK(cudaMemcpyAsync(o.hist_counts, d_hc, sizeof(unsigned long long) * 3 * (size_t)o.hist_bins, cudaMemcpyDeviceToHost, s));
        if (o.hist_counts && o.hist_skipped) CK(cudaMemcpyAsync(o.hist_skipped, d_hs, sizeof(unsigned long long) * 3, cudaMemcpyDeviceToHost, s));
    }
    Small hs;
    CK(cudaMemcpyAsync(&hs, small, sizeof hs, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    CK(cudaGetLastError());
    for (int i = 0; i < 3; ++i) CK(cudaEventElapsedTime(&g_ms[i], c.ev[i], c.ev[i + 1]));
    if (o.hist_counts) CK(cudaEventElapsedTime(&g_ms[3], c.ev[3], c.ev[4]));
    memcpy(g_counters, hs.counters, sizeof g_counters);
    g_redo_count = hs.redo_count;
    return hs.status;
}

extern "C" int pn_integrate(const double* init_states, const double* masses, long long N, double omega0,
                            double omegaf, double rtol, double atol, int precision, double* out_final,
                            int* out_steps)
{
    return pn_integrate_ex(init_states, masses, N, omega0, omegaf, rtol, atol, precision, out_final, out_steps, nullptr);
}

extern "C" int pn_histogram_ex(const double* final_states, long long N, int bins, unsigned long long* counts,
                               unsigned long long* n_skipped, const pn_options* opt_in)
{
    pn_options o;
    default_options(&o);
    if (opt_in) {
        if (opt_in->size != (int)sizeof(pn_options)) return PN_EINVAL;
        o = *opt_in;
    }
    if (N < 0 || bins < 1 || bins > (1 << 24) || !counts) return PN_EINVAL;
    if (N > 0 && !final_states) return PN_EINVAL;
    if (o.async && o.host_buffers) return PN_EINVAL;
    cudaStream_t s = (cudaStream_t)o.stream;
    Ctx& c = *ctx_for(o.stream);
    int rc;
    if ((rc = ensure_events(c)) != PN_OK) return rc;
    const double* d_st = final_states;
    unsigned long long* d_counts = counts;
    unsigned long long* d_skip = n_skipped;
    if (o.host_buffers) {
        if (N > 0) {
            if ((rc = c.h_final.ensure(sizeof(double) * 10 * (size_t)N)) != PN_OK) return rc;
            CK(cudaMemcpyAsync(c.h_final.p, final_states, sizeof(double) * 10 * (size_t)N, cudaMemcpyHostToDevice, s));
            d_st = (const double*)c.h_final.p;
        }
        if ((rc = c.h_counts.ensure(sizeof(unsigned long long) * (3 * (size_t)bins + 3))) != PN_OK) return rc;
        d_counts = (unsigned long long*)c.h_counts.p;
        d_skip = d_counts + 3 * (size_t)bins;
    }
    // AoS, 16-byte aligned, moderate bin count: the bulk-copy streaming kernel of pn_stats.cu in its final-only mode
    // (3.1 TB/s at 2^22 systems); otherwise (SoA layout, odd alignment, huge bin counts) the plain kernel of pn_aux.cu
    const bool bulk = o.layout == 0 && N > 0 && bins <= 8192 && (((uintptr_t)d_st) & 15u) == 0;
    if (bulk && (rc = c.st_scratch.ensure(pn_stats_scratch_bytes(N, 0, nullptr))) != PN_OK) return rc;
    CK(cudaEventRecord(c.ev[3], s));
    if (bulk) {
        if (d_skip) CK(cudaMemsetAsync(d_skip, 0, sizeof(unsigned long long) * 3, s));
        CK(pn_launch_stats(nullptr, d_st, nullptr, N, 0, bins, 0, c.st_scratch.p, nullptr, nullptr, d_skip, d_counts, nullptr,
                           nullptr, nullptr, s));
    } else {
        CK(pn_launch_histogram(d_st, o.layout, N, bins, d_counts, d_skip, s));
    }
    CK(cudaEventRecord(c.ev[4], s));
    if (o.async) return PN_OK;
    if (o.host_buffers) {
        CK(cudaMemcpyAsync(counts, d_counts, sizeof(unsigned long long) * 3 * (size_t)bins, cudaMemcpyDeviceToHost, s));
        if (n_skipped) CK(cudaMemcpyAsync(n_skipped, d_skip, sizeof(unsigned long long) * 3, cudaMemcpyDeviceToHost, s));
    }
    CK(cudaStreamSynchronize(s));
    CK(cudaGetLastError());
    CK(cudaEventElapsedTime(&g_ms[3], c.ev[3], c.ev[4]));
    return PN_OK;
}

extern "C" int pn_histogram(const double* final_states, long long N, int bins, unsigned long long* counts,
                            unsigned long long* n_skipped)
{
    return pn_histogram_ex(final_states, N, bins, counts, n_skipped, nullptr);
}

extern "C" int pn_statistics(const double* init_states, const double* final_states, const int* steps, long long N,
                             long long group_size, int bins1, int bins2, const pn_stats_out* out_in,
                             const pn_options* opt_in)
{
    pn_options o;
    default_options(&o);
    if (opt_in) {
        if (opt_in->size != (int)sizeof(pn_options)) return PN_EINVAL;
        o = *opt_in;
    }
    if (!out_in || out_in->size != (int)sizeof(pn_stats_out)) return PN_EINVAL;
    pn_stats_out out = *out_in;
    if (N < 0 || N > 0x7fffffffLL * 8 || o.layout != 0) return PN_EINVAL;
    if (N > 0 && !final_states) return PN_EINVAL;
    if (o.async && o.host_buffers) return PN_EINVAL;
    if (bins1 > 8192 || bins2 > 4096) return PN_EINVAL;
    if (bins1 < 1) { bins1 = 0; out.hist1 = nullptr; }
    if (bins2 < 1 || !init_states) { bins2 = 0; out.hist2 = nullptr; }
    if (!out.hist2) { if (out.hist2_max || out.hist2_norm) return PN_EINVAL; }
    const long long gs = group_size > 0 ? group_size : N;
    if (N > 0 && N % gs != 0) return PN_EINVAL;
    const long long G = N > 0 ? N / gs : 0;
    if (N == 0) return PN_OK;
    if (!o.host_buffers && (((uintptr_t)final_states & 15u) || ((uintptr_t)init_states & 15u))) return PN_EINVAL;
    cudaStream_t s = (cudaStream_t)o.stream;
    Ctx& c = *ctx_for(o.stream);
    int rc;
    if ((rc = ensure_events(c)) != PN_OK) return rc;
    if ((rc = c.st_scratch.ensure(pn_stats_scratch_bytes(N, group_size, nullptr))) != PN_OK) return rc;

    const double* d_init = init_states;
    const double* d_fin = final_states;
    const int* d_steps = steps;
    pn_stats_out d = out;
    // host buffers: stage inputs and outputs through device scratch
    const size_t row = sizeof(double) * 10 * (size_t)N;
    const size_t b_r = sizeof(double) * 3 * (size_t)G, b_m = 6 * b_r, b_sk = sizeof(unsigned long long) * 3 * (size_t)G;
    const size_t b_h1 = sizeof(unsigned long long) * 3 * (size_t)bins1 * G, b_h2 = sizeof(unsigned long long) * 3 * (size_t)bins2 * bins2 * G;
    if (o.host_buffers) {
        const size_t in_bytes = row * (init_states ? 2 : 1) + (steps ? sizeof(int) * (size_t)N : 0);
        if ((rc = c.st_in.ensure(in_bytes)) != PN_OK) return rc;
        char* q = (char*)c.st_in.p;
        CK(cudaMemcpyAsync(q, final_states, row, cudaMemcpyHostToDevice, s));
        d_fin = (const double*)q; q += row;
        if (init_states) { CK(cudaMemcpyAsync(q, init_states, row, cudaMemcpyHostToDevice, s)); d_init = (const double*)q; q += row; }
        if (steps) { CK(cudaMemcpyAsync(q, steps, sizeof(int) * (size_t)N, cudaMemcpyHostToDevice, s)); d_steps = (const int*)q; }
        if ((rc = c.st_out.ensure(b_r + b_m + 2 * b_sk + b_h1 + 2 * b_h2 + 64)) != PN_OK) return rc;
        char* w = (char*)c.st_out.p;
        auto take = [&](size_t bytes) { char* r = w; w += (bytes + 15) & ~(size_t)15; return r; };
        if (out.pearson_r) d.pearson_r = (double*)take(b_r);
        if (out.moments) d.moments = (double*)take(b_m);
        if (out.n_skipped) d.n_skipped = (unsigned long long*)take(b_sk);
        if (out.hist1) d.hist1 = (unsigned long long*)take(b_h1);
        if (out.hist2) d.hist2 = (unsigned long long*)take(b_h2);
        if (out.hist2_max) d.hist2_max = (unsigned long long*)take(b_sk);
        if (out.hist2_norm) d.hist2_norm = (double*)take(b_h2);
    }
    CK(cudaEventRecord(c.ev[3], s));
    CK(pn_launch_stats(d_init, d_fin, d_steps, N, group_size, bins1, bins2, c.st_scratch.p, d.pearson_r, d.moments,
                       d.n_skipped, d.hist1, d.hist2, d.hist2_max, d.hist2_norm, s));
    CK(cudaEventRecord(c.ev[4], s));
    if (o.async) return PN_OK;
    if (o.host_buffers) {
        if (out.pearson_r) CK(cudaMemcpyAsync(out.pearson_r, d.pearson_r, b_r, cudaMemcpyDeviceToHost, s));
        if (out.moments) CK(cudaMemcpyAsync(out.moments, d.moments, b_m, cudaMemcpyDeviceToHost, s));
        if (out.n_skipped) CK(cudaMemcpyAsync(out.n_skipped, d.n_skipped, b_sk, cudaMemcpyDeviceToHost, s));
        if (out.hist1) CK(cudaMemcpyAsync(out.hist1, d.hist1, b_h1, cudaMemcpyDeviceToHost, s));
        if (out.hist2) CK(cudaMemcpyAsync(out.hist2, d.hist2, b_h2, cudaMemcpyDeviceToHost, s));
        if (out.hist2_max) CK(cudaMemcpyAsync(out.hist2_max, d.hist2_max, b_sk, cudaMemcpyDeviceToHost, s));
        if (out.hist2_norm) CK(cudaMemcpyAsync(out.hist2_norm, d.hist2_norm, b_h2, cudaMemcpyDeviceToHost, s));
    }
    CK(cudaStreamSynchronize(s));
    CK(cudaGetLastError());
    CK(cudaEventElapsedTime(&g_ms[3], c.ev[3], c.ev[4]));
    return PN_OK;
}

extern "C" int pn_merge_statistics(const double* parts, int n_parts, int n_groups, double* moments_out, double* pearson_r_out,
                                   const pn_options* opt_in)
{
    pn_options o;
    default_options(&o);
    if (opt_in) {
        if (opt_in->size != (int)sizeof(pn_options)) return PN_EINVAL;
        o = *opt_in;
    }
    if (n_parts < 1 || n_groups < 0 || o.host_buffers || (n_groups > 0 && !parts)) return PN_EINVAL;
    cudaStream_t s = (cudaStream_t)o.stream;
    CK(pn_launch_stats_merge(parts, n_parts, n_groups, moments_out, pearson_r_out, s));
    if (o.async) return PN_OK;
    CK(cudaStreamSynchronize(s));
    CK(cudaGetLastError());
    return PN_OK;
}

extern "C" int pn_generate(const pn_ensemble* ens, int n_ensembles, long long n_total, long long first, long long count,
                           double* init_states, double* masses, const pn_options* opt_in)
{
    pn_options o;
    default_options(&o);
    if (opt_in) {
        if (opt_in->size != (int)sizeof(pn_options)) return PN_EINVAL;
        o = *opt_in;
    }
    if (!ens || n_ensembles < 1 || n_ensembles > 65536 || n_total < 0 || first < 0 || count < 0 || first + count > n_total ||
        o.layout != 0 || (o.async && o.host_buffers))
        return PN_EINVAL;
    if (n_total > (1LL << 59)) return PN_EINVAL;                       // 7 n_total variates must fit the 2^64 word stream
    if (count == 0) return PN_OK;
    if (!init_states || !masses) return PN_EINVAL;
    if (!o.host_buffers && ((((uintptr_t)init_states) | ((uintptr_t)masses)) & 15u)) return PN_EINVAL;
    struct Spec { unsigned long long k0, k1; double v[9]; };
    std::vector<Spec> h(n_ensembles);
    for (int e = 0; e < n_ensembles; ++e) {
        const pn_ensemble& x = ens[e];
        if (x.size != (int)sizeof(pn_ensemble) || !(x.omega0 > 0.0) || !(x.q_lo > 0.0) || !(x.chi1_lo >= 0.0) || !(x.chi2_lo >= 0.0) ||
            !(x.m1_fixed < 1.0))
            return PN_EINVAL;
        h[e].k0 = x.key[0]; h[e].k1 = x.key[1];
        const double v[9] = {x.omega0, x.q_lo, x.q_hi, x.m1_fixed, x.chi1_lo, x.chi1_hi, x.chi2_lo, x.chi2_hi, x.s1_tilt_deg};
        memcpy(h[e].v, v, sizeof v);
    }
    cudaStream_t s = (cudaStream_t)o.stream;
    Ctx& c = *ctx_for(o.stream);
    int rc;
    if ((rc = ensure_events(c)) != PN_OK) return rc;
    if ((rc = c.gen_specs.ensure(sizeof(Spec) * (size_t)n_ensembles)) != PN_OK) return rc;
    CK(cudaMemcpyAsync(c.gen_specs.p, h.data(), sizeof(Spec) * (size_t)n_ensembles, cudaMemcpyHostToDevice, s));
    CK(cudaStreamSynchronize(s));      // h is a local: the copy must have left it before we return
    const size_t rows = (size_t)n_ensembles * (size_t)count;
    double* d_y = init_states;
    double* d_m = masses;
    if (o.host_buffers) {
        if ((rc = c.gen_y.ensure(sizeof(double) * 10 * rows)) != PN_OK) return rc;
        if ((rc = c.gen_m.ensure(sizeof(double) * 2 * rows)) != PN_OK) return rc;
        d_y = (double*)c.gen_y.p; d_m = (double*)c.gen_m.p;
    }
    CK(cudaEventRecord(c.ev[0], s));
    CK(pn_launch_generate(c.gen_specs.p, n_ensembles, n_total, first, count, d_y, d_m, s));
    CK(cudaEventRecord(c.ev[1], s));
    if (o.async) return PN_OK;
    if (o.host_buffers) {
        CK(cudaMemcpyAsync(init_states, d_y, sizeof(double) * 10 * rows, cudaMemcpyDeviceToHost, s));
        CK(cudaMemcpyAsync(masses, d_m, sizeof(double) * 2 * rows, cudaMemcpyDeviceToHost, s));
    }
    CK(cudaStreamSynchronize(s));
    CK(cudaGetLastError());
    CK(cudaEventElapsedTime(&g_ms[0], c.ev[0], c.ev[1]));
    return PN_OK;
}

// Systems per launch of a fused ensemble run: bounds the redo list (4 B per system) so that the device memory a run
// needs does not grow with its size; 2^22 systems keep the persistent grid busy for > 100 resident-lane refills.
#define PN_FUSED_CHUNK (1LL << 22)

extern "C" int pn_run_ensembles(const pn_ensemble* ens, int n_ensembles, long long n_total, long long first, long long count,
                                double omegaf, double rtol, double atol, int precision, int bins1, int bins2,
                                const pn_stats_out* out_in, const pn_options* opt_in)
{
    pn_options o;
    default_options(&o);
    if (opt_in) {
        if (opt_in->size != (int)sizeof(pn_options)) return PN_EINVAL;
        o = *opt_in;
    }
    if (!out_in || out_in->size != (int)sizeof(pn_stats_out)) return PN_EINVAL;
    pn_stats_out out = *out_in;
    if (!ens || n_ensembles < 1 || n_ensembles > 65536 || n_total < 0 || first < 0 || count < 0 || first + count > n_total ||
        o.layout != 0 || (o.async && o.host_buffers) || o.fixed_steps > 0)
        return PN_EINVAL;
    if (n_total > (1LL << 59) || (long long)n_ensembles * count > (1LL << 40)) return PN_EINVAL;
    if (precision != PN_FP64) return PN_EINVAL;                          // the fused kernel is the FP64 integrator
    if (!(rtol > 0.0) || !(atol >= 0.0) || !(omegaf > 0.0)) return PN_EINVAL;
    if (bins1 > (1 << 24) || bins2 > 4096) return PN_EINVAL;
    if (bins1 < 1) { bins1 = 0; out.hist1 = nullptr; }
    if (bins2 < 1) { bins2 = 0; out.hist2 = nullptr; }
    if (!out.hist2 && (out.hist2_max || out.hist2_norm)) return PN_EINVAL;
    struct Spec { unsigned long long k0, k1; double v[9]; };
    std::vector<Spec> h(n_ensembles);
    for (int e = 0; e < n_ensembles; ++e) {
        const pn_ensemble& x = ens[e];
        if (x.size != (int)sizeof(pn_ensemble) || !(x.omega0 > 0.0) || !(x.omega0 < omegaf) || !(x.q_lo > 0.0) || !(x.chi1_lo >= 0.0) ||
            !(x.chi2_lo >= 0.0) || !(x.m1_fixed < 1.0))
            return PN_EINVAL;
        h[e].k0 = x.key[0]; h[e].k1 = x.key[1];
        const double v[9] = {x.omega0, x.q_lo, x.q_hi, x.m1_fixed, x.chi1_lo, x.chi1_hi, x.chi2_lo, x.chi2_hi, x.s1_tilt_deg};
        memcpy(h[e].v, v, sizeof v);
    }
    if (count == 0) return PN_OK;
    cudaStream_t s = (cudaStream_t)o.stream;
    Ctx& c = *ctx_for(o.stream);
    int rc;
    if ((rc = ensure_events(c)) != PN_OK) return rc;
    const long long G = n_ensembles, N = G * count;
    if ((rc = c.gen_specs.ensure(sizeof(Spec) * (size_t)n_ensembles)) != PN_OK) return rc;
    CK(cudaMemcpyAsync(c.gen_specs.p, h.data(), sizeof(Spec) * (size_t)n_ensembles, cudaMemcpyHostToDevice, s));
    CK(cudaStreamSynchronize(s));      // h is a local: the copy must have left it before we return

    // outputs (device, or staged for host buffers) and scratch: running moments, locks, skipped counts, redo list
    const size_t b_r = sizeof(double) * 3 * (size_t)G, b_m = 6 * b_r, b_sk = sizeof(unsigned long long) * 3 * (size_t)G;
    const size_t b_h1 = sizeof(unsigned long long) * 3 * (size_t)bins1 * G, b_h2 = sizeof(unsigned long long) * 3 * (size_t)bins2 * bins2 * G;
    pn_stats_out d = out;
    if (o.host_buffers) {
        if ((rc = c.st_out.ensure(b_r + b_m + 2 * b_sk + b_h1 + 2 * b_h2 + 128)) != PN_OK) return rc;
        char* w = (char*)c.st_out.p;
        auto take = [&](size_t bytes) { char* r = w; w += (bytes + 15) & ~(size_t)15; return r; };
        if (out.pearson_r) d.pearson_r = (double*)take(b_r);
        if (out.moments) d.moments = (double*)take(b_m);
        if (out.n_skipped) d.n_skipped = (unsigned long long*)take(b_sk);
        if (out.hist1) d.hist1 = (unsigned long long*)take(b_h1);
        if (out.hist2) d.hist2 = (unsigned long long*)take(b_h2);
        if (out.hist2_max) d.hist2_max = (unsigned long long*)take(b_sk);
        if (out.hist2_norm) d.hist2_norm = (double*)take(b_h2);
    }
    const long long chunk = N < PN_FUSED_CHUNK ? N : PN_FUSED_CHUNK;
    const size_t scr_bytes = b_m + b_sk + sizeof(int) * (size_t)G + sizeof(int) * (size_t)chunk + 64;
    if ((rc = c.fu_scr.ensure(scr_bytes)) != PN_OK) return rc;
    if ((rc = c.small.ensure(sizeof(Small))) != PN_OK) return rc;
    Small* small = (Small*)c.small.p;
    char* q = (char*)c.fu_scr.p;
    double* f_mom = (double*)q; q += b_m;
    unsigned long long* f_skip = (unsigned long long*)q; q += b_sk;
    int* f_lock = (int*)q; q += sizeof(int) * (size_t)G;
    q = (char*)(((uintptr_t)q + 15) & ~(uintptr_t)15);
    int* redo_list = (int*)q;
    CK(cudaMemsetAsync(c.fu_scr.p, 0, b_m + b_sk + sizeof(int) * (size_t)G, s));
    CK(cudaMemsetAsync(small, 0, sizeof(Small), s));
    if (d.hist1) CK(cudaMemsetAsync(d.hist1, 0, b_h1, s));
    if (d.hist2) CK(cudaMemsetAsync(d.hist2, 0, b_h2, s));

    PnKernelParams p;
    memset(&p, 0, sizeof p);
    p.omega0 = 0.0; p.omegaf = omegaf; p.rtol = rtol; p.atol = atol; p.h0 = o.h0;
    p.tau = o.tau_land > 0.0 ? o.tau_land : 1e-13;
    p.emax = 0.03;
    if (rtol > 1e-10) { p.emax = pow(1e-3 * rtol / 0.0852, 1.0 / 9.0); if (p.emax > 0.2) p.emax = 0.2; }
    pn_host_series(o.term_mask, p.qc);
    p.max_steps = o.max_steps > 0 ? o.max_steps : 10000000;
    p.mask = o.term_mask;
    p.queue = &small->queue; p.counters = small->counters; p.status = &small->status;
    p.queue2 = &small->queue2; p.redo_count = &small->redo_count; p.redo_list = redo_list;
    p.nonuniform = &small->nonuniform; p.uni_row = small->uni_row;
    p.uni_slot = -1;
    p.f_specs = c.gen_specs.p; p.f_n_total = n_total; p.f_first = first; p.f_count = count;
    p.f_mom = f_mom; p.f_lock = f_lock; p.f_skipped = f_skip; p.f_hist1 = d.hist1; p.f_hist2 = d.hist2;
    p.f_bins1 = bins1; p.f_bins2 = bins2;
    // Ensembles that all have the SAME fixed masses (every ensemble of an equal-mass sweep over chi of the paper's section V;
    // the 3.6e8-system uniformity run): the uniform-mass fast kernel, constants from this stream context's row of the table
    // (DESIGN.md 7.8).  Ensembles with different masses share chunks, so they take the generic kernel (a launch per ensemble
    // would pay a drain tail per ensemble).
    // Cost order mixes the ensembles of a chunk: consecutive finishes of a thread then belong to arbitrary ensembles, and
    // with more ensembles than the block's table holds (PN_FW) nearly every finish evicts a table entry into the global
    // record under the ensemble's global lock.  Measured on a B200, 2^20 systems, equal-mass chi sweep: 16 ensembles 335 ms
    // in cost order against 61.6 ms in index order, 64 ensembles 133 against 63 ms; up to 4 ensembles the two orders take
    // the same time (profiles/r3_fused_sweep_order.md).  So: cost order only while every ensemble has a table entry.
    if (!o.input_order && N > 1024 && (G <= PN_FW || (o.variant & 4))) {
        // longest-expected-first queue order inside every chunk: keys + order, 8 bytes per system of a chunk
        const size_t nc = (size_t)(N < chunk ? N : chunk);
        if ((rc = c.keys.ensure(sizeof(float) * nc)) != PN_OK) return rc;
        if ((rc = c.order.ensure(sizeof(int) * nc)) != PN_OK) return rc;
        if ((rc = c.ord_scr.ensure(sizeof(unsigned) * (PN_ORDER_BUCKETS + 2))) != PN_OK) return rc;
        p.keys = (float*)c.keys.p; p.order_out = (int*)c.order.p; p.order_scratch = (unsigned*)c.ord_scr.p;
    }
    // The same decision the unfused chain takes over the concatenated batch (pn_seed_kernel compares every system's masses
    // with system 0's): uniform iff EVERY ensemble of the call has fixed masses and they are the same pair of doubles.  The
    // masses are formed here exactly as pn_fused_row_kernel / the generator form them (one rounded operation each).
    auto fixed_pair = [](const pn_ensemble& x, double& m1, double& m2) {
        if (x.m1_fixed > 0.0) { m1 = x.m1_fixed; m2 = 1.0 - m1; return true; }
        if (!(x.q_hi > x.q_lo)) { const double dq = 1.0 + x.q_lo; m1 = 1.0 / dq; m2 = x.q_lo / dq; return true; }
        return false;
    };
    double um1 = 0.0, um2 = 0.0;
    bool fixed_masses = fixed_pair(ens[0], um1, um2);
    for (int e = 1; e < n_ensembles && fixed_masses; ++e) {
        double a = 0.0, b = 0.0;
        fixed_masses = fixed_pair(ens[e], a, b) && a == um1 && b == um2;
    }
    const int uni_slot = (fixed_masses && !(o.variant & 1)) ? c.slot : -1;
    CK(cudaEventRecord(c.ev[1], s));
    for (long long lo = 0; lo < N; lo += chunk) {
        if (lo > 0) {                    // fresh work counters for every chunk; step counters and status accumulate
            CK(cudaMemsetAsync(&small->queue, 0, sizeof(unsigned), s));
            CK(cudaMemsetAsync(&small->queue2, 0, 2 * sizeof(unsigned), s));
        }
        p.n = (int)(N - lo < chunk ? N - lo : chunk);
        p.f_base = lo;
        CK(pn_launch_fused(p, o.grid_blocks, s, uni_slot, 0));
    }
    CK(cudaEventRecord(c.ev[2], s));
    if (d.pearson_r || d.moments) CK(pn_launch_stats_merge(f_mom, 1, (int)G, d.moments, d.pearson_r, s));
    if (d.n_skipped) CK(cudaMemcpyAsync(d.n_skipped, f_skip, b_sk, cudaMemcpyDeviceToDevice, s));
    if (d.hist2 && (d.hist2_max || d.hist2_norm)) CK(pn_launch_stats_norm(d.hist2, G * 3, bins2 * bins2, d.hist2_max, d.hist2_norm, s));
    if (o.async) {
        if ((rc = c.sticky.ensure(sizeof(int))) != PN_OK) return rc;
        if (!c.async_pending) CK(cudaMemsetAsync(c.sticky.p, 0, sizeof(int), s));
        CK(pn_launch_fold_status(&small->status, (int*)c.sticky.p, s));
        c.async_pending = true;
        return PN_OK;
    }
    if (o.host_buffers) {
        if (out.pearson_r) CK(cudaMemcpyAsync(out.pearson_r, d.pearson_r, b_r, cudaMemcpyDeviceToHost, s));
        if (out.moments) CK(cudaMemcpyAsync(out.moments, d.moments, b_m, cudaMemcpyDeviceToHost, s));
        if (out.n_skipped) CK(cudaMemcpyAsync(out.n_skipped, d.n_skipped, b_sk, cudaMemcpyDeviceToHost, s));
        if (out.hist1) CK(cudaMemcpyAsync(out.hist1, d.hist1, b_h1, cudaMemcpyDeviceToHost, s));
        if (out.hist2) CK(cudaMemcpyAsync(out.hist2, d.hist2, b_h2, cudaMemcpyDeviceToHost, s));
        if (out.hist2_max) CK(cudaMemcpyAsync(out.hist2_max, d.hist2_max, b_sk, cudaMemcpyDeviceToHost, s));
        if (out.hist2_norm) CK(cudaMemcpyAsync(out.hist2_norm, d.hist2_norm, b_h2, cudaMemcpyDeviceToHost, s));
    }
    Small hs;
    CK(cudaMemcpyAsync(&hs, small, sizeof hs, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    CK(cudaGetLastError());
    CK(cudaEventElapsedTime(&g_ms[1], c.ev[1], c.ev[2]));
    memcpy(g_counters, hs.counters, sizeof g_counters);
    g_redo_count = hs.redo_count;          // of the last chunk
    return hs.status;
}

extern "C" int pn_selfcheck(const double* init_states, const double* masses, const double* final_states, const double* times,
                            long long N, double omegaf, double fraction, const unsigned long long key[2], double rtol_ref,
                            double atol_ref, pn_check_out* out, long long* checked_indices, long long max_indices,
                            const pn_options* opt_in)
{
    pn_options o;
    default_options(&o);
    if (opt_in) {
        if (opt_in->size != (int)sizeof(pn_options)) return PN_EINVAL;
        o = *opt_in;
    }
    if (!out || out->size != (int)sizeof(pn_check_out) || !key || N < 0 || N > 0x7fffffffLL / 16 || o.async || o.layout != 0 ||
        !(fraction >= 0.0) || !(fraction <= 1.0) || !(omegaf > 0.0))
        return PN_EINVAL;
    if (N > 0 && (!init_states || !masses || !final_states)) return PN_EINVAL;
    if (!(rtol_ref > 0.0)) rtol_ref = 1e-10;
    if (!(atol_ref > 0.0)) atol_ref = 1e-12;
    out->n_checked = out->n_failed_ref = 0;
    out->max_time_rel_dev = 0.0; out->ms_reference = 0.0f;
    for (int k = 0; k < 3; ++k) { out->max_dot_dev[k] = 0.0; out->worst_index[k] = -1; }
    if (N == 0) return PN_OK;
    cudaStream_t s = (cudaStream_t)o.stream;
    Ctx& c = *ctx_for(o.stream);
    int rc;
    const double* d_init = init_states; const double* d_m = masses; const double* d_fin = final_states; const double* d_t = times;
    if (o.host_buffers) {
        const size_t rows = sizeof(double) * (size_t)N;
        if ((rc = c.ck_in.ensure(rows * 23)) != PN_OK) return rc;
        double* q = (double*)c.ck_in.p;
        CK(cudaMemcpyAsync(q, init_states, rows * 10, cudaMemcpyHostToDevice, s)); d_init = q; q += 10 * N;
        CK(cudaMemcpyAsync(q, final_states, rows * 10, cudaMemcpyHostToDevice, s)); d_fin = q; q += 10 * N;
        CK(cudaMemcpyAsync(q, masses, rows * 2, cudaMemcpyHostToDevice, s)); d_m = q; q += 2 * N;
        if (times) { CK(cudaMemcpyAsync(q, times, rows, cudaMemcpyHostToDevice, s)); d_t = q; }
    }
    // 1. selection (sorted index list + count)
    const size_t tb = pn_check_select_temp_bytes(N);
    if ((rc = c.ck_idx.ensure(sizeof(long long) * ((size_t)N + 1))) != PN_OK) return rc;
    if ((rc = c.ck_tmp.ensure(tb)) != PN_OK) return rc;
    long long* d_idx = (long long*)c.ck_idx.p;
    long long* d_cnt = d_idx + N;
    CK(pn_launch_check_select(N, fraction, key[0], key[1], d_idx, d_cnt, c.ck_tmp.p, s));
    long long m = 0;
    CK(cudaMemcpyAsync(&m, d_cnt, sizeof m, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    out->n_checked = m;
    if (checked_indices && m > 0) {
        if (m > max_indices) return PN_EINVAL;
        CK(cudaMemcpyAsync(checked_indices, d_idx, sizeof(long long) * (size_t)m,
                           o.host_buffers ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, s));
    }
    if (m == 0) { CK(cudaStreamSynchronize(s)); return PN_OK; }
    // 2. gather + FP64 reference integration of the subset (the library's own integrator)
    if ((rc = c.ck_sub.ensure(sizeof(double) * 23 * (size_t)m + sizeof(int) * (size_t)m)) != PN_OK) return rc;
    double* sub_init = (double*)c.ck_sub.p;
    double* sub_fin = sub_init + 10 * m;
    double* sub_m = sub_fin + 10 * m;
    double* sub_t = sub_m + 2 * m;
    int* sub_steps = (int*)(sub_t + m);
    CK(pn_launch_check_gather(d_idx, m, d_init, d_m, sub_init, sub_m, s));
    pn_options ro;
    default_options(&ro);
    ro.stream = o.stream;
    ro.out_time = sub_t;
    const int st = pn_integrate_ex(sub_init, sub_m, m, 0.0, omegaf, rtol_ref, atol_ref, PN_FP64, sub_fin, sub_steps, &ro);
    if (st == PN_ECUDA) return st;
    out->ms_reference = g_ms[1];
    // 3. comparison
    if ((rc = c.ck_out.ensure(64)) != PN_OK) return rc;
    CK(pn_launch_check_compare(d_idx, m, d_fin, d_t, sub_fin, sub_t, sub_steps, (double*)c.ck_out.p, s));
    double h[8];
    CK(cudaMemcpyAsync(h, c.ck_out.p, sizeof h, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    CK(cudaGetLastError());
    long long hi[8];
    memcpy(hi, h, sizeof hi);
    for (int k = 0; k < 3; ++k) { out->max_dot_dev[k] = h[k]; out->worst_index[k] = hi[4 + k]; }
    out->max_time_rel_dev = h[3];
    out->n_failed_ref = hi[7];
    return st;
}

extern "C" int pn_stream_status(void* stream)
{
    cudaStream_t s = (cudaStream_t)stream;
    CK(cudaStreamSynchronize(s));
    CK(cudaGetLastError());
    int st = PN_OK;
    auto it = g_ctx.find(CtxKey(current_device(), stream));
    if (it != g_ctx.end() && it->second->async_pending) {
        Ctx& c = *it->second;
        Small hs;
        CK(cudaMemcpy(&st, c.sticky.p, sizeof st, cudaMemcpyDeviceToHost));      // worst status since the last collection
        CK(cudaMemcpy(&hs, c.small.p, sizeof hs, cudaMemcpyDeviceToHost));       // counters of the LAST call on the stream
        memcpy(g_counters, hs.counters, sizeof g_counters);
        g_redo_count = hs.redo_count;
        c.async_pending = false;
    }
    return st;
}

extern "C" int pn_measure_fma_peak(int precision, double seconds, double* tflops, double* sm_mhz)
{
    if (!tflops || (precision != PN_FP64 && precision != PN_FP32 && precision != 3)) return PN_EINVAL;
    CK(pn_run_fma_peak(precision, 0, seconds, tflops, sm_mhz, nullptr));
    return PN_OK;
}

extern "C" int pn_measure_fma_operands(int precision, int n_register_sources, double* cycles_per_warp_inst)
{
    if (!cycles_per_warp_inst || n_register_sources < 1 || n_register_sources > 4 ||
        (precision != PN_FP64 && precision != PN_FP32))
        return PN_EINVAL;
    CK(pn_run_fma_peak(precision, n_register_sources - 1, 0.1, nullptr, nullptr, cycles_per_warp_inst));
    return PN_OK;
}

extern "C" int pn_last_counters(unsigned long long* trial_steps, unsigned long long* rejected,
                                unsigned long long* landing_trials, unsigned long long* failed)
{
    if (trial_steps) *trial_steps = g_counters[0];
    if (rejected) *rejected = g_counters[1];
    if (landing_trials) *landing_trials = g_counters[2];
    if (failed) *failed = g_counters[3];
    return PN_OK;
}

extern "C" unsigned long long pn_last_redo_count(void) { return g_redo_count; }

extern "C" int pn_last_kernel_ms(float ms[4])
{
    if (!ms) return PN_EINVAL;
    memcpy(ms, g_ms, sizeof g_ms);
    return PN_OK;
}

extern "C" unsigned long long pn_launch_count(void) { return g_pn_launches; }

extern "C" const char* pn_strerror(int st)
{
    switch (st) {
        case PN_OK: return "ok";
        case PN_EINVAL: return "invalid argument or input system";
        case PN_ECUDA: return "CUDA call or kernel launch failed";
        case PN_ENOTCONVERGED: return "a system hit max_steps, step-size underflow or failed to land on omega_f";
        case PN_ENONFINITE: return "a system produced a non-finite error norm";
        case PN_ETOOLARGE: return "request exceeds the fixed capacity of a no-allocation entry point (pn_statistics_static)";
        default: return "unknown status";
    }
}

extern "C" const char* pn_last_cuda_error(void) { return g_last_err.c_str(); }

extern "C" int pn_shutdown(void)
{
    int rc = PN_OK;
    if (cudaDeviceSynchronize() != cudaSuccess) rc = PN_ECUDA;
    for (auto& kv : g_ctx) if (free_ctx(kv.second) != PN_OK) rc = PN_ECUDA;
    g_ctx.clear();
    memset(g_slot_used, 0, sizeof g_slot_used);
    return rc;
}

extern "C" int pn_stream_release(void* stream)
{
    auto it = g_ctx.find(CtxKey(current_device(), stream));
    if (it == g_ctx.end()) return PN_OK;
    CK(cudaStreamSynchronize((cudaStream_t)stream));
    Ctx* c = it->second;
    const int dev = it->first.first;
    if (c->slot >= 0 && dev >= 0 && dev < PN_MAX_DEVICES) g_slot_used[dev][c->slot] = false;
    g_ctx.erase(it);
    return free_ctx(c);
}

extern "C" int pn_version(void) { return PN_VERSION; }
