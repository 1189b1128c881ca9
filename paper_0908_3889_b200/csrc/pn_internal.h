// pn_internal.h -- declarations shared by the translation units of libpn_b200 (host side only).
#pragma once
#include <cuda_runtime.h>

#define PN_ORDER_BUCKETS 2048
#define PN_UNI_SLOTS 4
#define PN_UNI_ROW 32
#define PN_FW 4                   /* fused mode: ensembles a block accumulates at a time (the block's moment table) */

// Arguments of the integrator kernels.  All arrays are DEVICE pointers in SoA layout with stride n:
// y0[c*n + i], masses[j*n + i], yf[c*n + i].
struct PnKernelParams {
    const double* y0;
    const double* masses;
    double* yf;
    int* steps;
    double* time;        // may be null
    int* rejected;       // may be null
    const int* order;    // may be null: queue position -> system index
    void* seed;          // [n][40] reals of the launch precision: per-system seed records (pn_integrate.cu)
    int n;
    double omega0;       // > 0: every initial omega must match it to 1e-12 relative
    double omegaf, rtol, atol, h0, tau;
    double emax;         // FP64 fast kernel: range of the cbrt/log series, |1 - x/x0| <= emax (pn_rhs.cuh)
    double qc[7];        // FP64 fast kernel: cl / k, the log series with its coefficient folded in (pn_host_series, pn_rhs.cuh)
    int max_steps;
    int fixed_steps;
    unsigned mask;
    unsigned int* queue;            // global work counter (zeroed before launch)
    unsigned int* queue2;           // work counter of the redo pass
    int* redo_list;                 // [n] systems handed to the redo pass (FP64 only)
    unsigned int* redo_count;
    unsigned long long* counters;   // [0] trial steps [1] rejected [2] landing trials [3] failed systems
    int* status;                    // worst pn_status seen on the device (atomicMax)
    int* nonuniform;                // set by the seed kernel if some system's masses differ from system 0's (or system 0 is bad)
    double* uni_row;                // [PN_UNI_ROW] written by the seed kernel: system 0's constants in the form the uniform-mass kernel reads
    int uni_slot;                   // FP64 uniform-mass path: slot of the __constant__ table that holds system 0's PnConsts; < 0: off
    float* keys;                    // [n] or null: expected-cost keys written by the seed kernel (queue ordering)
    unsigned int* order_scratch;    // [PN_ORDER_BUCKETS + 2]: bucket cursors, then the bit patterns of the smallest / largest key
    int* order_out;                 // [n]: the queue order the bucket sort writes (= order when keys != null)
    int rec_pairs;                  // FP32 seed records with y0 and K1 in the pair order of the pair-packed kernel (pn_rhs.cuh)
    // ---- fused ensemble mode (pn_run_ensembles): seed in, statistics out, no state arrays ----
    // queue position q of this launch <-> system g = f_base + q of the run; ensemble e = g / f_count, index inside the
    // ensemble's variate stream j = f_first + g % f_count.  y0, masses, yf, steps, time, rejected, seed are unused.
    const void* f_specs;            // device array of GenSpec (pn_gen.cuh), one per ensemble; null: not a fused launch
    long long f_n_total, f_first, f_count, f_base;
    double* f_mom;                  // [G][3][6] running moments n, xbar, ybar, M2x, M2y, Cxy (merged under f_lock[g])
    int* f_lock;                    // [G] spin locks, zero-initialised
    unsigned long long* f_skipped;  // [G][3]
    unsigned long long* f_hist1;    // [G][3][bins1] or null
    unsigned long long* f_hist2;    // [G][3][bins2][bins2] or null
    int f_bins1, f_bins2;
    unsigned f_resident;            // lanes of the persistent grid (grid x block): the length of the queue's last wave
};

// cl / k, k = 1 ... 7, for PnKernelParams::qc: cl = -(856/105)(2/3) is the coefficient of ln(M omega) in the v^6 term of
// Eq. (1) (pn_rhs.cuh: pn_make_uni; term_mask bit 6 switches the 3PN term off, mask 0 means all terms)
static inline void pn_host_series(unsigned mask, double (&qc)[7])
{
    const bool on = mask == 0 || ((mask >> 6) & 1u);
    const double cl = on ? -(856.0 / 105.0) * (2.0 / 3.0) : 0.0;
    for (int k = 0; k < 7; ++k) qc[k] = cl / (double)(k + 1);
}

// launchers (pn_integrate.cu); block_threads / grid_blocks = 0 choose the defaults
// variant bits (pn_options.variant): 1 = always the generic FP64 kernel (per-lane constants), 2 = always the scalar FP32 kernel
cudaError_t pn_launch_integrate(PnKernelParams& p, int precision, int block_threads, int grid_blocks,
                                cudaStream_t s, int variant);
// fused ensemble run (pn_integrate.cu): one chunk of systems [p.f_base, p.f_base + p.n); fast kernel + redo pass;
// uni_slot >= 0: all of them in the fixed-mass ensemble uni_ens -> the uniform-mass fast kernel with table row uni_slot
cudaError_t pn_launch_fused(PnKernelParams& p, int grid_blocks, cudaStream_t s, int uni_slot, int uni_ens);
// pair-packed FP32 integrator (pn_integrate_packed.cu); the seed records must be float ones written with rec_pairs = 1
cudaError_t pn_launch_integrate_packed(PnKernelParams& p, int grid_blocks, cudaStream_t s, int uni_slot);
// staging + histogram + peak (pn_aux.cu)
cudaError_t pn_launch_aos_to_soa(const double* aos, double* soa, int n, int width, cudaStream_t s);
cudaError_t pn_launch_soa_to_aos(const double* soa, double* aos, int n, int width, cudaStream_t s);
cudaError_t pn_launch_histogram(const double* states, int layout_soa, long long n, int bins,
                                unsigned long long* counts /*[3][bins]*/, unsigned long long* skipped /*[3]*/,
                                cudaStream_t s);
// queue order, longest expected first (pn_aux.cu): bucket sort of the keys the seed kernel wrote.
// scratch: PN_ORDER_BUCKETS + 2 unsigned: bucket cursors (0), then min / max key bits (0xffffffff / 0), set by the init call
// async calls: *sticky = max(*sticky, *status), one thread (pn_api.cu folds a call's status into its stream's sticky word)
cudaError_t pn_launch_fold_status(const int* status, int* sticky, cudaStream_t s);
cudaError_t pn_launch_order_init(unsigned int* scratch, cudaStream_t s);
// n_flat > 0: a batch of >= n_flat systems whose keys span less than a factor 2 stays in (block-wise) input order
cudaError_t pn_launch_cost_order(const float* keys, int n, unsigned int* scratch, int* order, cudaStream_t s, int n_flat);
// ensemble statistics (pn_stats.cu)
size_t pn_stats_scratch_bytes(long long n, long long group_size, int* n_blocks_out);
cudaError_t pn_launch_stats_merge(const double* parts, int n_parts, int n_groups, double* mom_out, double* r_out, cudaStream_t s);
cudaError_t pn_launch_stats_norm(const unsigned long long* hist2, long long n_hists, int cells, unsigned long long* max_out,
                                 double* norm_out, cudaStream_t s);
cudaError_t pn_launch_stats(const double* init, const double* fin, const int* steps, long long n, long long group_size,
                            int bins1, int bins2, void* scratch, double* r_out, double* mom_out,
                            unsigned long long* skipped_out, unsigned long long* hist1, unsigned long long* hist2,
                            unsigned long long* hist2_max, double* hist2_norm, cudaStream_t s);
// on-device initial data (pn_gen.cu); specs_dev: n_ens packed {u64 key0, key1; double omega0, q_lo, q_hi, m1_fixed,
// chi1_lo, chi1_hi, chi2_lo, chi2_hi, s1_tilt_deg}
cudaError_t pn_launch_generate(const void* specs_dev, int n_ens, long long n_total, long long first, long long count,
                               double* init_states, double* masses, cudaStream_t s);
// cross-check (pn_check.cu)
size_t pn_check_select_temp_bytes(long long n);
cudaError_t pn_launch_check_select(long long n, double fraction, unsigned long long k0, unsigned long long k1,
                                   long long* indices, long long* n_selected, void* temp, cudaStream_t s);
cudaError_t pn_launch_check_gather(const long long* indices, long long m, const double* init, const double* masses,
                                   double* sub_init, double* sub_masses, cudaStream_t s);
cudaError_t pn_launch_check_compare(const long long* indices, long long m, const double* fin, const double* times,
                                    const double* ref_fin, const double* ref_times, const int* ref_steps, double* out,
                                    cudaStream_t s);
cudaError_t pn_run_fma_peak(int precision, int mode, double seconds, double* tflops, double* sm_mhz,
                            double* cycles_per_warp_inst);

extern unsigned long long g_pn_launches;
// records "<where> -> <CUDA error string>" as the text pn_last_cuda_error() returns (pn_api.cu); for entry points that live
// in another translation unit
void pn_note_cuda_error(const char* where, cudaError_t e);
