/*
 * pn.h -- C ABI of libpn_b200: batched integration of post-Newtonian precessing circular-inspiral
 * ODE systems on one NVIDIA B200 (sm_100a), after arXiv:0908.3889.
 *
 * What is computed (citations are lines of the paper text, PAPER.md, and sections of DESIGN.md):
 *   - every system has the 10 state variables  y = (omega, S1x,S1y,S1z, S2x,S2y,S2z, Lx,Ly,Lz)
 *      and two parameters (m1, m2); its right-hand side is Eq. (1) for omega
 *     (PAPER.md:45), Eq. (2) with Omega_i of Eq. (4) for the spins and
 *     Eq. (3) for L^, with the readings of DESIGN.md section 3;
 *   - each system is integrated in time from its initial state until omega = omega_f
 *      by an adaptive Dormand-Prince 5(4) stepper with per-system
 *     error control; the last step lands on omega_f to a relative tau (R12);
 *   - pn_histogram bins the unit-vector dot products S1^.S2^, S1^.L^, S2^.L^ of the final
 *     states.
 *
 * Conventions
 *   - Every function returns a pn_status.  Nothing throws.  Every CUDA call and kernel launch is
 *     checked (unchecked kernels fail silently).
 *   - Pointers are DEVICE pointers (cudaMalloc'ed, this process, current device) unless
 *     pn_options.host_buffers != 0, in which case ALL array arguments of that call are HOST
 *     pointers and the library stages them through its own device scratch (H2D before, D2H after).
 *   - The caller owns every buffer.  The library keeps a small cached device scratch (SoA staging
 *     arrays, work counter, status word) that pn_shutdown() frees.
 *   - Calls are synchronous: on return the outputs are complete (the stream has been synchronised).
 *     If pn_options.async != 0 and device pointers are used, the call only enqueues on
 *     pn_options.stream; pn_stream_status(stream) later returns the worst status of ALL async calls
 *     enqueued on that stream since the last pn_stream_status.  Any number of async calls may be in
 *     flight, on one stream or several: the library keeps one scratch context (staging arrays, work
 *     counters, status words) per stream, and calls on one stream are ordered by the stream.  The
 *     caller's own buffers must of course not be reused by a second call before the first has finished
 *     unless both calls are on the same stream.
 *   - N = 0 is a successful no-op.  Not thread-safe: one caller thread per process.
 */
#ifndef PN_B200_H
#define PN_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { PN_FP64 = 0, PN_FP32 = 1, PN_MIXED = 2 } pn_precision;

typedef enum {
    PN_OK = 0,
    PN_EINVAL = 1,         /* bad argument (N < 0, null pointer, rtol <= 0, bins < 1, omega_f <= omega_0, m_i <= 0) */
    PN_ECUDA = 2,          /* a CUDA call or launch failed; outputs unspecified; see pn_last_cuda_error() */
    PN_ENOTCONVERGED = 3,  /* some system hit max_steps, step-size underflow or failed to land on omega_f */
    PN_ENONFINITE = 4,     /* some system produced a non-finite error norm */
    PN_ETOOLARGE = 5       /* pn_statistics_static only: the request does not fit the fixed scratch array; nothing was done */
} pn_status;

/* Per-system failure codes, written to out_steps[i] (which is otherwise the positive trial-step count). */
#define PN_FAIL_MAXSTEPS   (-1)
#define PN_FAIL_HUNDERFLOW (-2)
#define PN_FAIL_NONFINITE  (-3)
#define PN_FAIL_LANDING    (-4)
#define PN_FAIL_BADINPUT   (-5)   /* m_i <= 0 or omega_0 >= omega_f for that system */

/*
 * pn_integrate -- adaptive DP5(4) integration of N independent systems to omega_f.
 *   init_states [N][10] row-major doubles, order (omega, S1, S2, L^).  Read only.
 *   masses      [N][2]  (m1, m2), any M = m1+m2 > 0 (the paper fixes M = 1).
 *   omega0      consistency check only (the state is authoritative): if > 0, every
 *               init_states[i][0] must equal it to 1e-12 relative, else PN_EINVAL.  <= 0: ignored.
 *   omegaf      termination frequency, must exceed every initial omega.
 *   rtol, atol  error control: a trial step is accepted when
 *               sqrt(mean_j (err_j / (atol*N_j + rtol*max(|y_j|,|ynew_j|)))^2) <= 1, with N_j = 1 for
 *               omega and L^, |S_i(0)| for the components of S_i (R6-R7).
 *   precision   PN_FP64: all arithmetic in double.  PN_FP32: state, slopes, RHS and error norm in
 *               float; time accumulation, step counters and all arrays of this interface in double.
 *               PN_MIXED: as PN_FP32, but the state is carried in double: an accepted step adds the float
 *               increment sum_s b_s K_s to it, and omega is compared with omega_f in double ("only a few
 *               critical computations in double").  Usable down to rtol ~ 1e-8.
 *   out_final   [N][10] final states (the omega slot holds the landed omega, within tau of omega_f).
 *   out_steps   [N] trial steps taken (accepted + rejected + discarded landing trials), or a
 *               negative PN_FAIL_* code.  RHS evaluations of a system = 6*steps + 1.
 * Returns PN_OK, or the worst status over all systems; the other systems still complete.
 */
int pn_integrate(const double* init_states, const double* masses, long long N,
                 double omega0, double omegaf, double rtol, double atol, int precision,
                 double* out_final, int* out_steps);

typedef struct pn_options {
    int size;              /* = sizeof(pn_options); checked */
    int fixed_steps;       /* > 0: fixed-step mode: exactly this many DP5 steps of size h0, no error
                              control, no omega_f stop (omegaf, rtol, atol ignored) */
    double h0;             /* first step (adaptive) or the step (fixed); <= 0: 10*M */
    int max_steps;         /* per system; <= 0: 10,000,000 */
    unsigned term_mask;    /* tests only.  bit k (0..7) keeps the (M omega)^{k/3} term of the brace of
                              Eq. (1); bit 16 keeps the spin terms of Eq. (1).  0: everything */
    double tau_land;       /* landing tolerance |omega - omega_f| <= tau*omega_f; <= 0: 1e-13 (FP64), 3e-7 (FP32), 1e-8 (MIXED) */
    int layout;            /* 0: AoS [N][10] / [N][2] as above.  1: SoA [10][N] / [2][N] for
                              init_states, masses and out_final (no staging pass) */
    int host_buffers;      /* != 0: every array argument is a HOST pointer (see Conventions) */
    int async;             /* != 0: enqueue only (device pointers only) */
    int input_order;       /* 0 (default): systems are issued to the work queue longest-expected-first
                              (cost model in DESIGN.md 7.5); != 0: in input order.  Results do not
                              depend on the order */
    double* out_time;      /* [N] or NULL: time t_f at which omega_f was reached */
    int* out_rejected;     /* [N] or NULL: rejected trial steps */
    void* stream;          /* cudaStream_t, or NULL for the default stream */
    int block_threads;     /* tuning: threads per block of the integrator (0: default) */
    int grid_blocks;       /* tuning: blocks of the persistent grid (0: SMs x resident blocks) */
    int variant;           /* tests / tuning: kernel selection bits, results are unchanged (FP64 bit 0: to rounding).  1: always
                              the generic kernel (per-lane constants) even for uniform-mass batches; 2: always the
                              scalar FP32 kernel instead of the packed two-systems-per-lane one; 4: pn_run_ensembles
                              orders the queue by cost even for more than 4 ensembles (measurement only: several times slower) */
    int hist_bins;         /* pn_integrate_ex only.  hist_counts != NULL: the call also bins the final states it has just
                              written, as pn_histogram(out_final, N, hist_bins, hist_counts, hist_skipped) would, while they
                              are still on the device: a host-buffer caller does not upload the 80 bytes per system again
                              (the state goes to the device once and comes back once).  1 <= hist_bins <= 2^24 */
    unsigned long long* hist_counts;   /* [3][hist_bins] or NULL (no histogram); host pointer iff host_buffers */
    unsigned long long* hist_skipped;  /* [3] or NULL */
} pn_options;

/* Same as pn_integrate with explicit options (opt == NULL: defaults). */
int pn_integrate_ex(const double* init_states, const double* masses, long long N,
                    double omega0, double omegaf, double rtol, double atol, int precision,
                    double* out_final, int* out_steps, const pn_options* opt);

/*
 * pn_histogram -- three histograms of the final configuration (R14).
 *   final_states [N][10] (device, or host with the _ex variant), as written by pn_integrate.
 *   bins         >= 1 equal-width bins over [-1, 1]; d = +1 falls in the last bin.
 *   counts       [3][bins] unsigned 64-bit, overwritten: rows are S1^.S2^, S1^.L^, S2^.L^, where
 *                A^.B^ = (A.B)/(|A||B|) with the norms taken from the state itself.
 *   n_skipped    [3] or NULL: systems left out of each histogram because a norm is zero or the
 *                quotient is not finite.
 */
int pn_histogram(const double* final_states, long long N, int bins,
                 unsigned long long* counts, unsigned long long* n_skipped);

/* As pn_histogram; layout/host_buffers/stream of opt are honoured (opt == NULL: defaults). */
int pn_histogram_ex(const double* final_states, long long N, int bins,
                    unsigned long long* counts, unsigned long long* n_skipped, const pn_options* opt);

/*
 * pn_statistics -- one pass over the (initial, final) states of an integrated batch: the ensemble
 * statistics of the paper's section V.  For each of the three unit dot
 * products d = S1^.S2^, S1^.L^, S2^.L^ (A^.B^ = (A.B)/(|A||B|), norms from the state itself), with
 * x = d(initial state) and y = d(final state) of every system of an ensemble:
 *   - the Pearson product-moment coefficient r = 1/(n-1) sum ((x-xbar)/sigma_x)((y-ybar)/sigma_y)
 *     (sigma = sample standard deviation, DESIGN.md 3 R18), NaN if n < 2 or a variance is 0;
 *   - the moments n, xbar, ybar, M2x = sum (x-xbar)^2, M2y, Cxy = sum (x-xbar)(y-ybar);
 *   - the histogram of y on bins1 equal bins of [-1,1] and the bivariate histogram of
 *     (x, y) on bins2 x bins2 equal cells (row = bin of x, column = bin of y), its largest
 *     count, and the histogram divided by that count ("normalized such that the maximum value is 1").
 * Ensembles ("groups"): group g is the contiguous range [g*group_size, (g+1)*group_size) of systems, so a
 * parameter sweep (Figs. 6-7) is one pn_integrate call and one pn_statistics call.
 * group_size <= 0 means one group of N systems; otherwise N must be a multiple of group_size.  G = N/group_size.
 * A system is left out of the statistics of a dot product (and counted in n_skipped) if either value is
 * undefined (zero norm, non-finite), and out of all three if steps != NULL and steps[i] < 0.
 *   init_states, final_states  [N][10] AoS doubles, 16-byte aligned (read with bulk copies).  Read only.
 *                              init_states == NULL: only hist1 and n_skipped (of the final states) are computed.
 *   steps                      [N] out_steps of pn_integrate, or NULL.
 *   out                        any member may be NULL (not computed); bins1 / bins2 < 1 disable hist1 / hist2*.
 * Bin rule on every axis: bin = clamp(floor((d+1) bins/2), 0, bins-1) (R14).
 * Results are bit-identical from run to run (no floating-point atomics).
 * opt: host_buffers, async and stream are honoured; layout must be 0.
 */
typedef struct pn_stats_out {
    int size;                       /* = sizeof(pn_stats_out); checked */
    double* pearson_r;              /* [G][3] */
    double* moments;                /* [G][3][6]: n, xbar, ybar, M2x, M2y, Cxy */
    unsigned long long* n_skipped;  /* [G][3] */
    unsigned long long* hist1;      /* [G][3][bins1] */
    unsigned long long* hist2;      /* [G][3][bins2][bins2] */
    unsigned long long* hist2_max;  /* [G][3]; needs hist2 */
    double* hist2_norm;             /* [G][3][bins2][bins2]; needs hist2 */
} pn_stats_out;

int pn_statistics(const double* init_states, const double* final_states, const int* steps, long long N,
                  long long group_size, int bins1, int bins2, const pn_stats_out* out,
                  const struct pn_options* opt);

/*
 * pn_merge_statistics -- the exchange step of pn_statistics over several GPUs: `parts` holds the
 * `moments` outputs of n_parts pn_statistics calls over disjoint parts of the SAME G ensembles, [n_parts][G][3][6]
 * (e.g. gathered from all ranks with one all-gather); they are merged in part order with the pairwise update used
 * inside a launch.  moments_out [G][3][6] and pearson_r_out [G][3] (either may be NULL).  Histogram counters need no
 * such call: they are summed by an integer all-reduce.  DEVICE pointers; opt: stream and async only.
 */
int pn_merge_statistics(const double* parts, int n_parts, int n_groups, double* moments_out, double* pearson_r_out,
                        const struct pn_options* opt);

/*
 * pn_statistics_static -- pn_statistics for callers that must not allocate device memory.
 *
 * Who needs it.  pn_statistics keeps its per-block moment records in scratch that the library obtains with cudaMalloc
 * the first time (and again whenever a call needs more).  Some programs that embed this library cannot afford, or are
 * not able, to do that at the moment they want the statistics:
 *   - a host framework (a PyTorch job, say) that has already handed the whole HBM to its own caching allocator, so a
 *     cudaMalloc from a library comes back with "out of memory" although the job has room to spare in its pool;
 *   - an analysis loop that runs next to other streams (the integrator of the next batch, a copy engine): cudaMalloc
 *     and cudaFree are device-wide synchronisation points, so one allocation stalls every one of those streams;
 *   - a process that lives under a fixed memory budget (an MPS or MIG slice with a limit) and has to know its
 *     footprint when it starts, not discover it call by call.
 * For them this entry point computes the same ensemble statistics (Pearson r of PAPER.md:138, the
 * histograms of PAPER.md:116-120 and 132) with the same kernels, launch geometry and merge order as pn_statistics, so
 * every output is the same number for number, but the kernels' scratch is a fixed array that is part of the library image
 * (`static __device__`, PN_STATIC_SCRATCH_BYTES = 344,064 bytes).  Every GPU on which the library is loaded carries
 * that array from the moment the module is loaded until the process exits, whether or not this function is ever called.
 * The call itself issues no cudaMalloc, cudaFree, event or stream creation and calls no library routine that allocates.
 *
 * Arguments are those of pn_statistics, with these differences:
 *   - DEVICE pointers only (a host-buffer variant would need staging memory, i.e. an allocation); inputs and outputs
 *     stay the caller's: nothing but the scratch comes from the library.
 *   - `stream` is the cudaStream_t to run on (NULL: the default stream); `async` != 0 only enqueues, otherwise the
 *     stream has been synchronised on return.
 *   - Limit: n_groups = N / group_size <= PN_STATIC_MAX_GROUPS (1024), and n_groups + (SMs of the device) + 1 records
 *     of 168 bytes must fit the array (they do for any device of up to 1023 SMs).  A call beyond that changes nothing
 *     and returns PN_ETOOLARGE ("request exceeds the fixed capacity of a no-allocation entry point"); the number of
 *     systems N is not limited by the array (a block's record does not grow with N).
 * Set-up: the first call on each device looks up the device address of the array (cudaGetSymbolAddress with that
 * device current; the array's name means nothing to host code) and opts the kernel in to its shared-memory size.  Make
 * that first call outside any stream capture, once per device you use; later calls do neither.
 * Sharing: all calls in the process use the one array per device.  The part a call uses is zeroed on the stream before
 * its kernels run, so nothing is inherited from the previous call; but two calls that can overlap on the GPU (different
 * streams without an ordering between them, or two host threads) race on it and corrupt each other's moments.  Calls
 * on one stream, or ordered by events, are safe.  pn_last_kernel_ms is not updated (timing needs events).
 */
#define PN_STATIC_MAX_GROUPS 1024
#define PN_STATIC_SCRATCH_BYTES 344064 /* 2048 records x 3 dot products x (6 doubles + 1 counter) */
int pn_statistics_static(const double* init_states, const double* final_states, const int* steps, long long N,
                         long long group_size, int bins1, int bins2, const pn_stats_out* out, void* stream, int async);

/*
 * pn_generate -- random initial data on the device ("generated on the GPU"; recipe of
 * PAPER.md:68, 102-104 as fixed in DESIGN.md 5 and 12): for every system seven uniform variates
 * (q, chi1, chi2, z1, phi1, z2, phi2) from ONE counter-based Philox4x64-10 stream per ensemble, laid out
 * like numpy.random.Philox: variate (k, i) = U(word (e mod 4) of Philox(counter = e/4 + 1, key)),
 * e = k*n_total + i, U(x) = (x >> 11) 2^-53.  q = m2/m1 uniform in [q_lo, q_hi] (q_lo if q_hi <= q_lo),
 * m1 = 1/(1+q), m2 = q/(1+q), or (m1_fixed, 1 - m1_fixed) if m1_fixed > 0; chi_i uniform in
 * [chi_i_lo, chi_i_hi]; unit spins (sqrt(1-z^2) cos phi, sqrt(1-z^2) sin phi, z), z = 2u - 1,
 * phi = 2 pi u' (uniform on the sphere), or S^_1 = (sin t, 0, cos t) if s1_tilt_deg = t >= 0;
 * S_i = chi_i m_i^2 S^_i; L^ = (0,0,1); omega = omega0.
 *   ens           HOST array of n_ensembles descriptions (a parameter sweep is several ensembles).
 *   n_total       systems per ensemble: fixes the layout of the variate stream.
 *   first, count  the chunk [first, first+count) of every ensemble to generate (first+count <= n_total);
 *                 chunks of one ensemble generated by separate calls (or GPUs) are identical to one big call.
 *   init_states   [n_ensembles*count][10], masses [n_ensembles*count][2], AoS, 16-byte aligned; ensemble e
 *                 occupies rows [e*count, (e+1)*count).  Device pointers (host with opt->host_buffers).
 * A system's state is a pure function of (key, n_total, index): results are bit-identical from run to run.
 */
typedef struct pn_ensemble {
    int size;                          /* = sizeof(pn_ensemble); checked */
    unsigned long long key[2];         /* Philox4x64 key */
    double omega0;
    double q_lo, q_hi;
    double m1_fixed;                   /* > 0: fixed masses (m1_fixed, 1 - m1_fixed); q_* then only consume their variate */
    double chi1_lo, chi1_hi, chi2_lo, chi2_hi;
    double s1_tilt_deg;                /* >= 0: S^_1 fixed in the x-z plane, tilted from L^ by this angle; < 0: isotropic */
} pn_ensemble;

int pn_generate(const pn_ensemble* ens, int n_ensembles, long long n_total, long long first, long long count,
                double* init_states, double* masses, const struct pn_options* opt);

/*
 * pn_run_ensembles -- seed in, statistics out: ONE fused launch sequence that draws the initial data (as pn_generate),
 * integrates every system to omegaf (as pn_integrate, PN_FP64) and reduces the ensemble statistics (as pn_statistics with
 * group_size = count), without any state array in device memory: the persistent integrator draws a system from the
 * counter-based Philox stream when a lane pulls work, and folds a finished system into the statistics instead of storing
 * it ("generated on the GPU", 104, 112-138).  The device memory a
 * run needs is independent of its size (the paper's 3.6e8-system run of PAPER.md:120 is one call).
 *   ens, n_ensembles, n_total, first, count   as in pn_generate: ensemble e contributes the systems
 *               [first, first+count) of its variate stream; every ens[e].omega0 must be below omegaf.
 *   omegaf, rtol, atol                        as in pn_integrate; precision must be PN_FP64.
 *   bins1, bins2, out                         as in pn_statistics with G = n_ensembles groups: pearson_r [G][3],
 *               moments [G][3][6], n_skipped [G][3] (undefined dot product, or the system failed), hist1 [G][3][bins1],
 *               hist2 [G][3][bins2][bins2], hist2_max, hist2_norm; any member may be NULL.  DEVICE pointers (host with
 *               opt->host_buffers).  bins1 <= 2^24, bins2 <= 4096.
 *   opt         h0, max_steps, term_mask, tau_land, input_order, host_buffers, async, stream, grid_blocks, variant bit 0 are honoured.
 *               A call whose ensembles ALL have the same fixed masses (one ensemble, or an equal-mass sweep over chi) runs
 *               the uniform-mass kernel, exactly when pn_integrate would for the concatenated batch; otherwise the generic one.
 * Results equal the chain pn_generate -> pn_integrate -> pn_statistics on the same arguments: n, n_skipped and every
 * histogram count exactly (and reproducibly); means, M2x, M2y, Cxy and r to rounding (the order in which partial moments
 * are merged depends on timing: r agrees to ~1e-13, not bit for bit).  For a call of at most 4 ensembles the queue of every
 * chunk of 2^22 systems is issued longest-expected-first like pn_integrate's (a draw-only pass writes the keys: 8 bytes of
 * scratch per system of a chunk; opt->input_order != 0: index order, no scratch).  A call of more ensembles is issued in
 * index order: cost order would interleave the ensembles and make the blocks' 4-entry moment tables thrash.
 * Returns the worst per-system status like pn_integrate; pn_last_counters / pn_last_kernel_ms()[1] refer to the run.
 */
int pn_run_ensembles(const pn_ensemble* ens, int n_ensembles, long long n_total, long long first, long long count,
                     double omegaf, double rtol, double atol, int precision, int bins1, int bins2,
                     const pn_stats_out* out, const struct pn_options* opt);

/*
 * pn_selfcheck -- the paper's cross-check ("a random ~1 % subset" evolved in double precision next to
 * the single-precision GPU run and compared afterwards), on the device.
 *   selection   system i is checked iff u_i < fraction, u_i = element i of the uniform stream of `key`
 *               (Philox4x64-10 in numpy.random.Philox's layout, as in pn_generate); expected subset size fraction*N.
 *   reference   the selected systems are re-integrated from init_states by pn_integrate in PN_FP64 at
 *               (rtol_ref, atol_ref) (<= 0: 1e-10, 1e-12) to omegaf.
 *   comparison  per unit dot product (S1^.S2^, S1^.L^, S2^.L^; norms from the states) the largest
 *               |d(final_states[i]) - d(reference)| over the subset and the lowest index where it occurs; the largest
 *               |times[i]/t_ref - 1| if times != NULL.  Systems whose reference failed are counted and left out.
 *   init_states, masses, final_states [N][10] / [N][2] / [N][10] AoS, times [N] or NULL: DEVICE pointers
 *               (host with opt->host_buffers).  out: HOST struct.  checked_indices: DEVICE (host with host_buffers)
 *               array of capacity >= max_indices receiving the sorted subset, or NULL.
 * Synchronous (opt->async is rejected).  Deterministic.  Returns the status of the reference integration.
 */
typedef struct pn_check_out {
    int size;                     /* = sizeof(pn_check_out); checked */
    long long n_checked;          /* size of the subset */
    long long n_failed_ref;       /* subset systems whose FP64 reference integration failed */
    double max_dot_dev[3];        /* worst absolute deviation per dot product (0 if nothing comparable) */
    long long worst_index[3];     /* system index of that deviation, -1 if none */
    double max_time_rel_dev;      /* worst relative deviation of the final time (0 without times) */
    float ms_reference;           /* duration of the reference integrator kernels, CUDA events */
} pn_check_out;

int pn_selfcheck(const double* init_states, const double* masses, const double* final_states, const double* times,
                 long long N, double omegaf, double fraction, const unsigned long long key[2], double rtol_ref,
                 double atol_ref, pn_check_out* out, long long* checked_indices, long long max_indices,
                 const struct pn_options* opt);

/* Worst pn_status of the async calls enqueued on `stream` since the last pn_stream_status (a later call never
 * erases an earlier call's status); synchronises the stream.  pn_last_counters() then refers to the last call
 * enqueued on that stream. */
int pn_stream_status(void* stream);

/*
 * pn_stream_release -- gives back what the library holds for `stream` on the current device: its scratch context
 * (device staging buffers, work counters, events, a pending async status, which is discarded) and its row of the
 * uniform-mass constant table.  Synchronises the stream first.  Call it before destroying a stream the library has
 * been used on: contexts are keyed by (device, stream handle), the runtime may hand the same handle value to a later
 * stream, and that stream would otherwise inherit the old context (harmless for results, but with a stale pending
 * status); and every stream ever used would keep its buffers until pn_shutdown.
 * The table has 4 rows per device: the first 4 live (unreleased) streams of a device get one, further streams run the
 * generic FP64 kernel even on uniform-mass batches, which is slower by a few percent and rounds differently
 * (same step counts for ~98 % of systems, final states to ~1e-11).  A stream that was never used, or
 * was already released, is a successful no-op.
 */
int pn_stream_release(void* stream);

/*
 * pn_measure_fma_peak -- measured FMA throughput of this device at its current clocks: every thread
 * runs `chains` independent dependent-FMA chains (no memory traffic) for about `seconds`.
 * Writes achieved TFLOP/s (2 flops per FMA) and, if not NULL, the SM clock in MHz estimated from
 * clock64() over the run (the longest per-block span).  The denominator of the reported roofline fraction.
 * precision: PN_FP64, PN_FP32 (scalar FFMA), or 3 = FP32 with packed f32x2 FMAs (FFMA2, 4 flops per instruction and lane).
 */
int pn_measure_fma_peak(int precision, double seconds, double* tflops, double* sm_mhz);

/*
 * pn_measure_fma_operands -- issue cost of an FMA as a function of how many DISTINCT register sources it
 * reads (1, 2 or 3; the other operands are uniform): cycles per warp instruction per scheduler with 8 warps
 * x 8 independent chains resident.  Evidence for the operand-port model of DESIGN.md 7.2.
 * n_register_sources = 4 is the issue-overlap probe: a two-source FMA plus two independent integer instructions
 * (LOP3, IADD3) per group; the result is cycles per GROUP (2 if the integer instructions issue in the FMA's shadow,
 * 4 if every instruction takes its own issue cycles).
 */
int pn_measure_fma_operands(int precision, int n_register_sources, double* cycles_per_warp_inst);

/* Device-side counters of the last synchronous pn_integrate* call: total trial steps, rejected
 * steps, discarded landing trials, systems that failed.  Any pointer may be NULL. */
int pn_last_counters(unsigned long long* trial_steps, unsigned long long* rejected,
                     unsigned long long* landing_trials, unsigned long long* failed);

/* FP64 only: number of systems of the last synchronous pn_integrate* call that were re-integrated by the
 * wide-range redo pass because one of their steps changed omega by more than 3 %. */
unsigned long long pn_last_redo_count(void);

/* Duration in milliseconds of the kernels of the last synchronous pn_integrate* / pn_histogram* call,
 * measured with CUDA events on the call's stream: [0] stage-in, [1] integrator, [2] stage-out,
 * [3] histogram or statistics.  Entries a call did not run are left unchanged. */
int pn_last_kernel_ms(float ms[4]);

/* Number of kernel launches issued by this library since load (for bench.py's gpu_launches). */
unsigned long long pn_launch_count(void);

const char* pn_strerror(int status);
const char* pn_last_cuda_error(void);   /* text of the last failing CUDA call, "" if none */
int pn_shutdown(void);                  /* frees cached scratch; the library stays usable */
int pn_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PN_B200_H */
