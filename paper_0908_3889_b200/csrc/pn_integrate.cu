// pn_integrate.cu -- persistent-grid adaptive Dormand-Prince 5(4) integrator for sm_100a.
//
// One inspiral per lane.  Every warp iteration is one DP5 trial step executed by all 32 lanes in
// lock-step (accept / reject / landing are per-lane selects, not branches around the RHS); a lane
// whose inspiral has reached omega_f stores its result and immediately pulls the next system off a
// global atomic work queue (warp-aggregated atomicAdd), so adaptive-step and termination divergence
// cost only the short refill section.  All state (y, k1..k7, per-system constants) lives in
// registers; global memory is touched only at refill and at finish.  (DESIGN.md 2, 7.)
#include "pn_step_common.cuh"
#include "pn_dots.cuh"
#include "pn_gen.cuh"
#include "pn_moments.cuh"

// E^2 of the scaled RMS error norm, returned in FP32 (see the call site).
__device__ __forceinline__ float pn_err_norm2(const double (&y)[10], const double (&ynew)[10], const double (&err)[10],
                                              float rtol, float atol1, float atS1, float atS2)
{
    const double rt = (double)rtol;
    double sum = 0.0, sum1 = 0.0;          // two accumulators: the ten dependent FMAs were a 10-deep chain at the end of a step
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        const double at = (double)((i >= 1 && i <= 3) ? atS1 : ((i >= 4 && i <= 6) ? atS2 : atol1));
        // larger magnitude to ~1e-6: the high words of two doubles order like floats of the same bit patterns (sign,
        // then exponent, then mantissa), so ONE FMNMX with |.| modifiers picks the larger high word; the low word is
        // dropped (the scale is then low by < 2^-20, the accuracy class of the MUFU reciprocal below).  A zero or tiny
        // component (|y| < 2^-1015) reads as a float denormal or zero and stays that.
        const float mh = fmaxf(fabsf(__int_as_float(__double2hiint(y[i]))), fabsf(__int_as_float(__double2hiint(ynew[i]))));
        const double m = __hiloint2double(__float_as_int(mh), 0);
        const double sc = fma(rt, m, at);
        double r;
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(sc));
        const double q = err[i] * r;
        if (i & 1) sum1 = fma(q, q, sum1); else sum = fma(q, q, sum);
    }
    return (float)((sum + sum1) * 0.1);
}
__device__ __forceinline__ float pn_err_norm2(const float (&y)[10], const float (&ynew)[10], const float (&err)[10],
                                              float rtol, float atol1, float atS1, float atS2)
{
    float sum = 0.0f;
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        const float at = (i >= 1 && i <= 3) ? atS1 : ((i >= 4 && i <= 6) ? atS2 : atol1);
        const float scl = fmaf(rtol, fmaxf(fabsf(y[i]), fabsf(ynew[i])), at);      // at >= 1e-30 (clamped at refill): never 0
        const float q = err[i] * pn_rcp_f(scl);
        sum = fmaf(q, q, sum);
    }
    return sum * 0.1f;
}

// ---- per-system seed records (stage-in, row a1/a2 of the scope table) ------------------------------------
// Everything a lane needs to start an inspiral is computed ONCE per system by a plain one-thread-per-system
// kernel at full lane efficiency, instead of inside the divergent refill section of the persistent kernel
// (where one lane works and 31 wait): the per-system constants (~10 FP64 divides), the base powers
// (rcbrt + log), the scaled seed slope K1 = h0 f(y0) and the norm-scaled atol.  One contiguous record of
// PN_REC reals per system (FP64 320 B, FP32 160 B), so a lane's refill is 20 (10) 16-byte loads.
//   [0..9] y0   [10..19] K1 = h0 f(y0)   [20..34] PnConsts   [35..37] PnBase (r0, r0^3, k6b)   [38] atol |S1|   [39] atol |S2|
// A record with [38] < 0 marks a system the seed kernel has already failed (bad input).
// The seed record of one valid system: constants, base powers, K1 = h0 f(y0), norm-scaled atol (layout above).
template <typename real>
__device__ __forceinline__ void pn_make_record(const double (&y0)[10], double m1, double m2, const PnKernelParams& p, real (&out)[PN_REC])
{
    real y[10], k1[10];
#pragma unroll
    for (int j = 0; j < 10; ++j) y[j] = (real)y0[j];
    PnConsts<real> c;
    PnBase<real> base;
    PnUni<real> u;
    pn_make_uni<real>(p.mask, u);
    u.emax = (real)p.emax;
    pn_make_consts<real>(m1, m2, p.mask, c);
    pn_base_init(c.M * y[0], c.c6, u.cl, base);
    const real h = p.h0 > 0.0 ? (real)p.h0 : (real)10 * c.M;      // first step (R13); same expression at refill
    real r_tmp, l_tmp;
    PnFlag bad_tmp;
    PnScaled<real> sc;
    pn_make_scaled(c, h, sc);
    pn_rhs<true>(y, c, u, sc, base, k1, r_tmp, l_tmp, bad_tmp);      // K1 = h0 f(y0)
    // atol scaled by the conserved spin norms (R7)
    const double s1 = sqrt(y0[1] * y0[1] + y0[2] * y0[2] + y0[3] * y0[3]);
    const double s2 = sqrt(y0[4] * y0[4] + y0[5] * y0[5] + y0[6] * y0[6]);
#pragma unroll
    for (int j = 0; j < 10; ++j) {
        // rec_pairs: the pair-packed FP32 kernel wants each register pair as two adjacent, 8-byte aligned words
        const int pos = p.rec_pairs ? 2 * PN_PAIR_OF[j] + PN_PAIR_HALF[j] : j;
        out[pos] = y[j]; out[10 + pos] = k1[j];
    }
    out[20] = c.M; out[21] = c.c2; out[22] = c.c4; out[23] = c.c5; out[24] = c.c6; out[25] = c.c7;
    out[26] = c.p1; out[27] = c.p2; out[28] = c.q1; out[29] = c.q2; out[30] = c.K0; out[31] = c.A1;
    out[32] = c.A2; out[33] = c.Bc; out[34] = c.G;
    out[35] = base.r0; out[36] = base.r03; out[37] = base.k6b;
    out[38] = (real)(p.atol * (s1 > 0.0 ? s1 : 1.0));
    out[39] = (real)(p.atol * (s2 > 0.0 ? s2 : 1.0));
}

// The uniform-mass kernel's constants, in the form it evaluates the brace of Eq. (1) in: everything the
// brace is linear in arrives multiplied by KB = K0/Bc (pn_rhs.cuh, FOLD), so omega_dot = (beta v^5) brace'
//   [0..14] PnConsts (c2 ... c7, p1, p2, q1, q2 folded)   [15] c0'   [16] c3'   [17] cl'   [18..24] qc'   [25] KB
__device__ __forceinline__ void pn_write_uni_row(double m1, double m2, const PnKernelParams& p, double* row)
{
    PnConsts<double> c;
    PnUni<double> u;
    pn_make_uni<double>(p.mask, u);
    pn_make_consts<double>(m1, m2, p.mask, c);
    const double KB = c.K0 / c.Bc;
    row[0] = c.M; row[1] = KB * c.c2; row[2] = KB * c.c4; row[3] = KB * c.c5; row[4] = KB * c.c6; row[5] = KB * c.c7;
    row[6] = KB * c.p1; row[7] = KB * c.p2; row[8] = KB * c.q1; row[9] = KB * c.q2; row[10] = c.K0; row[11] = c.A1;
    row[12] = c.A2; row[13] = c.Bc; row[14] = c.G; row[15] = KB * u.c0; row[16] = KB * u.c3; row[17] = KB * u.cl;
#pragma unroll
    for (int k = 0; k < 7; ++k) row[18 + k] = KB * p.qc[k];
    row[25] = KB;
}

// Expected cost of a system: the number of precession cycles of the faster-precessing body,
//   key = (4 + 3 m_big/m_small)/eta (1/(M omega_0) - 1/(M omega_f))      (Eq. (4) over Eq. (1) at leading order),
// times a spin correction: the precession rate goes with |J| ~ |L| + (S1 + S2).L^, |L| = eta M^{5/3} omega^{-1/3}; integrated
// over the inspiral (dt = d omega / omega_dot, omega_dot ~ omega^{11/3}) the spin part is
// (3/2) S_par (omega_0^{-2/3} - omega_f^{-2/3}) / (eta M^{5/3}) next to 1/omega_0 - 1/omega_f.  Taken at half weight
// (measured step counts follow it with a slope of 0.44 on C2) and clamped: the order only needs to be approximate.
// The bucket sort that follows issues the queue longest-expected-first.  Positive floats order like their bit patterns, so
// the range of the keys is found with integer atomics: one pair per warp.  Bad inputs get key 0 (last in the queue; the
// refill skips them) and stay out of the range.  Called by whole warps (`in`: the thread has a system).
__device__ __forceinline__ void pn_write_cost_key(const PnKernelParams& p, int i, bool in, bool bad_input, const double (&y0)[10],
                                                  double m1, double m2)
{
    // single precision is ample for a sort key (and the seed kernel of an FP32 batch of 2^22 systems would otherwise spend
    // more time on double-precision divides and cube roots here than on its records)
    const float a = (float)m1, b = (float)m2, w0 = (float)y0[0], wf = (float)p.omegaf;
    const float M = a + b, eta = a * b / (M * M), dinv = 1.0f / w0 - 1.0f / wf;
    float key = (4.0f + 3.0f * fmaxf(a, b) / fminf(a, b)) / eta * dinv / M;
    const float s_par = (float)((y0[1] + y0[4]) * y0[7] + (y0[2] + y0[5]) * y0[8] + (y0[3] + y0[6]) * y0[9]);
    const float r0 = rcbrtf(w0), rf = rcbrtf(wf);
    const float rel = 1.5f * (r0 * r0 - rf * rf) / (eta * M * cbrtf(M * M) * dinv);
    key *= fmaxf(1.0f + 0.5f * s_par * rel, 0.3f);
    const bool key_ok = !bad_input && key > 0.0f && key < 3e38f;
    const float kf = key_ok ? key : 0.0f;
    if (in) p.keys[i] = kf;
    const unsigned kb = __float_as_uint(kf);
    const unsigned lo = __reduce_min_sync(0xffffffffu, key_ok ? kb : 0xffffffffu);
    const unsigned hi = __reduce_max_sync(0xffffffffu, key_ok ? kb : 0u);
    if ((threadIdx.x & 31) == 0) {
        // only a warp that widens the range issues the atomic (2^17 warps hammering two addresses cost 0.2 ms at 2^22 systems)
        volatile unsigned* rng = p.order_scratch + PN_ORDER_BUCKETS;
        if (lo < rng[0]) atomicMin(p.order_scratch + PN_ORDER_BUCKETS, lo);
        if (hi > rng[1]) atomicMax(p.order_scratch + PN_ORDER_BUCKETS + 1, hi);
    }
}

// fused mode: the expected-cost keys of the chunk's systems, drawn exactly as the integrator will draw them (pn_gen.cuh)
__global__ void __launch_bounds__(128) pn_fused_keys_kernel(const PnKernelParams p)
{
    const int i = blockIdx.x * 128 + threadIdx.x;
    const bool in = i < p.n;
    const long long gsys = p.f_base + (in ? i : p.n - 1);
    const long long e = gsys / p.f_count;
    const GenSpec sp = ((const GenSpec*)p.f_specs)[e];
    double y0[10], m1, m2;
    gen_system_at(sp, (unsigned long long)p.f_n_total, (unsigned long long)(p.f_first + (gsys - e * p.f_count)), y0, m1, m2);
    const bool bad_input = !(m1 > 0.0) || !(m2 > 0.0) || !(y0[0] < p.omegaf) || !(y0[0] > 0.0);
    pn_write_cost_key(p, i, in, bad_input, y0, m1, m2);
}

// fused mode, one fixed-mass ensemble: the row from the masses pn_gen.cuh gives every system of ensemble e (one thread)
__global__ void pn_fused_row_kernel(const PnKernelParams p, int e)
{
    const GenSpec sp = ((const GenSpec*)p.f_specs)[e];
    double m1, m2;
    if (sp.m1_fixed > 0.0) { m1 = sp.m1_fixed; m2 = __dsub_rn(1.0, m1); }
    else { const double d = __dadd_rn(1.0, sp.q_lo); m1 = __ddiv_rn(1.0, d); m2 = __ddiv_rn(sp.q_lo, d); }
    pn_write_uni_row(m1, m2, p, p.uni_row);
}

template <typename real>
__global__ void __launch_bounds__(128) pn_seed_kernel(const PnKernelParams p)
{
    const int i = blockIdx.x * 128 + threadIdx.x;
    const bool in = i < p.n;
    const int ii = in ? i : p.n - 1;            // out-of-range threads shadow the last system up to the key reduction
    double y0[10];
#pragma unroll
    for (int j = 0; j < 10; ++j) y0[j] = p.y0[(size_t)j * p.n + ii];
    const double m1 = p.masses[ii], m2 = p.masses[(size_t)p.n + ii];
    const bool bad_input = !(m1 > 0.0) || !(m2 > 0.0) || !(y0[0] < p.omegaf) || !(y0[0] > 0.0) ||
                           (p.omega0 > 0.0 && !(fabs(y0[0] - p.omega0) <= 1e-12 * p.omega0));
    if (p.keys) pn_write_cost_key(p, i, in, bad_input, y0, m1, m2);
    if (!in) return;
    real* rec = (real*)p.seed + (size_t)i * PN_REC;
    real y[10], k1[10];
#pragma unroll
    for (int j = 0; j < 10; ++j) y[j] = (real)y0[j];
    if (bad_input) {
        pn_store_result(p, i, y, PN_F_BADINPUT, 0.0, 0);
        atomicMax(p.status, PN_ST_EINVAL);
        atomicAdd(p.counters + 3, 1ull);
        rec[38] = (real)-1;
        if (i == 0) *p.nonuniform = 1;          // the uniform-mass kernel takes its constants from system 0's record
        return;
    }
    if (m1 != p.masses[0] || m2 != p.masses[p.n]) *p.nonuniform = 1;      // benign race: every writer stores 1
    real out[PN_REC];
    pn_make_record<real>(y0, m1, m2, p, out);
    if (i == 0 && p.uni_slot >= 0) {
        if (sizeof(real) == 8) pn_write_uni_row(m1, m2, p, p.uni_row);
        else {                                   // FP32: the record's own constants, as floats (pn_integrate_packed.cu)
            float* row = (float*)p.uni_row;
#pragma unroll
            for (int k = 0; k < 15; ++k) row[k] = (float)out[20 + k];
        }
    }
    using vec = typename PnVec<real>::type;           // 16-byte stores
    vec* dst = (vec*)rec;
    constexpr int W = 16 / (int)sizeof(real);
#pragma unroll
    for (int j = 0; j < PN_REC / W; ++j) dst[j] = PnVec<real>::make(&out[j * W]);
}

// SLOW = true: the redo pass.  Systems whose step left the range of the cbrt/log series in the fast kernel
// are re-integrated from their initial state with the wide-range evaluation (pn_rhs.cuh) in every stage.
// MIXED = true (real = float only; PN_MIXED): slopes, RHS, stage sums and error norm in float, but the
// state itself is carried in double: an accepted step adds the float increment dy = sum b_s K_s to the double copy,
// so the per-step rounding error is eps32 |dy| instead of eps32 |y| ("only a few critical computations in
// double"); omega is compared with omega_f in double.
// UNI >= 0 (FP64): every system of the batch has the masses of system 0 (checked by the seed kernel), so the 15
// mass-dependent constants come from row UNI of a __constant__ table (uniform-register operands instead of per-lane
// registers; the row must be a compile-time constant for that, a run-time row index makes ptxas load the values into
// per-lane registers again, so there is one instantiation per row and one row per stream context, PN_UNI_SLOTS in all).
// The launcher copies system 0's record into the row on the stream and launches BOTH the uniform-mass and the generic
// kernel (p.uni_slot >= 0 marks such a pair); each looks at the seed kernel's verdict and the one that does not apply
// returns at once, so no host synchronisation is needed and async calls keep the fast path.
__constant__ double pn_uni_table[PN_UNI_SLOTS][PN_UNI_ROW];

// ---- fused ensemble mode (FUSED = true; pn_run_ensembles): seed in, statistics out ----------------
// The work pull DRAWS the system (counter-based Philox + sphere sampling, pn_gen.cuh: the same bits as pn_generate)
// instead of loading it, and a finished system is folded into the ensemble statistics instead of being stored, so the
// launch reads and writes no state arrays at all.  To keep the draw off the divergent path (one lane working, 31
// waiting: ~2000 instructions for the Philox blocks, the two sincos, the per-system constants and the seed slope),
// a warp draws 32 systems AT ONCE, one per lane, into a shared-memory ring ([word][slot], conflict-free), and lanes
// whose inspiral has finished pop records off the ring; the global queue counter is advanced by 32 per draw.
// Statistics, three levels.  (1) Every THREAD keeps Welford moments (n, xbar, ybar, M2x, M2y, Cxy) per dot product in
// its own shared-memory words, for one ensemble at a time: a finished system is added without any lock.  (In index order a
// thread's ensembles only grow; in cost order they alternate, which is why pn_run_ensembles orders the queue by cost only
// for calls of at most PN_FW ensembles, pn_api.cu.)  (2) When its ensemble changes, and at kernel exit, a thread merges
// them (pairwise update) into the BLOCK's table of PN_FW ensembles under a shared-memory spin lock.  (3) A table entry
// that has to make room, and every entry when the last thread of the block leaves, is merged into the ensemble's
// global record under a per-ensemble global spin lock: a few hundred uncontended merges per ensemble.  (Tried before:
// threads merging straight into the global record -- 38 K threads taking one lock at kernel exit took 8.7 s; and every
// finished system added to the block's table under the lock -- at ~170 steps per inspiral the ~3000-cycle critical
// section was longer than the time between two finishes of a block, and the run took 43 % longer than the unfused one.)
// All locks are try-lock loops, safe under intra-warp contention.  Histogram counts go straight to global memory with
// integer atomics (one per finished system and dot product).  Counts are exact and reproducible; moments are
// reproducible to rounding (the merge order depends on timing).
#define PN_FREC (PN_REC + 4)      /* ring record: seed record + the three initial unit dot products (+ pad) */
#define PN_FDONE 13               /* done-ring record: 9 final components (S1, S2, L^), 3 initial dot products, {index, code} */
template <int BLOCK> struct PnFusedSmem {
    // one base pointer; every array is at a compile-time offset (seven stored pointers would cost 14 registers in a
    // kernel that has none to spare)
    static constexpr int NW = BLOCK / 32;
    static constexpr size_t O_XIN = (size_t)NW * PN_FREC * 32, O_ACC = O_XIN + 3 * BLOCK, O_MOM = O_ACC + 18 * BLOCK,
                            O_DONE = O_MOM + PN_FW * 18, N_DBL = O_DONE + (size_t)NW * PN_FDONE * 32;
    static constexpr size_t bytes() { return sizeof(double) * N_DBL + sizeof(int) * (NW * 32 + BLOCK + PN_FW + 4 + NW * 4); }
    unsigned char* base;
    __device__ explicit PnFusedSmem(unsigned char* b) : base(b) {}
    __device__ __forceinline__ double* ring() const { return reinterpret_cast<double*>(base); }                 // [NW][PN_FREC][32]
    __device__ __forceinline__ double* xin() const { return ring() + O_XIN; }    // [3][BLOCK] initial unit dot products of the lane's system (NaN: undefined)
    __device__ __forceinline__ double* acc() const { return ring() + O_ACC; }    // [3][6][BLOCK] every thread's own moments (no lock), ONE ensemble at a time
    __device__ __forceinline__ double* mom() const { return ring() + O_MOM; }    // [PN_FW][3][6] the block's moments
    __device__ __forceinline__ double* done() const { return ring() + O_DONE; }  // [NW][PN_FDONE][32] finished systems waiting for the warp's next batch
    __device__ __forceinline__ int* ring_idx() const { return reinterpret_cast<int*>(ring() + N_DBL); }        // [NW][32]
    __device__ __forceinline__ int* acc_g() const { return ring_idx() + NW * 32; }   // [BLOCK] ensemble of the thread's moments, -1: none
    __device__ __forceinline__ int* tag() const { return acc_g() + BLOCK; }          // [PN_FW] ensemble of each table entry, -1: free
    __device__ __forceinline__ int* lock() const { return tag() + PN_FW; }           // [0] table lock; [1] threads that have left the main loop
    // per warp, warp-uniform, touched only in the refill / finish sections (so they live here, not in registers):
    // [0] records popped off the ring, [1] records drawn into it, [2] finished systems parked in the done ring
    __device__ __forceinline__ volatile int* wstate() const { return lock() + 4 + (threadIdx.x >> 5) * 4; }
};

// merge one table entry (18 doubles in shared memory) into ensemble g's global record, then clear it.  Caller holds the
// block's table lock.
__device__ __noinline__ void pn_fused_flush(const PnKernelParams& p, volatile double* mom, int g)
{
    bool done = false;
    while (!done) {                                   // try-lock loop: a thread that fails simply tries again
        if (atomicCAS(p.f_lock + g, 0, 1) == 0) {
            __threadfence();
#pragma unroll 1
            for (int k = 0; k < 3; ++k) {
                StMom a = {mom[k * 6 + 0], mom[k * 6 + 1], mom[k * 6 + 2], mom[k * 6 + 3], mom[k * 6 + 4], mom[k * 6 + 5]};
                if (a.n > 0.0) {
                    volatile double* q = p.f_mom + ((size_t)g * 3 + k) * 6;
                    StMom m = {q[0], q[1], q[2], q[3], q[4], q[5]};
                    st_merge(m, a);
                    q[0] = m.n; q[1] = m.mx; q[2] = m.my; q[3] = m.m2x; q[4] = m.m2y; q[5] = m.cxy;
                }
            }
            __threadfence();
            atomicExch(p.f_lock + g, 0);
            done = true;
        } else {
            __nanosleep(200);
        }
    }
#pragma unroll 1
    for (int j = 0; j < 18; ++j) mom[j] = 0.0;
}

// draw system i of the launch's queue (pn_gen.cuh: the bits pn_generate would write), make its seed record and its
// initial unit dot products, and put them into slot `lane` of the warp's ring (ring points at word 0 of that slot,
// words are 32 doubles apart).  Out of line: ~2000 instructions that run once per 32 systems.
template <typename real>
__device__ __noinline__ void pn_fused_draw(const PnKernelParams& p, int i, double* ring, int* ring_idx)
{
    const long long gsys = p.f_base + i;
    const long long e = gsys / p.f_count;
    const GenSpec sp = ((const GenSpec*)p.f_specs)[e];
    double y0[10], m1, m2;
    gen_system_at(sp, (unsigned long long)p.f_n_total, (unsigned long long)(p.f_first + (gsys - e * p.f_count)), y0, m1, m2);
    real rec[PN_REC];
    pn_make_record<real>(y0, m1, m2, p, rec);
#pragma unroll
    for (int j = 0; j < PN_REC; ++j) ring[j * 32] = (double)rec[j];
    const double v9[9] = {y0[1], y0[2], y0[3], y0[4], y0[5], y0[6], y0[7], y0[8], y0[9]};
    double d0[3];
    bool ok0[3];
    pn_unit_dots(v9, d0, ok0);
#pragma unroll
    for (int k = 0; k < 3; ++k) ring[(PN_REC + k) * 32] = ok0[k] ? d0[k] : nan("");
    *ring_idx = i;
}

// merge the calling thread's moments for ensemble g into the block's table (shared-memory try-lock), then clear them
template <int BLOCK>
__device__ __noinline__ void pn_fused_thread_flush(const PnKernelParams& p, const PnFusedSmem<BLOCK>& fs, int g)
{
    double* acc = fs.acc() + threadIdx.x;
    volatile int* tag = fs.tag();
    bool done = false;
    while (!done) {
        if (atomicCAS(fs.lock(), 0, 1) == 0) {
            __threadfence_block();
            int slot = -1, lowest = 0;
#pragma unroll
            for (int w = 0; w < PN_FW; ++w) {
                if (tag[w] == g) slot = w;
                if (tag[w] < tag[lowest]) lowest = w;              // a free entry (-1) or the oldest ensemble
            }
            if (slot < 0) {
                slot = lowest;
                if (tag[slot] >= 0) pn_fused_flush(p, fs.mom() + slot * 18, tag[slot]);
                tag[slot] = g;
            }
            volatile double* m = fs.mom() + slot * 18;
#pragma unroll 1
            for (int k = 0; k < 3; ++k) {
                StMom a = {acc[(k * 6 + 0) * BLOCK], acc[(k * 6 + 1) * BLOCK], acc[(k * 6 + 2) * BLOCK],
                           acc[(k * 6 + 3) * BLOCK], acc[(k * 6 + 4) * BLOCK], acc[(k * 6 + 5) * BLOCK]};
                if (a.n > 0.0) {
                    StMom t = {m[k * 6 + 0], m[k * 6 + 1], m[k * 6 + 2], m[k * 6 + 3], m[k * 6 + 4], m[k * 6 + 5]};
                    st_merge(t, a);
                    m[k * 6 + 0] = t.n; m[k * 6 + 1] = t.mx; m[k * 6 + 2] = t.my; m[k * 6 + 3] = t.m2x; m[k * 6 + 4] = t.m2y; m[k * 6 + 5] = t.cxy;
                }
            }
            __threadfence_block();
            atomicExch(fs.lock(), 0);
            done = true;
        }
    }
#pragma unroll
    for (int j = 0; j < 18; ++j) acc[j * BLOCK] = 0.0;
}

// Finished systems of the fused mode are not reduced by the lane that finished them (one lane working, 31 waiting, ~750
// instructions: 12 % of a run of 170-step inspirals): the lane only parks the final vectors, the initial dot products,
// the index and the code in the warp's done ring (14 shared-memory stores), and when the ring cannot take the next
// arrivals -- and at kernel exit -- the whole warp reduces it, one entry per lane: final unit dot products -> the
// thread's moments and the global histograms.
template <int BLOCK>
__device__ __noinline__ void pn_fused_finish_batch(const PnKernelParams& p, const PnFusedSmem<BLOCK>& fs, unsigned n_entries)
{
    const int tid = threadIdx.x, lane = tid & 31;
    if ((unsigned)lane >= n_entries) return;
    const double* e = fs.done() + (size_t)(tid >> 5) * PN_FDONE * 32 + lane;
    const long long packed = __double_as_longlong(e[12 * 32]);
    const int idx = (int)(packed & 0xffffffffll), code = (int)(packed >> 32);
    const long long gsys = p.f_base + idx;
    const int g = (int)(gsys / p.f_count);
    if (code <= 0) {                                  // failed: left out of all three statistics
#pragma unroll
        for (int k = 0; k < 3; ++k) atomicAdd(p.f_skipped + (size_t)g * 3 + k, 1ull);
        return;
    }
    const double v9[9] = {e[0], e[32], e[64], e[96], e[128], e[160], e[192], e[224], e[256]};
    double df[3], x[3];
    bool okf[3], ok[3];
    pn_unit_dots(v9, df, okf);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        x[k] = e[(9 + k) * 32];
        ok[k] = okf[k] && x[k] == x[k];
        if (!ok[k]) { atomicAdd(p.f_skipped + (size_t)g * 3 + k, 1ull); continue; }
        if (p.f_hist1) atomicAdd(p.f_hist1 + ((size_t)g * 3 + k) * p.f_bins1 + pn_bin_of(df[k], p.f_bins1), 1ull);
        if (p.f_hist2)
            atomicAdd(p.f_hist2 + (((size_t)g * 3 + k) * p.f_bins2 + pn_bin_of(x[k], p.f_bins2)) * p.f_bins2 + pn_bin_of(df[k], p.f_bins2), 1ull);
    }
    if (!(ok[0] || ok[1] || ok[2])) return;
    // the thread's own moments: no lock.  They belong to one ensemble at a time; when the ensemble changes (and at
    // kernel exit) they are merged into the block's table
    double* acc = fs.acc() + tid;
    if (fs.acc_g()[tid] != g) {
        if (fs.acc_g()[tid] >= 0) pn_fused_thread_flush<BLOCK>(p, fs, fs.acc_g()[tid]);
        fs.acc_g()[tid] = g;
    }
#pragma unroll 1
    for (int k = 0; k < 3; ++k) {
        if (!ok[k]) continue;
        StMom a = {acc[(k * 6 + 0) * BLOCK], acc[(k * 6 + 1) * BLOCK], acc[(k * 6 + 2) * BLOCK],
                   acc[(k * 6 + 3) * BLOCK], acc[(k * 6 + 4) * BLOCK], acc[(k * 6 + 5) * BLOCK]};
        st_add(a, x[k], df[k]);
        acc[(k * 6 + 0) * BLOCK] = a.n; acc[(k * 6 + 1) * BLOCK] = a.mx; acc[(k * 6 + 2) * BLOCK] = a.my;
        acc[(k * 6 + 3) * BLOCK] = a.m2x; acc[(k * 6 + 4) * BLOCK] = a.m2y; acc[(k * 6 + 5) * BLOCK] = a.cxy;
    }
}

// The redo pass of the fused mode calls the wide-range trial step out of line: inlined, the draw / statistics calls
// around it push that (rarely used) instantiation 4 bytes over the register file; out of line the arithmetic and the
// results are the same and nothing spills.
__device__ __noinline__ void pn_dp5_trial_outofline(const double (&y)[10], const double (&K1)[10], double h, const PnConsts<double>& c,
                                                    const PnUni<double>& u, const PnBase<double>& base, double (&ynew)[10],
                                                    double (&K7)[10], double (&err)[10], PnBase<double>& base_new, PnFlag& bad)
{
    pn_dp5_trial<true>(y, K1, h, c, u, base, ynew, K7, err, base_new, bad);
}

template <typename real, int BLOCK, int MINB, bool SLOW, bool MIXED = false, int UNI = -1, bool FUSED = false>
__global__ void __launch_bounds__(BLOCK, MINB) pn_integrate_adaptive_kernel(const PnKernelParams p)
{
    if (UNI >= 0) { if (*p.nonuniform != 0) return; }
    else if (!SLOW && p.uni_slot >= 0) { if (*p.nonuniform == 0) return; }
    const unsigned n_queue = SLOW ? *p.redo_count : (unsigned)p.n;     // length of the work queue
    const int* order = SLOW ? p.redo_list : p.order;      // null: index order
    if (SLOW && n_queue == 0u) return;
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    extern __shared__ __align__(16) unsigned char pn_fused_smem[];
    PnFusedSmem<BLOCK> fs(pn_fused_smem);                 // FUSED only (no dynamic shared memory otherwise)
#define ring_used ((unsigned)fs.wstate()[0])
#define ring_count ((unsigned)fs.wstate()[1])
#define done_n ((unsigned)fs.wstate()[2])
    if constexpr (FUSED) {
#pragma unroll
        for (int j = 0; j < 18; ++j) fs.acc()[j * BLOCK + threadIdx.x] = 0.0;
        fs.acc_g()[threadIdx.x] = -1;
        if (threadIdx.x < PN_FW * 18) fs.mom()[threadIdx.x] = 0.0;
        if (threadIdx.x < PN_FW) fs.tag()[threadIdx.x] = -1;
        if (threadIdx.x < 2) fs.lock()[threadIdx.x] = 0;
        if ((threadIdx.x & 31) < 3) fs.wstate()[threadIdx.x & 31] = 0;
        __syncthreads();
    }

    // lane state.  k1 holds the SCALED slope h*f(y).  Idle lanes are frozen (h = 0, k1 = 0) on a benign
    // dummy state, so the lock-step arithmetic stays finite and never leaves the series' range.
    real y[10], k1[10];
    double yd[10];                   // MIXED only: the state in double (y is its rounded copy)
    PnConsts<real> c;
    PnBase<real> base;
    PnUni<real> u;
    pn_make_uni<real>(p.mask, u);
    u.emax = (real)p.emax;
#pragma unroll
    for (int k = 0; k < 7; ++k) u.qc[k] = (real)p.qc[k];
    pn_make_consts<real>(0.5, 0.5, 0u, c);
    real KB = (real)1;               // UNI: the factor K0/Bc the brace constants of the table row carry (pn_rhs.cuh, FOLD)
    if constexpr (UNI >= 0) {
        const double* uc = pn_uni_table[UNI];
        c.M = (real)uc[0]; c.c2 = (real)uc[1]; c.c4 = (real)uc[2]; c.c5 = (real)uc[3]; c.c6 = (real)uc[4]; c.c7 = (real)uc[5];
        c.p1 = (real)uc[6]; c.p2 = (real)uc[7]; c.q1 = (real)uc[8]; c.q2 = (real)uc[9]; c.K0 = (real)uc[10];
        c.A1 = (real)uc[11]; c.A2 = (real)uc[12]; c.Bc = (real)uc[13]; c.G = (real)uc[14];
        u.c0 = (real)uc[15]; u.c3 = (real)uc[16]; u.cl = (real)uc[17];
#pragma unroll
        for (int k = 0; k < 7; ++k) u.qc[k] = (real)uc[18 + k];
        KB = (real)uc[25];
    }
#pragma unroll
    for (int i = 0; i < 10; ++i) { y[i] = (real)0; k1[i] = (real)0; yd[i] = 0.0; }
    y[0] = (real)0.01; y[9] = (real)1; yd[0] = 0.01; yd[9] = 1.0;
    pn_base_init(c.M * y[0], c.c6, u.cl, base);
    real h = (real)0;
    float atS1 = fmaxf((float)p.atol, 1e-30f), atS2 = atS1;
    double t = 0.0;
    int idx = -1, steps = 0, nrej = 0, nland = 0;
    bool after_reject = false, landing = false;
    bool queue_empty = false;   // warp-uniform
    unsigned tot_steps = 0, tot_rej = 0, tot_land = 0, tot_fail = 0;

    const real omegaf = (real)p.omegaf;
    const real om_hi = (real)(p.omegaf * (1.0 + p.tau));
    const real om_tol = (real)(p.tau * p.omegaf);
    const float rtol = (float)p.rtol, atol1 = fmaxf((float)p.atol, 1e-30f);

    // a lane starts the system whose seed record is rec
    auto start_system = [&](const real (&rec)[PN_REC], int i) {
#pragma unroll
        for (int j = 0; j < 10; ++j) { y[j] = rec[j]; k1[j] = rec[10 + j]; }
        if constexpr (UNI < 0) {
            c.M = rec[20]; c.c2 = rec[21]; c.c4 = rec[22]; c.c5 = rec[23]; c.c6 = rec[24]; c.c7 = rec[25];
            c.p1 = rec[26]; c.p2 = rec[27]; c.q1 = rec[28]; c.q2 = rec[29]; c.K0 = rec[30]; c.A1 = rec[31];
            c.A2 = rec[32]; c.Bc = rec[33]; c.G = rec[34];
        }
        base.r0 = rec[35]; base.r03 = rec[36]; base.k6b = UNI >= 0 ? KB * rec[37] : rec[37];
        atS1 = fmaxf((float)rec[38], 1e-30f); atS2 = fmaxf((float)rec[39], 1e-30f);   // keeps every scale > 0 (atol = 0 is allowed)
        t = 0.0; steps = 0; nrej = 0; nland = 0; after_reject = false; landing = false;
        idx = i;
        h = p.h0 > 0.0 ? (real)p.h0 : (real)10 * c.M;
    };

    for (;;) {
        if constexpr (FUSED) {
            // ---------------- fused refill: draw 32 systems per warp into the ring, idle lanes pop ----------------
            if (__any_sync(FULL, idx < 0) && !(queue_empty && ring_used >= ring_count)) {
                double* ring_w = fs.ring() + (size_t)(threadIdx.x >> 5) * PN_FREC * 32;
                int* ring_idx_w = fs.ring_idx() + (threadIdx.x >> 5) * 32;
                if (ring_used >= ring_count) {
                    // 32 systems per draw, except in the last wave of the queue (fewer systems left than resident lanes):
                    // there a warp draws only what its idle lanes start right now, so that no warp sits on drawn but
                    // unstarted systems while lanes elsewhere have run dry (the drain tail stays one inspiral long)
                    unsigned* qptr = SLOW ? p.queue2 : p.queue;
                    const unsigned idle_now = (unsigned)__popc(__ballot_sync(FULL, idx < 0));
                    unsigned qb = 0, take = 32u;
                    if (lane == 0) {
                        const unsigned seen = *(volatile unsigned*)qptr;
                        if (seen + p.f_resident >= n_queue) take = idle_now;
                        qb = atomicAdd(qptr, take);
                    }
                    qb = __shfl_sync(FULL, qb, 0);
                    take = __shfl_sync(FULL, take, 0);
                    const unsigned drawn = qb < n_queue ? min(take, n_queue - qb) : 0u;
                    __syncwarp();
                    if (lane == 0) { fs.wstate()[0] = 0; fs.wstate()[1] = (int)drawn; }
                    __syncwarp();
                    if (qb + take >= n_queue) queue_empty = true;
                    if ((unsigned)lane < drawn) pn_fused_draw<real>(p, order ? order[qb + lane] : (int)(qb + lane), ring_w + lane, ring_idx_w + lane);
                    __syncwarp();
                }
                const unsigned need = __ballot_sync(FULL, idx < 0);
                const unsigned used = ring_used, avail = ring_count - used;
                const unsigned rank = (unsigned)__popc(need & ((1u << lane) - 1u));
                if (idx < 0 && rank < avail) {
                    const unsigned slot = used + rank;
                    real rec[PN_REC];
#pragma unroll
                    for (int j = 0; j < PN_REC; ++j) rec[j] = (real)ring_w[j * 32 + slot];
#pragma unroll
                    for (int k = 0; k < 3; ++k) fs.xin()[k * BLOCK + threadIdx.x] = ring_w[(PN_REC + k) * 32 + slot];
                    start_system(rec, ring_idx_w[slot]);
                }
                __syncwarp();
                if (lane == 0) fs.wstate()[0] = (int)(used + min((unsigned)__popc(need), avail));
                __syncwarp();
            }
        } else
        // ---------------- refill: lanes without a system pull the next queue entries ----------------
        if (!queue_empty && __any_sync(FULL, idx < 0)) {
            const unsigned wm = __ballot_sync(FULL, idx < 0);
            const int leader = __ffs(wm) - 1;
            unsigned qbase = 0;
            if (lane == leader) qbase = atomicAdd(SLOW ? p.queue2 : p.queue, (unsigned)__popc(wm));
            qbase = __shfl_sync(FULL, qbase, leader);
            if (qbase + (unsigned)__popc(wm) >= n_queue) queue_empty = true;
            if (idx < 0) {
                const unsigned q = qbase + (unsigned)__popc(wm & ((1u << lane) - 1u));
                if (q < n_queue) {
                    const int i = order ? order[q] : (int)q;
                    real rec[PN_REC];
                    pn_load_record<real>(p.seed, i, rec);
                    if (rec[38] < (real)0) {
                        // bad input: already failed and stored by the seed kernel; the lane stays frozen and
                        // asks again next iteration
                    } else {
                        if constexpr (MIXED)
#pragma unroll
                            for (int j = 0; j < 10; ++j) yd[j] = __ldg(p.y0 + (size_t)j * p.n + i);
                        start_system(rec, i);
                    }
                }
            }
        }
        if (__all_sync(FULL, idx < 0)) {
            if (queue_empty && (!FUSED || ring_used >= ring_count)) break;
            continue;                        // only bad-input lanes were drawn: ask again
        }

        // ---------------- one DP5(4) trial step, all lanes, one basic block ----------------
        real ynew[10], k7[10], err[10], dy[10];
        PnBase<real> base_new;
        PnFlag flag;
        if constexpr (MIXED) pn_dp5_trial<SLOW, real, true>(y, k1, h, c, u, base, ynew, k7, err, base_new, flag, dy);
        else if constexpr (FUSED && SLOW) pn_dp5_trial_outofline(y, k1, h, c, u, base, ynew, k7, err, base_new, flag);
        else pn_dp5_trial<SLOW, real, false, real, 10, (UNI >= 0)>(y, k1, h, c, u, base, ynew, k7, err, base_new, flag);
        const bool bad = flag.out_of_range(u.emax);
        // scaled RMS error norm (R6): sc_j = atol N_j + rtol max(|y_j|, |ynew_j|), E^2 = mean (err_j/sc_j)^2.
        // It only decides accept/reject and the next step size, so ~1e-6 relative accuracy is ample:
        // FP64: the larger magnitude is picked by comparing the high words (integer pipe), 1/sc_j is the raw
        // MUFU seed (rcp.approx.ftz.f64, ~2^-23, no Newton step): 3 FP64 instructions per component and no
        // F64<->F32 conversions (which issue at 1/8 rate and put a long serial tail at the end of the step).
        float E2 = pn_err_norm2(y, ynew, err, rtol, atol1, atS1, atS2);
        // a huge but finite error ratio (atol = 0 and a tiny scale) overflows the float to +inf: that is a rejection with
        // the smallest step factor, not a non-finite state; only NaN is reported as PN_FAIL_NONFINITE
        E2 = (E2 > FLT_MAX) ? 1e30f : E2;
        // `bad`: a stage of this trial left the range of the cbrt/log series (|1 - x/x0| > emax; only at loose
        // tolerances).  Fast kernel: if the trial fails error control anyway (the usual case: an overshoot while the
        // step size ramps up) it is an ordinary rejection (the estimate is inaccurate there, but it only sets the step-size
        // factor; a non-finite one gives the smallest factor); if it would be ACCEPTED, its slopes
        // cannot be trusted and the system is handed to the redo pass, which evaluates both functions over a wide
        // range.  Redo kernel: `bad` means omega more than doubled inside one step: rejected.
        if (!SLOW) {
            if (idx >= 0 && bad && E2 <= 1.0f) {
                p.redo_list[atomicAdd(p.redo_count, 1u)] = idx;
                idx = -1;
            }
            E2 = (bad && !(E2 <= FLT_MAX)) ? 1e30f : E2;      // keep a finite estimate: it sets the factor of the rejection
        } else {
            E2 = bad ? 1e30f : E2;
        }

        // ---------------- per-lane decision as straight-line selects ----------------
        // controller factor 0.9 (E^2)^{-1/10} on the FP32 special-function unit (R8)
        const float fac = 0.9f * pn_ex2_f(-0.1f * pn_lg2_f(fminf(fmaxf(E2, 1e-30f), 1e30f)));
        const bool active = idx >= 0;
        const bool finite = E2 <= FLT_MAX;                 // false for NaN and inf
        const bool ok = E2 <= 1.0f;
        const real om_new = ynew[0];
        // omega_new - omega_f; MIXED forms it in double from the double state (float could not resolve tau = 1e-8)
        real om_ex = om_new - omegaf;
        if constexpr (MIXED) om_ex = (real)((yd[0] + (double)dy[0]) - p.omegaf);
        const bool over = active && ok && (MIXED ? (om_ex > om_tol) : (om_new > om_hi));   // passes error control, overshoots omega_f
        const bool accept = active && ok && !over;
        const bool landed = accept && (pn_abs(om_ex) <= om_tol);
        const bool reject = active && finite && !ok;
        real ratio = (real)fminf(fmaxf(fac, 0.2f), (after_reject || reject) ? 1.0f : 5.0f);   // h_next / h
        if (!active) ratio = (real)0;                      // idle (or just handed to the redo pass): frozen
        steps += active ? 1 : 0;
        tot_steps += active ? 1u : 0u;
        if constexpr (!FUSED) nrej += reject ? 1 : 0;      // per-system count: an output of the unfused path only
        tot_rej += reject ? 1u : 0u;
        if (accept) t += (double)h;
        after_reject = reject || (after_reject && !accept);
        if (over || (accept && landing)) {
            // landing on omega_f (R12): Newton on h with d(omega_new)/dh ~ k7[0]/h.
            // over: discard the step and retry from the same state; accepted-short: first guess from the new state
            const real d = (over ? om_ex : -om_ex) / k7[0];
            ratio = over ? pn_max((real)1 - d, (real)0.1) : pn_min((real)1, d);
            if (over) { ++tot_land; ++nland; landing = true; }
        }
        if (accept) nland = 0;
        const real h_next = h * ratio;
        // rare exits: finished, non-finite, landing failure, max_steps, step-size underflow (t + h == t);
        // priority by overwrite order, all selects, one branch
        // step-size underflow exactly as the oracle defines it: t + h == t, or h not above 1e-300 (a landing correction of
        // a long inspiral can be one ulp of t ~ 2e5; a coarser test mistakes that for stagnation)
        const bool underflow = !(pn_abs(h_next) > PnLimits<real>::tiny()) || (t + (double)h_next == t);
        int code = 0;
        code = underflow ? PN_F_HUNDERFLOW : code;
        code = (steps >= p.max_steps) ? PN_F_MAXSTEPS : code;
        code = (nland > 50) ? PN_F_LANDING : code;
        code = landed ? steps : code;
        code = !finite ? PN_F_NONFINITE : code;
        code = active ? code : 0;
        if constexpr (FUSED) {
            const unsigned fm = __ballot_sync(FULL, code != 0);
            if (fm != 0u) {
                const unsigned nf = (unsigned)__popc(fm);
                unsigned parked = done_n;
                if (parked + nf > 32u) { pn_fused_finish_batch<BLOCK>(p, fs, parked); parked = 0u; __syncwarp(); }
                if (code != 0) {
                    double* e = fs.done() + (size_t)(threadIdx.x >> 5) * PN_FDONE * 32 + parked + (unsigned)__popc(fm & ((1u << lane) - 1u));
#pragma unroll
                    for (int i = 0; i < 9; ++i) e[i * 32] = (double)(accept ? ynew[i + 1] : y[i + 1]);
#pragma unroll
                    for (int k = 0; k < 3; ++k) e[(9 + k) * 32] = fs.xin()[k * BLOCK + threadIdx.x];
                    e[12 * 32] = __longlong_as_double(((long long)code << 32) | (long long)(unsigned)idx);
                    if (code < 0) {
                        atomicMax(p.status, code == PN_F_NONFINITE ? PN_ST_ENONFINITE : PN_ST_ENOTCONVERGED);
                        ++tot_fail;
                    }
                    idx = -1;
                    ratio = (real)0;              // freeze the lane
                }
                __syncwarp();
                if (lane == 0) fs.wstate()[2] = (int)(parked + nf);
                __syncwarp();
            }
        } else
        if (code != 0) {
            if constexpr (MIXED) {
                double yo[10];
#pragma unroll
                for (int i = 0; i < 10; ++i) yo[i] = accept ? yd[i] + (double)dy[i] : yd[i];
                pn_store_result(p, idx, yo, code, t, nrej);
            } else {
                if (accept) pn_store_result(p, idx, ynew, code, t, nrej);
                else pn_store_result(p, idx, y, code, t, nrej);
            }
            if (code < 0) {
                atomicMax(p.status, code == PN_F_NONFINITE ? PN_ST_ENONFINITE : PN_ST_ENOTCONVERGED);
                ++tot_fail;
            }
            idx = -1;
            ratio = (real)0;              // freeze the lane
        }
        // unified update: the kept slope vector is rescaled to the next step size (K1 <- (h'/h) K)
#pragma unroll
        for (int i = 0; i < 10; ++i) {
            k1[i] = ratio * (accept ? k7[i] : k1[i]);
            if constexpr (MIXED) {
                yd[i] = accept ? yd[i] + (double)dy[i] : yd[i];      // the one double-precision operation per component
                y[i] = (real)yd[i];
            } else {
                y[i] = accept ? ynew[i] : y[i];
            }
        }
        base.r0 = accept ? base_new.r0 : base.r0;
        base.r03 = accept ? base_new.r03 : base.r03;
        base.k6b = accept ? base_new.k6b : base.k6b;
        h *= ratio;
    }

    if constexpr (FUSED) {
        // the warp reduces what is left in its done ring; every thread merges its own moments into the block's table; the
        // last thread of the block to leave the loop merges the table into the global records
        if (done_n != 0u) pn_fused_finish_batch<BLOCK>(p, fs, done_n);
        __syncwarp();
        if (fs.acc_g()[threadIdx.x] >= 0) pn_fused_thread_flush<BLOCK>(p, fs, fs.acc_g()[threadIdx.x]);
        __threadfence_block();
        if (atomicAdd(fs.lock() + 1, 1) == BLOCK - 1) {
            __threadfence_block();
            for (int w = 0; w < PN_FW; ++w)
                if (((volatile int*)fs.tag())[w] >= 0) pn_fused_flush(p, fs.mom() + w * 18, ((volatile int*)fs.tag())[w]);
        }
    }
    // ---------------- per-launch counters: warp reduce, one atomic per warp ----------------
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        tot_steps += __shfl_xor_sync(FULL, tot_steps, o);
        tot_rej += __shfl_xor_sync(FULL, tot_rej, o);
        tot_land += __shfl_xor_sync(FULL, tot_land, o);
        tot_fail += __shfl_xor_sync(FULL, tot_fail, o);
    }
    if (lane == 0) {
        atomicAdd(p.counters + 0, (unsigned long long)tot_steps);
        atomicAdd(p.counters + 1, (unsigned long long)tot_rej);
        atomicAdd(p.counters + 2, (unsigned long long)tot_land);
        atomicAdd(p.counters + 3, (unsigned long long)tot_fail);
    }
}

#undef ring_used
#undef ring_count
#undef done_n

// Fixed-step mode (tests, R15): exactly fixed_steps DP5 steps of size h0, y <- y_new.
// SLOW = true is the redo pass over the systems that left the series' range in the fast pass.
template <typename real, int BLOCK, bool SLOW>
__global__ void __launch_bounds__(BLOCK) pn_integrate_fixed_kernel(const PnKernelParams p)
{
    const int q = blockIdx.x * BLOCK + threadIdx.x;
    const int nq = SLOW ? (int)*p.redo_count : p.n;
    if (q >= nq) return;
    const int i = SLOW ? p.redo_list[q] : q;
    double y0[10];
#pragma unroll
    for (int j = 0; j < 10; ++j) y0[j] = p.y0[(size_t)j * p.n + i];
    const double m1 = p.masses[i], m2 = p.masses[(size_t)p.n + i];
    real y[10], k1[10];
#pragma unroll
    for (int j = 0; j < 10; ++j) y[j] = (real)y0[j];
    if (!(m1 > 0.0) || !(m2 > 0.0)) {
        pn_store_result(p, i, y, PN_F_BADINPUT, 0.0, 0);
        atomicMax(p.status, PN_ST_EINVAL);
        return;
    }
    PnConsts<real> c;
    pn_make_consts<real>(m1, m2, p.mask, c);
    PnBase<real> base, base_new;
    PnUni<real> u;
    pn_make_uni<real>(p.mask, u);
    u.emax = (real)p.emax;
#pragma unroll
    for (int k = 0; k < 7; ++k) u.qc[k] = (real)p.qc[k];
    pn_base_init(c.M * y[0], c.c6, u.cl, base);
    const real h = (real)(p.h0 > 0.0 ? p.h0 : 10.0 * (m1 + m2));
    real r_tmp, l_tmp;
    PnScaled<real> sc;
    pn_make_scaled(c, h, sc);
    PnFlag flag0;
    pn_rhs<true>(y, c, u, sc, base, k1, r_tmp, l_tmp, flag0);
    double t = 0.0;
    for (int s = 0; s < p.fixed_steps; ++s) {
        real ynew[10], k7[10], err[10];
        PnFlag flag;
        pn_dp5_trial<SLOW>(y, k1, h, c, u, base, ynew, k7, err, base_new, flag);
        if (!SLOW && flag.out_of_range(u.emax)) {
            p.redo_list[atomicAdd(p.redo_count, 1u)] = i;
            return;
        }
        base = base_new;
#pragma unroll
        for (int j = 0; j < 10; ++j) { y[j] = ynew[j]; k1[j] = k7[j]; }
        t += (double)h;
    }
    pn_store_result(p, i, y, p.fixed_steps, t, 0);
    if (threadIdx.x == 0) atomicAdd(p.counters, 0ull);
}

unsigned long long g_pn_launches = 0;

template <typename real, int BLOCK, int MINB, bool SLOW, bool MIXED = false, int UNI = -1>
static cudaError_t launch_adaptive(const PnKernelParams& p, int grid_blocks, cudaStream_t s)
{
    auto kern = pn_integrate_adaptive_kernel<real, BLOCK, MINB, SLOW, MIXED, UNI>;
    // SMs x resident blocks, looked up once per (kernel, device): the occupancy query is a host-side call per launch otherwise
    static int grid_full[64] = {0};
    int dev = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    int& gf = grid_full[dev & 63];
    if (gf == 0) {
        int sms = 0, per_sm = 0;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, BLOCK, 0)) != cudaSuccess) return e;
        gf = sms * (per_sm < 1 ? 1 : per_sm);
    }
    int grid = grid_blocks > 0 ? grid_blocks : gf;
    const long long need = ((long long)p.n + BLOCK - 1) / BLOCK;
    if (need < grid) grid = (int)need;
    if (grid < 1) grid = 1;
    kern<<<grid, BLOCK, 0, s>>>(p);
    ++g_pn_launches;
    return cudaGetLastError();
}

// One chunk of a fused ensemble run: the fast kernel draws and integrates systems [p.f_base, p.f_base + p.n); the redo
// pass re-draws and re-integrates those that left the range of the cbrt/log series (their chunk-local indices are in
// p.redo_list).  p.queue, p.queue2, p.redo_count must be zero on entry.
// fast fused kernel (UNI = -1: generic; >= 0: one fixed-mass ensemble, constants from row UNI of the table) + redo pass
template <int UNI>
static cudaError_t launch_fused_pair(PnKernelParams& p, int grid_blocks, cudaStream_t s)
{
    constexpr int BLOCK = 128, MINB = 2;
    auto fast = pn_integrate_adaptive_kernel<double, BLOCK, MINB, false, false, UNI, true>;
    auto redo = pn_integrate_adaptive_kernel<double, BLOCK, MINB, true, false, -1, true>;
    const int shm = (int)PnFusedSmem<BLOCK>::bytes();
    static int grid_full[64] = {0};
    int dev = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    int& gf = grid_full[dev & 63];
    if (gf == 0) {
        int sms = 0, per_sm = 0;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaFuncSetAttribute(fast, cudaFuncAttributeMaxDynamicSharedMemorySize, shm)) != cudaSuccess) return e;
        if ((e = cudaFuncSetAttribute(redo, cudaFuncAttributeMaxDynamicSharedMemorySize, shm)) != cudaSuccess) return e;
        if ((e = cudaFuncSetAttribute(fast, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared)) != cudaSuccess) return e;
        if ((e = cudaFuncSetAttribute(redo, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fast, BLOCK, shm)) != cudaSuccess) return e;
        gf = sms * (per_sm < 1 ? 1 : per_sm);
    }
    int grid = grid_blocks > 0 ? grid_blocks : gf;
    const long long need = ((long long)p.n + BLOCK - 1) / BLOCK;
    if (need < grid) grid = (int)need;
    if (grid < 1) grid = 1;
    p.uni_slot = -1;
    p.f_resident = (unsigned)grid * BLOCK;
    fast<<<grid, BLOCK, shm, s>>>(p);
    redo<<<grid, BLOCK, shm, s>>>(p);
    g_pn_launches += 2;
    return cudaGetLastError();
}

// uni_slot >= 0: every system of this launch belongs to ONE ensemble with fixed masses (ensemble uni_ens): its constants go
// into row uni_slot of the uniform-mass table (one-thread kernel, then a device-to-device copy on the stream) and the fast
// kernel is the uniform-mass instantiation; the redo pass stays generic
cudaError_t pn_launch_fused(PnKernelParams& p, int grid_blocks, cudaStream_t s, int uni_slot, int uni_ens)
{
    if (p.n <= 0) return cudaSuccess;
    cudaError_t e;
    p.order = nullptr;
    if (p.keys) {
        // queue order, longest expected first: 8 bytes of scratch per system of the chunk
        if ((e = pn_launch_order_init(p.order_scratch, s)) != cudaSuccess) return e;
        pn_fused_keys_kernel<<<(p.n + 127) / 128, 128, 0, s>>>(p);
        ++g_pn_launches;
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        // 48 systems per resident lane and more with near-equal keys: input order (as pn_launch_integrate; SMs of THIS device)
        int dev = 0, sms = 148;
        if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        const long long n_flat = 48LL * sms * 256;
        if ((e = pn_launch_cost_order(p.keys, p.n, p.order_scratch, p.order_out, s, (int)(n_flat < 0x7fffffffLL ? n_flat : 0x7fffffffLL))) != cudaSuccess) return e;
        p.order = p.order_out;
    }
    if (uni_slot < 0) return launch_fused_pair<-1>(p, grid_blocks, s);
    pn_fused_row_kernel<<<1, 1, 0, s>>>(p, uni_ens);
    ++g_pn_launches;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if ((e = cudaMemcpyToSymbolAsync(pn_uni_table, p.uni_row, PN_UNI_ROW * sizeof(double),
                                     (size_t)uni_slot * PN_UNI_ROW * sizeof(double), cudaMemcpyDeviceToDevice, s)) != cudaSuccess)
        return e;
    static_assert(PN_UNI_SLOTS == 4, "one instantiation of the uniform-mass kernel per table row");
    if (uni_slot == 0) return launch_fused_pair<0>(p, grid_blocks, s);
    if (uni_slot == 1) return launch_fused_pair<1>(p, grid_blocks, s);
    if (uni_slot == 2) return launch_fused_pair<2>(p, grid_blocks, s);
    return launch_fused_pair<3>(p, grid_blocks, s);
}

cudaError_t pn_launch_integrate(PnKernelParams& p, int precision, int block_threads, int grid_blocks,
                                cudaStream_t s, int variant)
{
    if (p.n <= 0) return cudaSuccess;
    if (p.fixed_steps > 0) {
        const int B = 128;
        const int grid = (p.n + B - 1) / B;
        if (precision == 0) {
            pn_integrate_fixed_kernel<double, B, false><<<grid, B, 0, s>>>(p);
            pn_integrate_fixed_kernel<double, B, true><<<grid, B, 0, s>>>(p);
            ++g_pn_launches;
        } else {
            pn_integrate_fixed_kernel<float, B, false><<<grid, B, 0, s>>>(p);
        }
        ++g_pn_launches;
        return cudaGetLastError();
    }
    cudaError_t e;
    {
        // stage-in: per-system seed records (constants, base powers, K1 = h0 f(y0)), expected-cost keys; bad inputs fail here
        const int grid = (p.n + 127) / 128;
        if (p.keys && (e = pn_launch_order_init(p.order_scratch, s)) != cudaSuccess) return e;
        p.rec_pairs = (precision == 1 && block_threads == 0 && !(variant & 2)) ? 1 : 0;      // consumer: the pair-packed kernel
        if (precision == 0) pn_seed_kernel<double><<<grid, 128, 0, s>>>(p);
        else pn_seed_kernel<float><<<grid, 128, 0, s>>>(p);
        ++g_pn_launches;
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        // queue order: longest expected first
        if (p.keys) {
            // 48 systems per resident lane and more: the order is not worth the scattered stores (pn_aux.cu, pn_order_range)
            int dev = 0, sms = 148;
            cudaGetDevice(&dev);
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
            const long long n_flat = 48LL * sms * (precision == 1 ? 512 : 256);
            if ((e = pn_launch_cost_order(p.keys, p.n, p.order_scratch, p.order_out, s, (int)(n_flat < 0x7fffffffLL ? n_flat : 0x7fffffffLL))) != cudaSuccess) return e;
        }
    }
    const int ctx_slot = p.uni_slot;
    const int slot = (precision == 0 && block_threads != 256 && !(variant & 1)) ? p.uni_slot : -1;
    p.uni_slot = -1;                 // >= 0 only for the kernel pair below
    if (precision == 0) {
        if (block_threads == 256) e = launch_adaptive<double, 256, 1, false>(p, grid_blocks, s);
        else if (slot < 0) e = launch_adaptive<double, 128, 2, false>(p, grid_blocks, s);
        else {
            p.uni_slot = slot;
            // uniform-mass fast path, decided on the device: system 0's constants (bitwise those of its seed record) go
            // into the __constant__ table on the stream, then both kernels of the pair are launched
            if ((e = cudaMemcpyToSymbolAsync(pn_uni_table, p.uni_row, PN_UNI_ROW * sizeof(double),
                                             (size_t)p.uni_slot * PN_UNI_ROW * sizeof(double), cudaMemcpyDeviceToDevice, s)) != cudaSuccess)
                return e;
            static_assert(PN_UNI_SLOTS == 4, "one instantiation of the uniform-mass kernel per table row");
            if (slot == 0) e = launch_adaptive<double, 128, 2, false, false, 0>(p, grid_blocks, s);
            else if (slot == 1) e = launch_adaptive<double, 128, 2, false, false, 1>(p, grid_blocks, s);
            else if (slot == 2) e = launch_adaptive<double, 128, 2, false, false, 2>(p, grid_blocks, s);
            else e = launch_adaptive<double, 128, 2, false, false, 3>(p, grid_blocks, s);
            if (e != cudaSuccess) return e;
            e = launch_adaptive<double, 128, 2, false>(p, grid_blocks, s);
            p.uni_slot = -1;
        }
        if (e != cudaSuccess) return e;
        // redo pass for systems that left the series' range; its queue length is read on the device
        return launch_adaptive<double, 128, 2, true>(p, grid_blocks, s);
    }
    if (precision == 2) return launch_adaptive<float, 128, 3, false, true>(p, grid_blocks, s);   // PN_MIXED
    // PN_FP32: two systems per lane with packed f32x2 arithmetic (pn_integrate_packed.cu) unless the scalar kernel is
    // asked for (pn_options.variant bit 1, or an explicit block shape); the results are bit-identical
    if (block_threads == 128) return launch_adaptive<float, 128, 4, false>(p, grid_blocks, s);
    if (block_threads == 256 || (variant & 2)) return launch_adaptive<float, 256, 2, false>(p, grid_blocks, s);
    return pn_launch_integrate_packed(p, grid_blocks, s, (variant & 1) ? -1 : ctx_slot);     // its seed records were written with rec_pairs = 1 above
}
