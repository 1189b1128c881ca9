// pn_integrate_packed.cu -- the default FP32 integrator: one inspiral per lane with its ten components in five
// register pairs and packed f32x2 arithmetic (sm_100a FFMA2 / FMUL2 / FADD2), plus seed-record prefetch.
//
// The plain FP32 kernel (pn_integrate.cu, real = float) is issue-bound: ~965 warp instructions per trial step at one
// per cycle and scheduler (r1: 0.46 of the FP32 FMA peak at 77 % issue utilisation).  Two things changed here.
//  (1) Packing WITHIN a system.  Blackwell's FFMA2 does two FP32 FMAs per lane in one issue slot (measured 74.3 TFLOP/s
//      against 70.9 with FFMA: pn_measure_fma_peak(3) and (PN_FP32), in the bench line as roofline.peak_measured_ffma2 /
//      peak_measured_fma, profiles/r2_bench_lines.md).  Everything that treats the ten components alike --
//      the Dormand-Prince stage sums, the error vector, the state update: 270 of the ~780 FP32 operations of a trial
//      step -- and the x / y halves of the RHS's vector operations are packed (pn_rhs.cuh, pair layout), which removes
//      ~190 issue slots per trial step at an unchanged register count (16 resident warps per SM as before).
//      Tried first and dropped: TWO systems per lane in packed form.  It halves the issue slots but also the resident
//      warps (238 registers), and a packed instruction with three register-pair sources occupies the register-file
//      ports for 3 cycles, exactly like a DFMA: 10.9 ms on C4f against 9.8 ms for the scalar kernel.
//  (2) Record prefetch.  FP32 inspirals are short (C4f: 66 trial steps), so some lane of a warp finishes in almost
//      every iteration, and a refill that waits for the queue atomic (~600 cycles), the order lookup and the 160-byte
//      seed record from DRAM (~800 cycles) stalls the whole warp (r2 capture of the scalar kernel: long_scoreboard 0.75
//      warps per issue).  Every lane therefore reserves its next system while it integrates the current one, in three
//      stages a loop iteration apart -- atomicAdd issued / queue position -> system index (order lookup) issued /
//      cp.async of the record into the lane's shared-memory buffer issued -- so that no stage waits for the one before,
//      and the refill itself is ten 16-byte shared-memory loads.
// Per component the operations and their order are those of the scalar kernel: results are bit-identical (tested).
// (the paper's own runs are single precision.)
#include "pn_step_common.cuh"

// record word -> lane state.  Words 0..9 hold y0 and 10..19 hold K1 in pair order (rec_pairs layout of the seed kernel).
__device__ __forceinline__ void pn_pairs_fill(const float (&rec)[PN_REC], f2 (&y)[5], f2 (&k1)[5], PnConsts<float>& c, float& atS1, float& atS2)
{
#pragma unroll
    for (int j = 0; j < 5; ++j) { y[j] = f2(rec[2 * j], rec[2 * j + 1]); k1[j] = f2(rec[10 + 2 * j], rec[11 + 2 * j]); }
    c.M = rec[20]; c.c2 = rec[21]; c.c4 = rec[22]; c.c5 = rec[23]; c.c6 = rec[24]; c.c7 = rec[25];
    c.p1 = rec[26]; c.p2 = rec[27]; c.q1 = rec[28]; c.q2 = rec[29]; c.K0 = rec[30]; c.A1 = rec[31];
    c.A2 = rec[32]; c.Bc = rec[33]; c.G = rec[34];
    atS1 = fmaxf(rec[38], 1e-30f); atS2 = fmaxf(rec[39], 1e-30f);       // keeps every scale > 0 (atol = 0 is allowed)
}

#define PN_PK_CHUNKS (PN_REC / 4)       /* 16-byte chunks of a float record */

// UNI >= 0: every system of the batch has the masses of system 0 (checked by the seed kernel, as for the FP64 kernels,
// DESIGN.md 7.8): the 15 mass-dependent constants come from row UNI of this table -- uniform-register operands instead of
// per-lane registers (126 -> 114 registers, ~50 three-register FFMAs per trial step become two-register ones).  The row
// holds the very floats of system 0's seed record, so the results are bit-identical to the generic instantiation's.  The
// launcher starts both instantiations; the one that does not apply returns at once.
__constant__ float pn_uni_f[PN_UNI_SLOTS][32];

template <int BLOCK, int MINB, int UNI = -1>
__global__ void __launch_bounds__(BLOCK, MINB) pn_integrate_pairs_kernel(const PnKernelParams p)
{
    if (UNI >= 0) { if (*p.nonuniform != 0) return; }
    else if (p.uni_slot >= 0) { if (*p.nonuniform == 0) return; }
    const unsigned n_queue = (unsigned)p.n;
    const int* order = p.order;
    const unsigned FULL = 0xffffffffu;
    const int lane = threadIdx.x & 31;

    // lane state.  k1 holds the SCALED slope h*f(y).  Idle lanes are frozen (h = 0, k1 = 0) on a benign dummy state, so
    // the lock-step arithmetic stays finite.
    f2 y[5], k1[5];
    PnConsts<float> c;
    PnBase<float> base;
    PnUni<float> u;
    pn_make_uni<float>(p.mask, u);
    u.emax = (float)p.emax;
    pn_make_consts<float>(0.5, 0.5, 0u, c);
    if constexpr (UNI >= 0) {
        const float* uc = pn_uni_f[UNI];
        c.M = uc[0]; c.c2 = uc[1]; c.c4 = uc[2]; c.c5 = uc[3]; c.c6 = uc[4]; c.c7 = uc[5]; c.p1 = uc[6]; c.p2 = uc[7];
        c.q1 = uc[8]; c.q2 = uc[9]; c.K0 = uc[10]; c.A1 = uc[11]; c.A2 = uc[12]; c.Bc = uc[13]; c.G = uc[14];
    }
#pragma unroll
    for (int j = 0; j < 5; ++j) { y[j] = f2(0.0f); k1[j] = f2(0.0f); }
    pn_pair_set<0>(y, 0.01f); pn_pair_set<9>(y, 1.0f);
    pn_base_init(0.01f, 0.0f, 0.0f, base);
    float h = 0.0f;
    const float rtol = (float)p.rtol, atol1 = fmaxf((float)p.atol, 1e-30f);
    float atS1 = atol1, atS2 = atol1;
    double t = 0.0;
    int idx = -1, steps = 0, nrej = 0, nland = 0;
    bool after_reject = false, landing = false;
    bool queue_empty = false;   // warp-uniform
    unsigned tot_steps = 0, tot_rej = 0, tot_land = 0, tot_fail = 0;

    const float omegaf = (float)p.omegaf;
    const float om_hi = (float)(p.omegaf * (1.0 + p.tau));
    const float om_tol = (float)(p.tau * p.omegaf);

    // ---- prefetch pipeline (see the head of this file) ----
    extern __shared__ float4 pn_pf[];       // [2 buffers][PN_PK_CHUNKS][BLOCK] 16-byte words: conflict-free 128-bit accesses
    int nxt = -1;                           // the reserved system
    int stage = 0;                          // 0: none  1: atomicAdd issued  2: system index issued / known  3: record copy issued
    int pb = 0;                             // buffer the next copy goes to; a consumed buffer is not written again before
                                            // the other one has been consumed
    unsigned pend_q = 0, pend_wm = 0;       // lane 0: result of the pending atomicAdd; lanes it serves (warp-uniform)

    for (;;) {
        // ---------------- stage C: the system index has arrived: copy its record into this lane's buffer ----------------
        bool fresh = false;                                        // copy issued in THIS iteration: not readable yet
        const bool any_c = __any_sync(FULL, stage == 2);
        if (any_c) {
            if (stage == 2) {
                const float4* src = (const float4*)((const float*)p.seed + (size_t)nxt * PN_REC);
                const unsigned dst = (unsigned)__cvta_generic_to_shared(pn_pf + (size_t)pb * PN_PK_CHUNKS * BLOCK + threadIdx.x);
#pragma unroll
                for (int k = 0; k < PN_PK_CHUNKS; ++k)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst + (unsigned)(k * BLOCK * 16)), "l"(src + k) : "memory");
                stage = 3;
                fresh = true;
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
        // ---------------- stage B: the atomicAdd has returned: queue position -> system index ----------------
        if (pend_wm != 0u) {
            const unsigned qbase = __shfl_sync(FULL, pend_q, 0);
            if (qbase + (unsigned)__popc(pend_wm) >= n_queue) queue_empty = true;
            if ((pend_wm >> lane) & 1u) {
                const unsigned q = qbase + (unsigned)__popc(pend_wm & ((1u << lane) - 1u));
                if (q < n_queue) { nxt = order ? __ldg(order + q) : (int)q; stage = 2; }
                else stage = 0;                                    // the queue is exhausted
            }
            pend_wm = 0u;
        }
        // ---------------- refill: idle lanes take their prefetched system; stage A: reserve the one after it ----------------
        if (__any_sync(FULL, idx < 0)) {
            // copies issued in an earlier iteration must have landed; the group committed just above may stay in flight
            if (any_c) asm volatile("cp.async.wait_group 1;" ::: "memory");
            else asm volatile("cp.async.wait_group 0;" ::: "memory");
            if (idx < 0 && stage == 3 && !fresh) {
                float rec[PN_REC];
                const float4* src = pn_pf + (size_t)pb * PN_PK_CHUNKS * BLOCK + threadIdx.x;
#pragma unroll
                for (int k = 0; k < PN_PK_CHUNKS; ++k) {
                    const float4 w = src[k * BLOCK];
                    rec[4 * k] = w.x; rec[4 * k + 1] = w.y; rec[4 * k + 2] = w.z; rec[4 * k + 3] = w.w;
                }
                // rec[38] < 0: bad input, already failed and stored by the seed kernel; the lane stays idle and takes the
                // system after it once that one's record has arrived
                if (!(rec[38] < 0.0f)) {
                    if constexpr (UNI >= 0) { PnConsts<float> unused; pn_pairs_fill(rec, y, k1, unused, atS1, atS2); }
                    else pn_pairs_fill(rec, y, k1, c, atS1, atS2);
                    h = p.h0 > 0.0 ? (float)p.h0 : 10.0f * c.M;      // first step (R13)
                    t = 0.0; steps = 0; nrej = 0; nland = 0; after_reject = false; landing = false;
                    idx = nxt;
                }
                stage = 0;
                pb ^= 1;
            }
            if (!queue_empty) {
                const unsigned wm = __ballot_sync(FULL, stage == 0);
                if (wm != 0u) {
                    if (lane == 0) pend_q = atomicAdd(p.queue, (unsigned)__popc(wm));
                    pend_wm = wm;
                    if (stage == 0) stage = 1;
                }
            }
        }
        if (__all_sync(FULL, idx < 0)) {
            if (queue_empty && pend_wm == 0u && __all_sync(FULL, stage == 0)) break;
            continue;                        // a reserved system is on its way, or only bad-input systems were drawn
        }

        // ---------------- one DP5(4) trial step, all lanes, one basic block; stage sums packed ----------------
        f2 ynew[5], k7[5], err[5];
        PnBase<float> base_new;
        PnFlag bad;
        pn_dp5_trial<false, float, false, f2, 5>(y, k1, h, c, u, base, ynew, k7, err, base_new, bad);
        // scaled RMS error norm (R6): scales and ratios packed, the sum in component order as in the scalar kernel
        f2 q[5];
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            // atol per component of the pair: |S1| for S1, |S2| for S2, 1 for omega and L^ (R7)
            const f2 at = j == 0 ? f2(atS1) : (j == 1 ? f2(atS2) : (j == 2 ? f2(atol1) : (j == 3 ? f2(atol1, atS1) : f2(atS2, atol1))));
            const f2 scl = pn_fma(f2(rtol), pn_max(pn_abs(y[j]), pn_abs(ynew[j])), at);      // at >= 1e-30: never 0
            q[j] = err[j] * f2(pn_rcp_f(scl.v.x), pn_rcp_f(scl.v.y));
        }
        float sum = 0.0f;
        { float r;
          r = pn_pair_get<0>(q); sum = fmaf(r, r, sum); r = pn_pair_get<1>(q); sum = fmaf(r, r, sum);
          r = pn_pair_get<2>(q); sum = fmaf(r, r, sum); r = pn_pair_get<3>(q); sum = fmaf(r, r, sum);
          r = pn_pair_get<4>(q); sum = fmaf(r, r, sum); r = pn_pair_get<5>(q); sum = fmaf(r, r, sum);
          r = pn_pair_get<6>(q); sum = fmaf(r, r, sum); r = pn_pair_get<7>(q); sum = fmaf(r, r, sum);
          r = pn_pair_get<8>(q); sum = fmaf(r, r, sum); r = pn_pair_get<9>(q); sum = fmaf(r, r, sum); }
        float E2 = sum * 0.1f;
        E2 = (E2 > FLT_MAX) ? 1e30f : E2;        // an overflowed ratio is a rejection; only NaN is non-finite

        // ---------------- per-lane decision as straight-line selects (as in pn_integrate_adaptive_kernel) ----------------
        const float fac = 0.9f * pn_ex2_f(-0.1f * pn_lg2_f(fminf(fmaxf(E2, 1e-30f), 1e30f)));      // 0.9 (E^2)^{-1/10}, R8
        const bool active = idx >= 0;
        const bool finite = E2 <= FLT_MAX;                 // false for NaN
        const bool ok = E2 <= 1.0f;
        const float om_new = pn_pair_get<0>(ynew);
        const float om_ex = om_new - omegaf;
        const bool over = active && ok && (om_new > om_hi);   // passes error control, overshoots omega_f
        const bool accept = active && ok && !over;
        const bool landed = accept && (fabsf(om_ex) <= om_tol);
        const bool reject = active && finite && !ok;
        float ratio = fminf(fmaxf(fac, 0.2f), (after_reject || reject) ? 1.0f : 5.0f);   // h_next / h
        if (!active) ratio = 0.0f;                         // idle: frozen
        steps += active ? 1 : 0;
        tot_steps += active ? 1u : 0u;
        nrej += reject ? 1 : 0;
        tot_rej += reject ? 1u : 0u;
        if (accept) t += (double)h;
        after_reject = reject || (after_reject && !accept);
        if (over || (accept && landing)) {
            // landing on omega_f (R12): Newton on h with d(omega_new)/dh ~ k7[0]/h
            const float d = (over ? om_ex : -om_ex) / pn_pair_get<0>(k7);
            ratio = over ? fmaxf(1.0f - d, 0.1f) : fminf(1.0f, d);
            if (over) { ++tot_land; ++nland; landing = true; }
        }
        if (accept) nland = 0;
        const float h_next = h * ratio;
        const bool underflow = !(fabsf(h_next) > 1e-30f) || (t + (double)h_next == t);
        int code = 0;
        code = underflow ? PN_F_HUNDERFLOW : code;
        code = (steps >= p.max_steps) ? PN_F_MAXSTEPS : code;
        code = (nland > 50) ? PN_F_LANDING : code;
        code = landed ? steps : code;
        code = !finite ? PN_F_NONFINITE : code;
        code = active ? code : 0;
        if (code != 0) {
            const f2 (&src)[5] = accept ? ynew : y;
            const float yo[10] = {pn_pair_get<0>(src), pn_pair_get<1>(src), pn_pair_get<2>(src), pn_pair_get<3>(src), pn_pair_get<4>(src),
                                  pn_pair_get<5>(src), pn_pair_get<6>(src), pn_pair_get<7>(src), pn_pair_get<8>(src), pn_pair_get<9>(src)};
            pn_store_result(p, idx, yo, code, t, nrej);
            if (code < 0) {
                atomicMax(p.status, code == PN_F_NONFINITE ? PN_ST_ENONFINITE : PN_ST_ENOTCONVERGED);
                ++tot_fail;
            }
            idx = -1;
            ratio = 0.0f;              // freeze the lane
        }
        // unified update: the kept slope vector is rescaled to the next step size (K1 <- (h'/h) K)
#pragma unroll
        for (int j = 0; j < 5; ++j) {
            k1[j] = f2(ratio) * f2(accept ? k7[j].v.x : k1[j].v.x, accept ? k7[j].v.y : k1[j].v.y);
            y[j] = f2(accept ? ynew[j].v.x : y[j].v.x, accept ? ynew[j].v.y : y[j].v.y);
        }
        h *= ratio;
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

template <int UNI>
static cudaError_t launch_pairs(const PnKernelParams& p, int grid_blocks, cudaStream_t s)
{
    constexpr int BLOCK = 256, MINB = 2;
    auto kern = pn_integrate_pairs_kernel<BLOCK, MINB, UNI>;
    const int shm = 2 * PN_PK_CHUNKS * BLOCK * 16;      // record prefetch buffers: 80 KB per block
    static int grid_full[64] = {0};
    int dev = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    int& gf = grid_full[dev & 63];
    if (gf == 0) {
        int sms = 0, per_sm = 0;
        if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
        if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, shm)) != cudaSuccess) return e;
        if ((e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared)) != cudaSuccess) return e;
        if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, BLOCK, shm)) != cudaSuccess) return e;
        gf = sms * (per_sm < 1 ? 1 : per_sm);
    }
    int grid = grid_blocks > 0 ? grid_blocks : gf;
    const long long need = ((long long)p.n + BLOCK - 1) / BLOCK;
    if (need < grid) grid = (int)need;
    if (grid < 1) grid = 1;
    kern<<<grid, BLOCK, shm, s>>>(p);
    ++g_pn_launches;
    return cudaGetLastError();
}

// uni_slot >= 0: the seed kernel has put system 0's constants (floats) at the head of p.uni_row; they go into row uni_slot of
// the table on the stream and both the uniform-mass and the generic instantiation are launched (decided on the device)
cudaError_t pn_launch_integrate_packed(PnKernelParams& p, int grid_blocks, cudaStream_t s, int uni_slot)
{
    p.uni_slot = -1;
    if (uni_slot < 0) return launch_pairs<-1>(p, grid_blocks, s);
    cudaError_t e;
    if ((e = cudaMemcpyToSymbolAsync(pn_uni_f, p.uni_row, 32 * sizeof(float), (size_t)uni_slot * 32 * sizeof(float),
                                     cudaMemcpyDeviceToDevice, s)) != cudaSuccess)
        return e;
    p.uni_slot = uni_slot;
    static_assert(PN_UNI_SLOTS == 4, "one instantiation of the uniform-mass kernel per table row");
    if (uni_slot == 0) e = launch_pairs<0>(p, grid_blocks, s);
    else if (uni_slot == 1) e = launch_pairs<1>(p, grid_blocks, s);
    else if (uni_slot == 2) e = launch_pairs<2>(p, grid_blocks, s);
    else e = launch_pairs<3>(p, grid_blocks, s);
    if (e == cudaSuccess) e = launch_pairs<-1>(p, grid_blocks, s);
    p.uni_slot = -1;
    return e;
}
