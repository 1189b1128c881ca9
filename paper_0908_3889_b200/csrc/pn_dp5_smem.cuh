// pn_dp5_smem.cuh -- FP64 Dormand-Prince 5(4) trial step with the older slope vectors parked in shared
// memory, so that the integrator fits 168 registers and runs 3 warps per scheduler instead of 2.
//
// Why: the FP64 pipe issues one warp instruction every 2 cycles; with 2 resident warps per scheduler the
// dependent-issue latency of the DFMA chains is exposed ("wait" stalls, ~67 % pipe utilisation in
// profiles/r1_v2).  A third warp hides it, but y, k1..k6, the stage argument and 19 per-system constants
// are ~100 doubles = 200 registers.  k2, k3, k4, k5 and the partial error sum are each written once and
// read 1-3 times per step, so they live in shared memory: 50 doubles = 400 B per thread, slot-major
// (slot * BLOCK + thread) so that a warp access is 32 consecutive doubles (conflict-free), 150 KB per SM at
// 384 threads.  Traffic: 50 STS.64 + 100 LDS.64 per trial step against ~950 FP64 instructions.
// The freshest slope vector is always consumed from registers; only older ones are re-read.
#pragma once
#include "pn_dp5.cuh"

#define PN_SM_K2 0
#define PN_SM_K3 10
#define PN_SM_K4 20
#define PN_SM_K5 30
#define PN_SM_ERR 40
#define PN_SM_SLOTS 50

template <int BLOCK>
struct PnSmem {
    unsigned addr;   // shared-window byte address of this thread's slot 0
    __device__ __forceinline__ void st(int slot, double v) const
    {
        asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr + (unsigned)(slot * BLOCK * 8)), "d"(v));
    }
    __device__ __forceinline__ double ld(int slot) const
    {
        double v;
        asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr + (unsigned)(slot * BLOCK * 8)));
        return v;
    }
};

template <bool SLOW, int BLOCK>
__device__ __forceinline__ void pn_dp5_trial_smem(const double (&y)[10], const double (&K1)[10], double h,
                                                  const PnConsts<double>& c, const PnUni<double>& u, const PnBase<double>& base,
                                                  const PnSmem<BLOCK>& sm, double (&ynew)[10], double (&K7)[10],
                                                  double (&err)[10], PnBase<double>& base_new, bool& bad)
{
    double ys[10], kf[10];   // stage argument, freshest (scaled) slope vector
    double r_tmp, l_tmp;
    PnScaled<double> sc;
    pn_make_scaled(c, h, sc);
#pragma unroll
    for (int i = 0; i < 10; ++i) ys[i] = fma(DP_A21, K1[i], y[i]);
    pn_rhs<SLOW>(ys, c, u, sc, base, kf, r_tmp, l_tmp, bad);              // kf = K2
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        sm.st(PN_SM_K2 + i, kf[i]);
        ys[i] = fma(DP_A32, kf[i], fma(DP_A31, K1[i], y[i]));
    }
    pn_rhs<SLOW>(ys, c, u, sc, base, kf, r_tmp, l_tmp, bad);              // kf = K3
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        sm.st(PN_SM_K3 + i, kf[i]);
        ys[i] = fma(DP_A43, kf[i], fma(DP_A42, sm.ld(PN_SM_K2 + i), fma(DP_A41, K1[i], y[i])));
    }
    pn_rhs<SLOW>(ys, c, u, sc, base, kf, r_tmp, l_tmp, bad);              // kf = K4
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        sm.st(PN_SM_K4 + i, kf[i]);
        ys[i] = fma(DP_A54, kf[i], fma(DP_A53, sm.ld(PN_SM_K3 + i), fma(DP_A52, sm.ld(PN_SM_K2 + i), fma(DP_A51, K1[i], y[i]))));
    }
    pn_rhs<SLOW>(ys, c, u, sc, base, kf, r_tmp, l_tmp, bad);              // kf = K5
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        sm.st(PN_SM_K5 + i, kf[i]);
        ys[i] = fma(DP_A65, kf[i],
                    fma(DP_A64, sm.ld(PN_SM_K4 + i),
                        fma(DP_A63, sm.ld(PN_SM_K3 + i), fma(DP_A62, sm.ld(PN_SM_K2 + i), fma(DP_A61, K1[i], y[i])))));
    }
    pn_rhs<SLOW>(ys, c, u, sc, base, kf, r_tmp, l_tmp, bad);              // kf = K6
    // stage 7 = 5th-order solution; the error partial is parked while the last RHS runs
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        const double k3i = sm.ld(PN_SM_K3 + i), k4i = sm.ld(PN_SM_K4 + i), k5i = sm.ld(PN_SM_K5 + i);
        ynew[i] = fma(DP_B6, kf[i], fma(DP_B5, k5i, fma(DP_B4, k4i, fma(DP_B3, k3i, fma(DP_B1, K1[i], y[i])))));
        sm.st(PN_SM_ERR + i, fma(DP_E6, kf[i], fma(DP_E5, k5i, fma(DP_E4, k4i, fma(DP_E3, k3i, DP_E1 * K1[i])))));
    }
    pn_rhs<SLOW>(ynew, c, u, sc, base, K7, r_tmp, l_tmp, bad);
    base_new.r0 = r_tmp; base_new.r03 = r_tmp * r_tmp * r_tmp; base_new.l0 = l_tmp;
#pragma unroll
    for (int i = 0; i < 10; ++i) err[i] = fma(DP_E7, K7[i], sm.ld(PN_SM_ERR + i));
}
