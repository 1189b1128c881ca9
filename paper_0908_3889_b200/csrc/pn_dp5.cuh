// pn_dp5.cuh -- one Dormand-Prince 5(4) trial step in registers (PAPER.md:66 names the method; the
// tableau is the standard 7-stage FSAL pair, R5).  Written for register economy:
//   - the step size is folded into the coefficients once per stage (h*a_sj), so a stage argument costs
//     (s-1) FMAs per component;
//   - after k6 the 5th-order solution y_new and the partial error sum are formed together, so that
//     k2..k6 are dead while the seventh RHS is evaluated; only y, k1 (kept for a rejected step), y_new
//     and the error partial stay live.
#pragma once
#include "pn_rhs.cuh"

// tableau as compile-time doubles (converted to `real` at the use site)
#define DP_A21 (1.0 / 5.0)
#define DP_A31 (3.0 / 40.0)
#define DP_A32 (9.0 / 40.0)
#define DP_A41 (44.0 / 45.0)
#define DP_A42 (-56.0 / 15.0)
#define DP_A43 (32.0 / 9.0)
#define DP_A51 (19372.0 / 6561.0)
#define DP_A52 (-25360.0 / 2187.0)
#define DP_A53 (64448.0 / 6561.0)
#define DP_A54 (-212.0 / 729.0)
#define DP_A61 (9017.0 / 3168.0)
#define DP_A62 (-355.0 / 33.0)
#define DP_A63 (46732.0 / 5247.0)
#define DP_A64 (49.0 / 176.0)
#define DP_A65 (-5103.0 / 18656.0)
#define DP_B1 (35.0 / 384.0)
#define DP_B3 (500.0 / 1113.0)
#define DP_B4 (125.0 / 192.0)
#define DP_B5 (-2187.0 / 6784.0)
#define DP_B6 (11.0 / 84.0)
// e = b - b^ (b^ = 5179/57600, 0, 7571/16695, 393/640, -92097/339200, 187/2100, 1/40)
#define DP_E1 (71.0 / 57600.0)
#define DP_E3 (-71.0 / 16695.0)
#define DP_E4 (71.0 / 1920.0)
#define DP_E5 (-17253.0 / 339200.0)
#define DP_E6 (22.0 / 525.0)
#define DP_E7 (-1.0 / 40.0)

// Trial step from (y, k1 = f(y)) with step h.  Outputs y_new (5th order), k7 = f(y_new) and the error
// estimate err = h sum_s e_s k_s.  6 RHS evaluations, 200 + 60 FMAs, 26 coefficient multiplies.
template <typename real>
__device__ __forceinline__ void pn_dp5_trial(const real (&y)[10], const real (&k1)[10], real h,
                                             const PnConsts<real>& c, const PnBase<real>& base, real (&ynew)[10],
                                             real (&k7)[10], real (&err)[10], PnBase<real>& base_new)
{
    real k2[10], k3[10], k4[10], k5[10], k6[10], ys[10];
    real r_tmp, l_tmp;
    {
        const real a1 = h * (real)DP_A21;
#pragma unroll
        for (int i = 0; i < 10; ++i) ys[i] = pn_fma(a1, k1[i], y[i]);
        pn_rhs(ys, c, base, k2, r_tmp, l_tmp);
    }
    {
        const real a1 = h * (real)DP_A31, a2 = h * (real)DP_A32;
#pragma unroll
        for (int i = 0; i < 10; ++i) ys[i] = pn_fma(a2, k2[i], pn_fma(a1, k1[i], y[i]));
        pn_rhs(ys, c, base, k3, r_tmp, l_tmp);
    }
    {
        const real a1 = h * (real)DP_A41, a2 = h * (real)DP_A42, a3 = h * (real)DP_A43;
#pragma unroll
        for (int i = 0; i < 10; ++i) ys[i] = pn_fma(a3, k3[i], pn_fma(a2, k2[i], pn_fma(a1, k1[i], y[i])));
        pn_rhs(ys, c, base, k4, r_tmp, l_tmp);
    }
    {
        const real a1 = h * (real)DP_A51, a2 = h * (real)DP_A52, a3 = h * (real)DP_A53, a4 = h * (real)DP_A54;
#pragma unroll
        for (int i = 0; i < 10; ++i)
            ys[i] = pn_fma(a4, k4[i], pn_fma(a3, k3[i], pn_fma(a2, k2[i], pn_fma(a1, k1[i], y[i]))));
        pn_rhs(ys, c, base, k5, r_tmp, l_tmp);
    }
    {
        const real a1 = h * (real)DP_A61, a2 = h * (real)DP_A62, a3 = h * (real)DP_A63, a4 = h * (real)DP_A64,
                   a5 = h * (real)DP_A65;
#pragma unroll
        for (int i = 0; i < 10; ++i)
            ys[i] = pn_fma(a5, k5[i],
                           pn_fma(a4, k4[i], pn_fma(a3, k3[i], pn_fma(a2, k2[i], pn_fma(a1, k1[i], y[i])))));
        pn_rhs(ys, c, base, k6, r_tmp, l_tmp);
    }
    {
        const real b1 = h * (real)DP_B1, b3 = h * (real)DP_B3, b4 = h * (real)DP_B4, b5 = h * (real)DP_B5,
                   b6 = h * (real)DP_B6;
        const real e1 = h * (real)DP_E1, e3 = h * (real)DP_E3, e4 = h * (real)DP_E4, e5 = h * (real)DP_E5,
                   e6 = h * (real)DP_E6;
#pragma unroll
        for (int i = 0; i < 10; ++i) {
            ynew[i] = pn_fma(b6, k6[i], pn_fma(b5, k5[i], pn_fma(b4, k4[i], pn_fma(b3, k3[i], pn_fma(b1, k1[i], y[i])))));
            err[i] = pn_fma(e6, k6[i], pn_fma(e5, k5[i], pn_fma(e4, k4[i], pn_fma(e3, k3[i], e1 * k1[i]))));
        }
        pn_rhs(ynew, c, base, k7, r_tmp, l_tmp);
        base_new.r0 = r_tmp; base_new.r03 = r_tmp * r_tmp * r_tmp; base_new.l0 = l_tmp;
        const real e7 = h * (real)DP_E7;
#pragma unroll
        for (int i = 0; i < 10; ++i) err[i] = pn_fma(e7, k7[i], err[i]);
    }
}
