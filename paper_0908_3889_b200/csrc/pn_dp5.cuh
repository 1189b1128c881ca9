// pn_dp5.cuh -- one Dormand-Prince 5(4) trial step in registers (PAPER.md:66 names the method; the
// tableau is the standard 7-stage FSAL pair, R5).  Written for register economy:
//   - the step size is folded into the slopes (K_s = h k_s), so a stage argument costs (s-1) FMAs per
//     component with constant coefficients;
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

// Trial step from (y, K1 = h f(y)) with step h.  All slopes are "scaled" (K_s = h k_s, see pn_rhs.cuh), so
// every coefficient below is a compile-time constant.  Outputs y_new (5th order), K7 = h f(y_new) and the
// error estimate err = sum_s e_s K_s.  6 RHS evaluations, 200 + 60 FMAs.
// WANT_DY (mixed precision): the increment dy = sum_s b_s K_s is formed on its own and
// y_new = y + dy, so that the caller can add dy to a higher-precision copy of the state.
// vec / NV: the element type and length of the state and slope arrays.  Default: NV = 10 values of `real`.  The
// pair-packed FP32 kernel (pn_integrate_packed.cu) passes vec = f2, NV = 5: the ten components of ONE system in five
// register pairs, so that every stage sum below is a packed FFMA2 (two components per issue slot); pn_rhs has an
// overload for that layout.
template <bool SLOW, typename real, bool WANT_DY = false, typename vec = real, int NV = 10, bool FOLD = false>
__device__ __forceinline__ void pn_dp5_trial(const vec (&y)[NV], const vec (&K1)[NV], real h,
                                             const PnConsts<real>& c, const PnUni<real>& u, const PnBase<real>& base,
                                             vec (&ynew)[NV], vec (&K7)[NV], vec (&err)[NV], PnBase<real>& base_new, PnFlag& bad,
                                             vec* dy = nullptr)
{
    vec K2[NV], K3[NV], K4[NV], K5[NV], K6[NV], ys[NV];
    real r_tmp, l_tmp;
    PnScaled<real> sc;
    pn_make_scaled(c, h, sc);
#pragma unroll
    for (int i = 0; i < NV; ++i) ys[i] = pn_fma((vec)DP_A21, K1[i], y[i]);
    pn_rhs<SLOW, FOLD>(ys, c, u, sc, base, K2, r_tmp, l_tmp, bad);
#pragma unroll
    for (int i = 0; i < NV; ++i) ys[i] = pn_fma((vec)DP_A32, K2[i], pn_fma((vec)DP_A31, K1[i], y[i]));
    pn_rhs<SLOW, FOLD>(ys, c, u, sc, base, K3, r_tmp, l_tmp, bad);
#pragma unroll
    for (int i = 0; i < NV; ++i)
        ys[i] = pn_fma((vec)DP_A43, K3[i], pn_fma((vec)DP_A42, K2[i], pn_fma((vec)DP_A41, K1[i], y[i])));
    pn_rhs<SLOW, FOLD>(ys, c, u, sc, base, K4, r_tmp, l_tmp, bad);
#pragma unroll
    for (int i = 0; i < NV; ++i)
        ys[i] = pn_fma((vec)DP_A54, K4[i],
                       pn_fma((vec)DP_A53, K3[i], pn_fma((vec)DP_A52, K2[i], pn_fma((vec)DP_A51, K1[i], y[i]))));
    pn_rhs<SLOW, FOLD>(ys, c, u, sc, base, K5, r_tmp, l_tmp, bad);
#pragma unroll
    for (int i = 0; i < NV; ++i)
        ys[i] = pn_fma((vec)DP_A65, K5[i],
                       pn_fma((vec)DP_A64, K4[i],
                              pn_fma((vec)DP_A63, K3[i], pn_fma((vec)DP_A62, K2[i], pn_fma((vec)DP_A61, K1[i], y[i])))));
    pn_rhs<SLOW, FOLD>(ys, c, u, sc, base, K6, r_tmp, l_tmp, bad);
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        if (WANT_DY) {
            dy[i] = pn_fma((vec)DP_B6, K6[i],
                           pn_fma((vec)DP_B5, K5[i],
                                  pn_fma((vec)DP_B4, K4[i], pn_fma((vec)DP_B3, K3[i], (vec)DP_B1 * K1[i]))));
            ynew[i] = y[i] + dy[i];
        } else {
            ynew[i] = pn_fma((vec)DP_B6, K6[i],
                             pn_fma((vec)DP_B5, K5[i],
                                    pn_fma((vec)DP_B4, K4[i], pn_fma((vec)DP_B3, K3[i], pn_fma((vec)DP_B1, K1[i], y[i])))));
        }
        err[i] = pn_fma((vec)DP_E6, K6[i],
                        pn_fma((vec)DP_E5, K5[i],
                               pn_fma((vec)DP_E4, K4[i], pn_fma((vec)DP_E3, K3[i], (vec)DP_E1 * K1[i]))));
    }
    pn_rhs<SLOW, FOLD>(ynew, c, u, sc, base, K7, r_tmp, l_tmp, bad);
    base_new.r0 = r_tmp; base_new.r03 = r_tmp * r_tmp * r_tmp; base_new.k6b = l_tmp;
#pragma unroll
    for (int i = 0; i < NV; ++i) err[i] = pn_fma((vec)DP_E7, K7[i], err[i]);
}
