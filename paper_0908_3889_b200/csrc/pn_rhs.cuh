// pn_rhs.cuh -- register-resident right-hand side of the precessing PN inspiral ODEs for sm_100a.
//
// Eqs. (1)-(4) of arXiv:0908.3889 rewritten for the device:
//   x = M omega, v = x^{1/3};  everything that depends only on (m1, m2) is folded once per system into
//   PnConsts, the brace of Eq. (1) becomes a Horner polynomial in v whose v^3, v^4 and v^6 coefficients
//   carry the spin-orbit, spin-spin and log terms, and Eq. (4) collapses to
//     Omega_1 = beta (gamma1 L + S2),   gamma_i = A_i x^{-1/3} - 3 (L.S_j),  beta = x^2/(2 M^3),
//     Omega_2 = beta (gamma2 L + S1)    A_i = eta M^2 (4 + 3 m_j/m_i)
//   followed by the two cross products of Eq. (2), c_i = (gamma_i L + S_j) x S_i, S_i_dot = beta c_i, and
//   L_dot = -v/(eta M^2) beta (c_1 + c_2) of Eq. (3).
// This file shares nothing with oracle/ (which evaluates the equations as printed).
#pragma once
#include <cuda_runtime.h>
#include "pn_f2.cuh"

#define PN_MASK_ALL 0x100FFu
#define PN_MASK_SPIN (1u << 16)

// ---- scalar helpers, one overload per precision -------------------------------------------------
__device__ __forceinline__ double pn_fma(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float pn_fma(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double pn_abs(double a) { return fabs(a); }
__device__ __forceinline__ float pn_abs(float a) { return fabsf(a); }
__device__ __forceinline__ double pn_max(double a, double b) { return fmax(a, b); }
__device__ __forceinline__ float pn_max(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ double pn_min(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ float pn_min(float a, float b) { return fminf(a, b); }

// Per-system constants.  Computed in double from (m1, m2, term_mask), stored in `real`.
template <typename real>
struct PnConsts {
    real M;        // m1 + m2
    real c2, c4, c5, c6, c7;  // spin-independent, mass-dependent coefficients of v^k in the brace of Eq. (1)
    real p1, p2;   // spin-orbit: v^3 coefficient += p1 (L.S1) + p2 (L.S2)
    real q1, q2;   // spin-spin:  v^4 coefficient += q1 (S1.S2) + q2 (L.S1)(L.S2)
    real K0;       // omega_dot = K0 v^11 brace,  K0 = 96 eta / (5 M^2)
    real A1, A2;   // A_i = eta M^2 (4 + 3 m_j/m_i): Omega_i = beta (gamma_i L + S_j), gamma_i = A_i x^{-1/3} - 3 L.S_j
    real Bc;       // beta = Bc x^2,  Bc = 1/(2 M^3)
    real G;        // L_dot prefactor: -1/(eta M^2), times v
};

// Coefficients that depend only on term_mask: the same for every system of a launch, so they stay out of the
// per-lane register budget (warp-uniform values).
template <typename real>
struct PnUni {
    real c0;   // the "1" of the brace
    real c3;   // 4 pi, spin-independent part of the v^3 coefficient
    real cl;   // coefficient of ln(x) inside the v^6 term: -(856/105)(2/3)
    real emax; // FP64 fast kernel: largest |1 - x/x0| the cbrt/log series are trusted for (set by the launcher)
    real qc[7]; // FP64 fast kernel: cl / k, k = 1 ... 7: the log series with cl folded in (set by the launcher, pn_powers)
};
// Range flag of a trial step.  `bad`: a stage left the range of the wide-range (SLOW) evaluation.  `emx`: the FP64 fast
// path's running maximum of |e| = |1 - x/x0| over the stages, kept as the float whose bits are the HIGH word of |e|
// (high words of doubles order like floats): one FMNMX per stage instead of a DSETP, compared with emax once per step.
struct PnFlag {
    bool bad; float emx;
    __device__ __forceinline__ PnFlag() : bad(false), emx(0.0f) {}
    __device__ __forceinline__ bool out_of_range(double emax) const { return bad || emx > __int_as_float(__double2hiint(emax)); }
    __device__ __forceinline__ bool out_of_range(float) const { return bad; }
};
template <typename real>
__device__ __forceinline__ void pn_make_uni(unsigned mask, PnUni<real>& u)
{
    if (mask == 0) mask = PN_MASK_ALL;
    u.c0 = (real)((mask >> 0) & 1u ? 1.0 : 0.0);
    u.c3 = (real)((mask >> 3) & 1u ? 4.0 * 3.14159265358979323846 : 0.0);
    u.cl = (real)((mask >> 6) & 1u ? -(856.0 / 105.0) * (2.0 / 3.0) : 0.0);
    u.emax = (real)0.03;
#pragma unroll
    for (int k = 0; k < 7; ++k) u.qc[k] = (real)0;      // the FP64 kernels take them from the launch parameters (uniform operands)
}

template <typename real>
__device__ __forceinline__ void pn_make_consts(double m1, double m2, unsigned mask, PnConsts<real>& c)
{
    if (mask == 0) mask = PN_MASK_ALL;
    const double pi = 3.14159265358979323846, gammaE = 0.5772156649015329;
    const double M = m1 + m2, M2 = M * M;
    const double eta = m1 * m2 / M2;
    const double spin = (mask & PN_MASK_SPIN) ? 1.0 : 0.0;
    auto on = [&](int k) { return (mask >> k) & 1u ? 1.0 : 0.0; };
    c.M = (real)M;
    c.c2 = (real)(on(2) * (-(743.0 + 924.0 * eta) / 336.0));
    c.c4 = (real)(on(4) * (34103.0 / 18144.0 + (13661.0 / 2016.0) * eta + (59.0 / 18.0) * eta * eta));
    c.c5 = (real)(on(5) * (-(4159.0 + 15876.0 * eta) * pi / 672.0));
    // theta^ enters linearly in eta (R1); ln(16 x^{2/3}) = ln 16 + (2/3) ln x, natural log (R2)
    const double theta = 1039.0 / 4620.0;
    c.c6 = (real)(on(6) * (16447322263.0 / 139708800.0 - (1712.0 / 105.0) * gammaE + (16.0 / 3.0) * pi * pi +
                           (-273811877.0 / 1088640.0 + (451.0 / 48.0) * pi * pi - (88.0 / 3.0) * theta) * eta +
                           (541.0 / 896.0) * eta * eta - (5605.0 / 2592.0) * eta * eta * eta -
                           (856.0 / 105.0) * 2.772588722239781237669 /* ln 16 */));
    c.c7 = (real)(on(7) * ((-4415.0 / 4032.0 + (358675.0 / 6048.0) * eta + (91495.0 / 1512.0) * eta * eta) * pi));
    const double w1 = 113.0 * m1 * m1 / M2 + 75.0 * eta, w2 = 113.0 * m2 * m2 / M2 + 75.0 * eta;
    c.p1 = (real)(-on(3) * spin * w1 / (12.0 * m1 * m1));
    c.p2 = (real)(-on(3) * spin * w2 / (12.0 * m2 * m2));
    const double mm = (m1 * m1) * (m2 * m2);
    c.q1 = (real)(-on(4) * spin * 247.0 * eta / (48.0 * mm));
    c.q2 = (real)(on(4) * spin * 721.0 * eta / (48.0 * mm));
    c.K0 = (real)(96.0 * eta / (5.0 * M2));
    c.A1 = (real)(eta * M2 * (4.0 + 3.0 * m2 / m1));
    c.A2 = (real)(eta * M2 * (4.0 + 3.0 * m1 / m2));
    c.Bc = (real)(1.0 / (2.0 * M2 * M));
    c.G = (real)(-1.0 / (eta * M2));
}

// ---- v = x^{1/3} and ln x, once per stage ------------------------------------------------------------
// FP64: the library cbrt + log cost ~50 FP64-pipe instructions per stage, almost as much as the rest of
// the RHS.  Within one trial step omega moves by a fraction of a percent, so both are expanded about the
// step's base point x0 (the accepted state), for which r0 = x0^{-1/3} and l0 = ln x0 are carried:
//     e = 1 - x r0^3            (= 1 - x/x0, one FMA)
//     x^{-1/3} = r0 (1-e)^{-1/3} = r0 (1 + e/3 + 2e^2/9 + 14e^3/81 + ...)
//     ln x     = l0 + log1p(-e)  = l0 - e (1 + e/2 + e^2/3 + ...)
// The first expansion is self-correcting (it is exact in r0 whatever r0's own rounding error), so nothing
// accumulates in r; l0 is chained once per accepted step with a truncation error < 3e-15 at the switch
// point |e| = 0.03, beyond which the trial step is repeated with the library functions (rare).  ~22 FMA-pipe
// instructions per stage.  FP32 uses cbrtf and the MUFU log directly.
// k6b = c6 + cl ln x0: the coefficient of v^6 in the brace of Eq. (1) AT the base point.  The log enters the RHS only
// through k6 = c6 + cl ln x, so the series carries cl (k6 = k6b - e sum_k (cl/k) e^{k-1}) and one FMA per evaluation
// (forming ln x, then cl ln x + c6) is saved.
template <typename real> struct PnBase { real r0, r03, k6b; };

__device__ __forceinline__ void pn_base_init(double x, double c6, double cl, PnBase<double>& b)
{
    b.r0 = rcbrt(x);
    b.r03 = b.r0 * b.r0 * b.r0;
    b.k6b = fma(cl, log(x), c6);
}
__device__ __forceinline__ void pn_base_init(float, float, float, PnBase<float>& b) { b.r0 = b.r03 = b.k6b = 0.0f; }

// r = x^{-1/3} and k6 = c6 + cl ln x  ->  returned so that an accepted step can adopt them as the next base.
// SLOW = false: series only, branch-free; the running maximum of |e| is kept in `flag`, and when it leaves the series'
// range the caller repeats the whole trial step with SLOW = true (wide-range evaluation), so the hot loop stays one
// basic block.
template <bool SLOW>
__device__ __forceinline__ void pn_powers(double x, const PnBase<double>& b, double c6, const PnUni<double>& u, double& k6, double& r, PnFlag& flag)
{
    if (SLOW) {
        // wide-range, call-free evaluation about the same base, exact to rounding for x/x0 in [0.4, 2]:
        //   x^{-1/3} = r0 u,  u = rho^{-1/3} by five cubically convergent iterations u <- u (1 + d/3 + 2 d^2/9),
        //              d = 1 - rho u^3,  rho = x/x0 = 1 - e
        //   ln x     = l0 + 2 atanh(w),  w = (rho - 1)/(rho + 1) = -e/(2 - e);  1/(2 - e) by Newton, no divide
        //   (k6b stands for c6 + cl l0, so k6 = k6b + cl 2 atanh(w))
        // Outside that range (omega more than doubled or halved inside ONE step) e is clamped, the values are
        // finite but wrong, and `flag.bad` tells the caller to reject the step.
        const double e_raw = fma(-x, b.r03, 1.0);
        const double e = fmin(fmax(e_raw, -1.0), 0.6);
        flag.bad = flag.bad || (e_raw < -1.0) || (e_raw > 0.6);
        const double rho = 1.0 - e;
        double uu = 1.0;
#pragma unroll
        for (int it = 0; it < 5; ++it) {
            const double d = fma(-rho * uu, uu * uu, 1.0);
            uu = fma(uu * d, fma(d, 2.0 / 9.0, 1.0 / 3.0), uu);
        }
        r = b.r0 * uu;
        const double den = 2.0 - e;
        double t = fma(e, fma(e, 0.125, 0.25), 0.5);
#pragma unroll
        for (int it = 0; it < 5; ++it) t = t * fma(-den, t, 2.0);
        const double w = -e * t, w2 = w * w;
        double A = 1.0 / 45.0;
#pragma unroll
        for (int k = 21; k >= 1; --k) A = fma(A, w2, 1.0 / (double)(2 * k + 1));
        k6 = fma(u.cl, (2.0 * w) * fma(A, w2, 1.0), b.k6b);
    } else {
        const double e = fma(-x, b.r03, 1.0);
        // range check without a DSETP: running maximum of the high words of |e| (NaN is ignored: a non-finite state is
        // reported as such, not redone)
        flag.emx = fmaxf(flag.emx, fabsf(__int_as_float(__double2hiint(e))));
        // (1-e)^{-1/3} = 1 + e S(e),  S = sum_{k=1..9} s_k e^{k-1},  s_k = prod_{j<k}(1/3 + j)/k!
        // log1p(-e)    =   - e Q(e),  Q = sum_{k=1..7} e^{k-1}/k;  the series carries cl: qc_k = cl/k
        // truncation s10 e^9 < 6.1e-17 for |e| <= 0.03.  Even/odd split in e halves the dependent FMA chains.
        // emax = 0.03 at rtol <= 1e-10 and in fixed-step mode; at looser tolerances it grows as rtol^{1/9}, which keeps
        // the truncation below 1e-3 rtol: a run at rtol 1e-7 need not evaluate f to 1e-16.
        const double e2 = e * e;
        double Sa = 135850.0 / 1594323.0, Sb = 5434.0 / 59049.0;   // s9 | s8
        Sa = fma(Sa, e2, 1976.0 / 19683.0);  Sb = fma(Sb, e2, 728.0 / 6561.0);   // s7 | s6
        Sa = fma(Sa, e2, 91.0 / 729.0);      Sb = fma(Sb, e2, 35.0 / 243.0);     // s5 | s4
        Sa = fma(Sa, e2, 14.0 / 81.0);       Sb = fma(Sb, e2, 2.0 / 9.0);        // s3 | s2
        Sa = fma(Sa, e2, 1.0 / 3.0);                                             // s1
        const double S = fma(Sb, e, Sa);
        // ln x enters only through cl ln(x) x^2 in the brace (|cl| = 5.4, x^2 <= 2.5e-3 for omega <= 0.05/M), so an
        // absolute error of 8e-14 in ln x (the e^8/8 term at the |e| = 0.03 limit; 1e-17 at the typical |e| < 0.01)
        // is below 1.1e-15 relative in omega_dot: Q stops at e^6/7.
        double Qa = u.qc[6], Qb = u.qc[5];
        Qa = fma(Qa, e2, u.qc[4]);  Qb = fma(Qb, e2, u.qc[3]);
        Qa = fma(Qa, e2, u.qc[2]);  Qb = fma(Qb, e2, u.qc[1]);
        Qa = fma(Qa, e2, u.qc[0]);
        const double Q = fma(Qb, e, Qa);
        r = fma(b.r0 * e, S, b.r0);
        k6 = fma(-e, Q, b.k6b);
    }
}
template <bool SLOW>
__device__ __forceinline__ void pn_powers(float x, const PnBase<float>&, float c6, const PnUni<float>& u, float& k6, float& r, PnFlag&)
{
    // x > 0 always (omega > 0, M > 0): one lg2 serves both functions, no special-case code (cbrtf carries branches
    // for 0, inf and denormals).  ln x = lg2(x) ln 2; x^{-1/3} = ex2(-lg2(x)/3) polished by one Newton step
    // r <- r + r (1 - x r^3)/3 (seed error ~2e-7 -> ~1e-13, below float rounding).
    float l2, r0;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l2) : "f"(x));
    k6 = fmaf(u.cl, l2 * 0.693147180559945f, c6);
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r0) : "f"(l2 * (-1.0f / 3.0f)));
    const float e = fmaf(-x * r0, r0 * r0, 1.0f);
    r = fmaf(r0 * e, 1.0f / 3.0f, r0);
}

// The slopes are produced already multiplied by the step size h ("scaled slopes" K = h f): the four
// prefactors that enter every output linearly are pre-multiplied by h once per trial step, which costs
// nothing per evaluation and lets every stage sum of the stepper use compile-time tableau coefficients
// (constant-bank operands) instead of per-lane h*a_sj registers.  This matters on sm_100a because a DFMA
// with three distinct register sources issues every 3 cycles, one with two every 2 (measured,
// DESIGN.md 7.2).
template <typename real> struct PnScaled { real hK0, hBc; };
template <typename real>
__device__ __forceinline__ void pn_make_scaled(const PnConsts<real>& c, real h, PnScaled<real>& s)
{
    s.hK0 = h * c.K0; s.hBc = h * c.Bc;
}

// K = h f(y).  ~65 FMA-pipe instructions plus pn_powers; no memory traffic.  r_out = x^{-1/3} and k6_out = c6 + cl ln x
// of this evaluation are handed back for the base update of an accepted step.
// FOLD (the uniform-mass FP64 kernel): the constants of the brace (c2 ... c7, p, q in `c`; c0, c3, cl, qc in `u`) arrive
// multiplied by K0/Bc, so that omega_dot = (beta v^5) brace' with beta = h Bc x^2 (needed anyway): one multiply fewer.
template <bool SLOW, bool FOLD = false, typename real>
__device__ __forceinline__ void pn_rhs(const real (&y)[10], const PnConsts<real>& c, const PnUni<real>& u,
                                       const PnScaled<real>& sc, const PnBase<real>& base,
                                       real (&f)[10], real& r_out, real& k6_out, PnFlag& flag)
{
    const real x = c.M * y[0];
    real k6, r;
    pn_powers<SLOW>(x, base, c.c6, u, k6, r, flag);
    r_out = r; k6_out = k6;
    // x^{2/3} straight from r = x^{-1/3}, v = x^{1/3} from it with one more multiply
    const real x2 = x * x, v2 = x * r, v = v2 * r, v4 = v2 * v2, v5 = v4 * v;

    const real S1x = y[1], S1y = y[2], S1z = y[3];
    const real S2x = y[4], S2y = y[5], S2z = y[6];
    const real Lx = y[7], Ly = y[8], Lz = y[9];

    const real LS1 = pn_fma(Lx, S1x, pn_fma(Ly, S1y, Lz * S1z));
    const real LS2 = pn_fma(Lx, S2x, pn_fma(Ly, S2y, Lz * S2z));
    const real S12 = pn_fma(S1x, S2x, pn_fma(S1y, S2y, S1z * S2z));

    // Eq. (1): coefficients of v^3, v^4, v^6 carry the spin-orbit, spin-spin, log pieces
    const real k3 = pn_fma(c.p1, LS1, pn_fma(c.p2, LS2, u.c3));
    const real k4 = pn_fma(c.q1, S12, pn_fma(c.q2 * LS1, LS2, c.c4));
    // Estrin form, brace = c0 + v2 (c2 + k3 v) + v4 ((k4 + c5 v) + v2 (k6 + c7 v)): the same six FMAs as Horner's
    // rule in a dependency chain of three instead of six
    const real e67 = pn_fma(c.c7, v, k6), e45 = pn_fma(c.c5, v, k4), e23 = pn_fma(k3, v, c.c2);
    const real hi = pn_fma(e67, v2, e45);
    real B = pn_fma(e23, v2, u.c0);
    B = pn_fma(hi, v4, B);
    const real beta = sc.hBc * x2;
    f[0] = FOLD ? (beta * v5) * B : (sc.hK0 * (v5 * x2)) * B;

    // Eq. (4) over beta = h x^2/(2M^3): Omega_1/beta = gamma1 L + S2, Omega_2/beta = gamma2 L + S1.  gamma_i needs only
    // r and a dot product, so the cross products below do not wait for the powers of v; -3 is an immediate operand, so
    // the two FMAs read two registers (a DFMA with three register sources issues every 3 cycles).
    const real g1 = pn_fma((real)-3.0, LS2, c.A1 * r);
    const real g2 = pn_fma((real)-3.0, LS1, c.A2 * r);
    const real O1x = pn_fma(g1, Lx, S2x), O1y = pn_fma(g1, Ly, S2y), O1z = pn_fma(g1, Lz, S2z);
    const real O2x = pn_fma(g2, Lx, S1x), O2y = pn_fma(g2, Ly, S1y), O2z = pn_fma(g2, Lz, S1z);
    // Eq. (2): S_i_dot = beta (Omega_i/beta) x S_i
    const real c1x = pn_fma(O1y, S1z, -(O1z * S1y));
    const real c1y = pn_fma(O1z, S1x, -(O1x * S1z));
    const real c1z = pn_fma(O1x, S1y, -(O1y * S1x));
    const real c2x = pn_fma(O2y, S2z, -(O2z * S2y));
    const real c2y = pn_fma(O2z, S2x, -(O2x * S2z));
    const real c2z = pn_fma(O2x, S2y, -(O2y * S2x));
    f[1] = beta * c1x; f[2] = beta * c1y; f[3] = beta * c1z;
    f[4] = beta * c2x; f[5] = beta * c2y; f[6] = beta * c2z;
    // Eq. (3): L_dot = -v/(eta M^2) (S1_dot + S2_dot)
    const real gv = c.G * v;
    f[7] = gv * (f[1] + f[4]);
    f[8] = gv * (f[2] + f[5]);
    f[9] = gv * (f[3] + f[6]);
}

// ---- pair-packed FP32 layout (pn_integrate_packed.cu) -------------------------------------------------------------
// The ten components of ONE system in five register pairs, so that everything that treats the components alike (the
// Dormand-Prince stage sums, the error vector, the state update: 270 of the ~780 FP32 operations of a trial step) is
// a packed FFMA2 / FMUL2 (two components per issue slot), and the vector operations of the RHS whose x and y
// components share their scalar factors are packed too:
//     pair 0 = (S1x, S1y)   pair 1 = (S2x, S2y)   pair 2 = (Lx, Ly)   pair 3 = (omega, S1z)   pair 4 = (S2z, Lz)
// Component i of y = (omega, S1, S2, L^) lives in half PN_PAIR_HALF[i] of pair PN_PAIR_OF[i].  Per component the
// operations and their order are exactly those of the scalar pn_rhs above, so the results are bit-identical.
__device__ constexpr int PN_PAIR_OF[10] = {3, 0, 0, 3, 1, 1, 4, 2, 2, 4};
__device__ constexpr int PN_PAIR_HALF[10] = {0, 0, 1, 1, 0, 1, 0, 0, 1, 1};
template <int I> __device__ __forceinline__ float pn_pair_get(const f2 (&a)[5]) { return f2_get<PN_PAIR_HALF[I]>(a[PN_PAIR_OF[I]]); }
template <int I> __device__ __forceinline__ void pn_pair_set(f2 (&a)[5], float x) { f2_set<PN_PAIR_HALF[I]>(a[PN_PAIR_OF[I]], x); }

template <bool SLOW, bool FOLD = false>
__device__ __forceinline__ void pn_rhs(const f2 (&y)[5], const PnConsts<float>& c, const PnUni<float>& u,
                                       const PnScaled<float>& sc, const PnBase<float>& base,
                                       f2 (&f)[5], float& r_out, float& k6_out, PnFlag& flag)
{
    const float x = c.M * y[3].v.x;
    float k6, r;
    pn_powers<SLOW>(x, base, c.c6, u, k6, r, flag);
    r_out = r; k6_out = k6;
    const float x2 = x * x, v2 = x * r, v = v2 * r, v4 = v2 * v2, v5 = v4 * v;

    const float S1x = y[0].v.x, S1y = y[0].v.y, S1z = y[3].v.y;
    const float S2x = y[1].v.x, S2y = y[1].v.y, S2z = y[4].v.x;
    const float Lx = y[2].v.x, Ly = y[2].v.y, Lz = y[4].v.y;

    const float LS1 = fmaf(Lx, S1x, fmaf(Ly, S1y, Lz * S1z));
    const float LS2 = fmaf(Lx, S2x, fmaf(Ly, S2y, Lz * S2z));
    const float S12 = fmaf(S1x, S2x, fmaf(S1y, S2y, S1z * S2z));

    const float k3 = fmaf(c.p1, LS1, fmaf(c.p2, LS2, u.c3));
    const float k4 = fmaf(c.q1, S12, fmaf(c.q2 * LS1, LS2, c.c4));
    const float e67 = fmaf(c.c7, v, k6), e45 = fmaf(c.c5, v, k4), e23 = fmaf(k3, v, c.c2);
    const float hi = fmaf(e67, v2, e45);
    float B = fmaf(e23, v2, u.c0);
    B = fmaf(hi, v4, B);
    const float f0 = (sc.hK0 * (v5 * x2)) * B;

    // Eq. (4) over beta: Omega_i/beta = gamma_i L + S_j; x and y components packed
    const float g1 = fmaf(-3.0f, LS2, c.A1 * r);
    const float g2 = fmaf(-3.0f, LS1, c.A2 * r);
    const f2 O1 = pn_fma(f2(g1), y[2], y[1]);
    const f2 O2 = pn_fma(f2(g2), y[2], y[0]);
    const float O1z = fmaf(g1, Lz, S2z), O2z = fmaf(g2, Lz, S1z);
    // Eq. (2): S_i_dot = beta (Omega_i/beta) x S_i
    const float c1x = fmaf(O1.v.y, S1z, -(O1z * S1y));
    const float c1y = fmaf(O1z, S1x, -(O1.v.x * S1z));
    const float c1z = fmaf(O1.v.x, S1y, -(O1.v.y * S1x));
    const float c2x = fmaf(O2.v.y, S2z, -(O2z * S2y));
    const float c2y = fmaf(O2z, S2x, -(O2.v.x * S2z));
    const float c2z = fmaf(O2.v.x, S2y, -(O2.v.y * S2x));
    const float beta = sc.hBc * x2;
    const f2 c1(c1x, c1y), c2(c2x, c2y);
    // Eq. (3)
    const float gv = c.G * v;
    f[0] = f2(beta) * c1;
    f[1] = f2(beta) * c2;
    f[2] = f2(gv) * (f[0] + f[1]);
    const float f3 = beta * c1z, f6 = beta * c2z;
    f[3] = f2(f0, f3);
    f[4] = f2(f6, gv * (f3 + f6));
}
