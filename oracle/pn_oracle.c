/*
 * pn_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision restatement of the hot path of arXiv:0908.3889
 * ("Integrating Post-Newtonian Equations on Graphics Processing Units"):
 *   - the right-hand side of the precessing circular-inspiral ODEs, Eqs. (1)-(4)
 *     (PAPER.md:45-60), evaluated term by term AS PRINTED (no Horner form, no hoisted
 *     constants, library cbrt/log, explicit cross products);
 *   - the Dormand-Prince 5(4) adaptive stepper the paper names, one system
 *     at a time, with every choice the paper leaves open fixed as DESIGN.md section 3
 *     lists (readings R1..R16);
 *   - the dot-product histograms of the final state.
 *
 * Only tests/, __graft_entry__.smoke() and the cpu_baseline / --impl reference legs of
 * bench.py may load this library.  It shares no code, header, table or constant with the
 * CUDA path under paper_0908_3889_b200/csrc/ and neither includes the other.
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): leading-order closed form, aligned-spin
 * quadrature of an independently retyped Eq. (1), invariants |S_i|, |L|, RHS identities,
 * 1<->2 relabelling, scale freedom, rotation covariance, tableau order conditions in exact
 * rationals, step-halving order, tolerance self-convergence, numpy histogram.
 * PARITY UNPINNED: the absolute final state of an individual precessing system is printed
 * nowhere in the paper; it is pinned only through the properties above.
 *
 * Build:  gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC pn_oracle.c -o libpn_oracle.so -lm
 * Op-count build (same source, compiled as C++ with a counting scalar):
 *         g++ -x c++ -O1 -DPN_COUNT_OPS pn_oracle.c -o pn_oracle_opcount
 *
 * State order (north_star / DESIGN.md 2): y = (omega, S1x,S1y,S1z, S2x,S2y,S2z, Lx,Ly,Lz).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifdef PN_COUNT_OPS
/* ---- counting scalar: every +,-,*,/ and every cbrt/log/sqrt/pow whose operands depend on the
 * state counts one "dynamic" flop; operations among per-system constants (masses, literals)
 * are counted separately.  Used only by the op-count executable (main() at the bottom). */
#include <cstdio>
struct real {
    double v; bool dyn;
    real() : v(0), dyn(false) {}
    real(double x) : v(x), dyn(false) {}
    real(double x, bool d) : v(x), dyn(d) {}
};
static long g_add, g_mul, g_div, g_fun, g_cadd, g_cmul, g_cdiv, g_cfun;
static inline real operator+(real a, real b) { bool d = a.dyn || b.dyn; (d ? g_add : g_cadd)++; return real(a.v + b.v, d); }
static inline real operator-(real a, real b) { bool d = a.dyn || b.dyn; (d ? g_add : g_cadd)++; return real(a.v - b.v, d); }
static inline real operator*(real a, real b) { bool d = a.dyn || b.dyn; (d ? g_mul : g_cmul)++; return real(a.v * b.v, d); }
static inline real operator/(real a, real b) { bool d = a.dyn || b.dyn; (d ? g_div : g_cdiv)++; return real(a.v / b.v, d); }
static inline real operator-(real a) { return real(-a.v, a.dyn); }
static inline real& operator+=(real& a, real b) { a = a + b; return a; }
static inline real& operator*=(real& a, real b) { a = a * b; return a; }
static inline bool operator<=(real a, real b) { return a.v <= b.v; }
static inline bool operator<(real a, real b) { return a.v < b.v; }
static inline bool operator>(real a, real b) { return a.v > b.v; }
static inline bool operator>=(real a, real b) { return a.v >= b.v; }
static inline real r_cbrt(real a) { (a.dyn ? g_fun : g_cfun)++; return real(cbrt(a.v), a.dyn); }
static inline real r_log(real a) { (a.dyn ? g_fun : g_cfun)++; return real(log(a.v), a.dyn); }
static inline real r_sqrt(real a) { (a.dyn ? g_fun : g_cfun)++; return real(sqrt(a.v), a.dyn); }
static inline real r_pow(real a, real b) { ((a.dyn || b.dyn) ? g_fun : g_cfun)++; return real(pow(a.v, b.v), a.dyn || b.dyn); }
static inline real r_fabs(real a) { return real(fabs(a.v), a.dyn); }
static inline real r_fmax(real a, real b) { return real(fmax(a.v, b.v), a.dyn || b.dyn); }
static inline real r_fmin(real a, real b) { return real(fmin(a.v, b.v), a.dyn || b.dyn); }
static inline double r_val(real a) { return a.v; }
static inline int r_finite(real a) { return std::isfinite(a.v); }
#define RC(x) real(x)
#define RDYN(x) real((x), true)
#define PN_EXPORT static
#else
typedef double real;
#define r_cbrt cbrt
#define r_log log
#define r_sqrt sqrt
#define r_pow pow
#define r_fabs fabs
#define r_fmax fmax
#define r_fmin fmin
#define r_val(a) (a)
#define r_finite(a) isfinite(a)
#define RC(x) (x)
#define RDYN(x) (x)
#define PN_EXPORT
#endif

/* Euler's constant, "gamma_E = 0.577...", reading R3 */
#define PN_GAMMA_E 0.5772156649015329
#define PN_PI 3.14159265358979323846

/* per-system failure codes written to out_steps (negative) -- same convention as include/pn.h,
 * restated here because the two libraries share no header */
#define ORC_FAIL_MAXSTEPS (-1)
#define ORC_FAIL_HUNDERFLOW (-2)
#define ORC_FAIL_NONFINITE (-3)
#define ORC_FAIL_LANDING (-4)
#define ORC_FAIL_BADINPUT (-5)

/* term mask (tests only): bit k (k = 0..7) keeps the (M omega)^{k/3} term of the brace of Eq. (1);
 * bit 16 keeps the spin-dependent pieces of Eq. (1).  0 means "everything". */
#define ORC_MASK_ALL 0x100FFu
#define ORC_MASK_SPIN (1u << 16)

static real dot3(const real a[3], const real b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

static void cross3(const real a[3], const real b[3], real c[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

/* ---------------------------------------------------------------------------------------------
 * Right-hand side f(y; m1, m2): Eqs. (1)-(4).
 * The unit-spin products of Eq. (1) are formed from S_i = chi_i m_i^2 S^_i:
 *     chi_i L^.S^_i = (L^.S_i)/m_i^2,   chi_1 chi_2 S^_1.S^_2 = (S_1.S_2)/(m_1^2 m_2^2),
 * so chi_i = 0 needs no special case.
 * ------------------------------------------------------------------------------------------- */
static void orc_rhs(const real y[10], real m1, real m2, unsigned mask, real f[10])
{
    if (mask == 0) mask = ORC_MASK_ALL;
    const real omega = y[0];
    const real *S1 = y + 1, *S2 = y + 4, *L = y + 7;

    const real M = m1 + m2;
    const real eta = m1 * m2 / (M * M);
    const real theta_hat = RC(1039.0) / RC(4620.0);
    const real pi = PN_PI, gamma_E = PN_GAMMA_E;

    const real x = M * omega;               /* (M omega) */
    const real v = r_cbrt(x);               /* (M omega)^{1/3} */
    const real x23 = v * v;                 /* (M omega)^{2/3} */
    const real x43 = x23 * x23;             /* (M omega)^{4/3} */
    const real x53 = x43 * v;               /* (M omega)^{5/3} */
    const real x2 = x * x;                  /* (M omega)^2     */
    const real x73 = x2 * v;                /* (M omega)^{7/3} */

    /* chi_i L^.S^_i and chi_1 chi_2 S^_1.S^_2 */
    const real cLS1 = dot3(L, S1) / (m1 * m1);
    const real cLS2 = dot3(L, S2) / (m2 * m2);
    const real cS1S2 = dot3(S1, S2) / ((m1 * m1) * (m2 * m2));
    const real spin_on = (mask & ORC_MASK_SPIN) ? 1.0 : 0.0;

    /* ---- Eq. (1), the brace, one printed term per statement ---- */
    real brace = 0.0;
    if (mask & (1u << 0)) brace += 1.0;
    if (mask & (1u << 2)) brace += -(RC(743.0) + RC(924.0) * eta) / RC(336.0) * x23;
    if (mask & (1u << 3)) {
        const real so = RC(1.0) / RC(12.0) *
                        (cLS1 * (RC(113.0) * m1 * m1 / (M * M) + RC(75.0) * eta) +
                         cLS2 * (RC(113.0) * m2 * m2 / (M * M) + RC(75.0) * eta));
        brace += -(spin_on * so - RC(4.0) * pi) * x;
    }
    if (mask & (1u << 4)) {
        brace += (RC(34103.0) / RC(18144.0) + RC(13661.0) / RC(2016.0) * eta +
                  RC(59.0) / RC(18.0) * eta * eta) * x43;
        brace += -spin_on * (RC(1.0) / RC(48.0)) * eta *
                 (RC(247.0) * cS1S2 - RC(721.0) * cLS1 * cLS2) * x43;
    }
    if (mask & (1u << 5)) brace += -(RC(1.0) / RC(672.0)) * (RC(4159.0) + RC(15876.0) * eta) * pi * x53;
    if (mask & (1u << 6)) {
        /* reading R1: theta_hat enters linearly in eta, (-273811877/1088640 + 451/48 pi^2 - 88/3 theta_hat) eta;
         * the printed "(... - 88/3 theta_hat eta) eta" is available as -DPN_THETA_LITERAL for comparison only */
#ifdef PN_THETA_LITERAL
        const real lin = (-RC(273811877.0) / RC(1088640.0) + RC(451.0) / RC(48.0) * pi * pi -
                          RC(88.0) / RC(3.0) * theta_hat * eta) * eta;
#else
        const real lin = (-RC(273811877.0) / RC(1088640.0) + RC(451.0) / RC(48.0) * pi * pi -
                          RC(88.0) / RC(3.0) * theta_hat) * eta;
#endif
        /* reading R2: "log" is the natural logarithm */
        brace += ((RC(16447322263.0) / RC(139708800.0) - RC(1712.0) / RC(105.0) * gamma_E +
                   RC(16.0) / RC(3.0) * pi * pi) +
                  lin + RC(541.0) / RC(896.0) * eta * eta - RC(5605.0) / RC(2592.0) * eta * eta * eta -
                  RC(856.0) / RC(105.0) * r_log(RC(16.0) * x23)) * x2;
    }
    if (mask & (1u << 7))
        brace += (-RC(4415.0) / RC(4032.0) + RC(358675.0) / RC(6048.0) * eta +
                  RC(91495.0) / RC(1512.0) * eta * eta) * pi * x73;

    f[0] = omega * omega * (RC(96.0) / RC(5.0)) * eta * x53 * brace;   /* Eq. (1) */

    /* ---- Eq. (4): Omega_1 and, by 1<->2, Omega_2 ---- */
    real Om1[3], Om2[3];
    const real pref = x2 / (RC(2.0) * M);           /* (M omega)^2 / (2M) */
    const real S2L = dot3(S2, L), S1L = dot3(S1, L);
    for (int j = 0; j < 3; ++j) {
        Om1[j] = pref * (eta / v * (RC(4.0) + RC(3.0) * m2 / m1) * L[j] +
                         RC(1.0) / (M * M) * (S2[j] - RC(3.0) * S2L * L[j]));
        Om2[j] = pref * (eta / v * (RC(4.0) + RC(3.0) * m1 / m2) * L[j] +
                         RC(1.0) / (M * M) * (S1[j] - RC(3.0) * S1L * L[j]));
    }
    /* ---- Eq. (2): dS_i/dt = Omega_i x S_i ---- */
    cross3(Om1, S1, f + 1);
    cross3(Om2, S2, f + 4);
    /* ---- Eq. (3): dL^/dt = -(M omega)^{1/3}/(eta M^2) (dS_1/dt + dS_2/dt) ---- */
    for (int j = 0; j < 3; ++j) f[7 + j] = -v / (eta * M * M) * (f[1 + j] + f[4 + j]);
}

/* ---------------------------------------------------------------------------------------------
 * Dormand-Prince 5(4) tableau (reading R5; the paper names only "the Dormand-Prince method",
 * PAPER.md:66).  Kept as integer numerators / denominators so the tests can verify the order
 * conditions in exact rational arithmetic (pin P11).
 * ------------------------------------------------------------------------------------------- */
static const long long DP_C_NUM[7] = {0, 1, 3, 4, 8, 1, 1};
static const long long DP_C_DEN[7] = {1, 5, 10, 5, 9, 1, 1};
static const long long DP_A_NUM[7][6] = {
    {0, 0, 0, 0, 0, 0},
    {1, 0, 0, 0, 0, 0},
    {3, 9, 0, 0, 0, 0},
    {44, -56, 32, 0, 0, 0},
    {19372, -25360, 64448, -212, 0, 0},
    {9017, -355, 46732, 49, -5103, 0},
    {35, 0, 500, 125, -2187, 11}};
static const long long DP_A_DEN[7][6] = {
    {1, 1, 1, 1, 1, 1},
    {5, 1, 1, 1, 1, 1},
    {40, 40, 1, 1, 1, 1},
    {45, 15, 9, 1, 1, 1},
    {6561, 2187, 6561, 729, 1, 1},
    {3168, 33, 5247, 176, 18656, 1},
    {384, 1, 1113, 192, 6784, 84}};
/* 4th-order weights b^ (7 stages); the 5th-order weights b are row 7 of A (FSAL) */
static const long long DP_BH_NUM[7] = {5179, 0, 7571, 393, -92097, 187, 1};
static const long long DP_BH_DEN[7] = {57600, 1, 16695, 640, 339200, 2100, 40};

static double dp_a(int s, int j) { return (double)DP_A_NUM[s][j] / (double)DP_A_DEN[s][j]; }
static double dp_bhat(int j) { return (double)DP_BH_NUM[j] / (double)DP_BH_DEN[j]; }
static double dp_b(int j) { return j < 6 ? dp_a(6, j) : 0.0; }

/* One trial step from (y, k1 = f(y)) with step h:  k_s = f(y + h sum_{j<s} a_sj k_j), s = 2..7;
 * y_new = the stage-7 argument (5th-order solution, local extrapolation, reading R9);
 * err = h sum_s (b_s - b^_s) k_s.  k[0] must hold k1 on entry; k[1..6] are filled. */
static void orc_trial(const real y[10], real k[7][10], real h, real m1, real m2, unsigned mask,
                      real ynew[10], real err[10])
{
    real ys[10];
    for (int s = 1; s < 7; ++s) {
        for (int c = 0; c < 10; ++c) {
            real acc = 0.0;
            for (int j = 0; j < s; ++j) acc += RC(dp_a(s, j)) * k[j][c];
            ys[c] = y[c] + h * acc;
        }
        if (s == 6) for (int c = 0; c < 10; ++c) ynew[c] = ys[c];
        orc_rhs(ys, m1, m2, mask, k[s]);
    }
    for (int c = 0; c < 10; ++c) {
        real acc = 0.0;
        for (int j = 0; j < 7; ++j) acc += RC(dp_b(j) - dp_bhat(j)) * k[j][c];
        err[c] = h * acc;
    }
}

typedef struct {
    int fixed_steps;     /* >0: exactly this many steps of size h0, no error control, no omega_f */
    double h0;           /* <=0: 10*M (reading R13) */
    int max_steps;       /* <=0: 10,000,000 */
    unsigned term_mask;  /* 0: all */
    double tau_land;     /* <=0: 1e-13 */
} orc_opts;

/* Integrate ONE system.  Returns trial-step count (>0) or a negative failure code. */
static int orc_integrate_one(const double y0[10], double m1d, double m2d, double omegaf, double rtol,
                             double atol, const orc_opts *o, double yout[10], double *tout, int *nrej)
{
    const real m1 = m1d, m2 = m2d;
    const unsigned mask = o->term_mask;
    real y[10], k[7][10], ynew[10], err[10];
    for (int c = 0; c < 10; ++c) y[c] = RDYN(y0[c]);
    double t = 0.0;
    *nrej = 0;
    const double M = m1d + m2d;
    if (!(m1d > 0.0) || !(m2d > 0.0)) { for (int c = 0; c < 10; ++c) yout[c] = y0[c]; *tout = 0; return ORC_FAIL_BADINPUT; }
    real h = (o->h0 > 0.0) ? o->h0 : 10.0 * M;
    orc_rhs(y, m1, m2, mask, k[0]);

    if (o->fixed_steps > 0) { /* reading R15: plain fixed-step DP5, y <- y_new */
        for (int n = 0; n < o->fixed_steps; ++n) {
            orc_trial(y, k, h, m1, m2, mask, ynew, err);
            for (int c = 0; c < 10; ++c) { y[c] = ynew[c]; k[0][c] = k[6][c]; }
            t += r_val(h);
        }
        for (int c = 0; c < 10; ++c) yout[c] = r_val(y[c]);
        *tout = t;
        return o->fixed_steps;
    }

    if (!(y0[0] < omegaf)) { for (int c = 0; c < 10; ++c) yout[c] = y0[c]; *tout = 0; return ORC_FAIL_BADINPUT; }

    /* error-norm scales (reading R7): atol is multiplied by the conserved norm of the vector the
     * component belongs to: 1 for omega and L^, |S_i(0)| for S_i (1 if that norm is 0) */
    double nrm[10];
    {
        double s1 = sqrt(y0[1] * y0[1] + y0[2] * y0[2] + y0[3] * y0[3]);
        double s2 = sqrt(y0[4] * y0[4] + y0[5] * y0[5] + y0[6] * y0[6]);
        if (!(s1 > 0.0)) s1 = 1.0;
        if (!(s2 > 0.0)) s2 = 1.0;
        nrm[0] = 1.0;
        for (int c = 1; c < 4; ++c) nrm[c] = s1;
        for (int c = 4; c < 7; ++c) nrm[c] = s2;
        for (int c = 7; c < 10; ++c) nrm[c] = 1.0;
    }
    const double tau = (o->tau_land > 0.0) ? o->tau_land : 1e-13;
    const int max_steps = (o->max_steps > 0) ? o->max_steps : 10000000;
    int steps = 0, n_land = 0, after_reject = 0, landing = 0;

    for (;;) {
        if (steps >= max_steps) { steps = ORC_FAIL_MAXSTEPS; break; }
        if (!(r_fabs(h) > RC(1e-300)) || t + r_val(h) == t) { steps = ORC_FAIL_HUNDERFLOW; break; }
        orc_trial(y, k, h, m1, m2, mask, ynew, err);
        ++steps;
        /* scaled RMS norm (reading R6) */
        real sum = 0.0;
        for (int c = 0; c < 10; ++c) {
            const real sc = RC(atol * nrm[c]) + RC(rtol) * r_fmax(r_fabs(y[c]), r_fabs(ynew[c]));
            const real q = err[c] / sc;
            sum += q * q;
        }
        real E = r_sqrt(sum / RC(10.0));
        if (!r_finite(E)) { steps = ORC_FAIL_NONFINITE; break; }
        if (E < RC(1e-30)) E = 1e-30;
        /* controller factor (reading R8): 0.9 E^{-1/5}, clamped */
        const real fac = RC(0.9) * r_pow(E, RC(-0.2));
        if (E <= RC(1.0)) {
            const real om_new = ynew[0];
            if (om_new > RC(omegaf * (1.0 + tau))) {
                /* reading R12: the step passes error control but overshoots omega_f: discard it and
                 * retry from the same state with a Newton update of h, using d(omega_new)/dh ~ k7[0] */
                if (++n_land > 50) { steps = ORC_FAIL_LANDING; break; }
                landing = 1;
                real hn = h - (om_new - RC(omegaf)) / k[6][0];
                if (hn < RC(0.1) * h) hn = RC(0.1) * h;
                h = hn;
                continue;
            }
            /* accept */
            t += r_val(h);
            for (int c = 0; c < 10; ++c) { y[c] = ynew[c]; k[0][c] = k[6][c]; }
            if (r_fabs(om_new - RC(omegaf)) <= RC(tau * omegaf)) break; /* landed: finish */
            n_land = 0;
            if (landing) {
                /* an accepted step that ended just short of omega_f while landing: first Newton guess
                 * from the new state, h = (omega_f - omega)/omega_dot; growth stays suspended */
                h = r_fmin(h, (RC(omegaf) - y[0]) / k[0][0]);
            } else {
                h = h * r_fmin(r_fmax(fac, RC(0.2)), after_reject ? RC(1.0) : RC(5.0));
            }
            after_reject = 0;
        } else {
            ++*nrej;
            h = h * r_fmin(r_fmax(fac, RC(0.2)), RC(1.0));
            after_reject = 1;
        }
    }
    for (int c = 0; c < 10; ++c) yout[c] = r_val(y[c]);
    *tout = t;
    return steps;
}

#ifndef PN_COUNT_OPS
/* ============================= exported C ABI of the oracle ============================== */
#ifdef _OPENMP
#include <omp.h>
#endif

/* f = RHS(y) for n states: y[n][10], masses[n][2], f[n][10] (host pointers) */
void pn_oracle_rhs(const double *y, const double *masses, long long n, unsigned term_mask, double *f)
{
    for (long long i = 0; i < n; ++i) orc_rhs(y + 10 * i, masses[2 * i], masses[2 * i + 1], term_mask, f + 10 * i);
}

/* Tableau as exact rationals: a[7][6], c[7], bhat[7] (numerators, denominators) */
void pn_oracle_tableau(long long *a_num, long long *a_den, long long *c_num, long long *c_den,
                       long long *bh_num, long long *bh_den)
{
    memcpy(a_num, DP_A_NUM, sizeof DP_A_NUM);
    memcpy(a_den, DP_A_DEN, sizeof DP_A_DEN);
    memcpy(c_num, DP_C_NUM, sizeof DP_C_NUM);
    memcpy(c_den, DP_C_DEN, sizeof DP_C_DEN);
    memcpy(bh_num, DP_BH_NUM, sizeof DP_BH_NUM);
    memcpy(bh_den, DP_BH_DEN, sizeof DP_BH_DEN);
}

/* Integrate n systems (host pointers, AoS).  out_time / out_rejected may be NULL.
 * Returns 0 if every system finished, else the number of failed systems. */
long long pn_oracle_integrate(const double *init_states, const double *masses, long long n, double omegaf,
                              double rtol, double atol, int fixed_steps, double h0, int max_steps,
                              unsigned term_mask, double tau_land, double *out_final, int *out_steps,
                              double *out_time, int *out_rejected, int n_threads)
{
    orc_opts o;
    o.fixed_steps = fixed_steps; o.h0 = h0; o.max_steps = max_steps; o.term_mask = term_mask; o.tau_land = tau_land;
    long long n_fail = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 8) reduction(+ : n_fail)
    for (long long i = 0; i < n; ++i) {
        double tf; int nrej;
        int st = orc_integrate_one(init_states + 10 * i, masses[2 * i], masses[2 * i + 1], omegaf, rtol, atol, &o,
                                   out_final + 10 * i, &tf, &nrej);
        out_steps[i] = st;
        if (out_time) out_time[i] = tf;
        if (out_rejected) out_rejected[i] = nrej;
        if (st < 0) ++n_fail;
    }
    return n_fail;
}

int pn_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Histograms of S^_1.S^_2, S^_1.L^, S^_2.L^ of n final states (reading R14):
 * d = (A.B)/(|A||B|) with all three norms taken from the state; `bins` equal bins on [-1,1],
 * bin = min(bins-1, max(0, floor((d+1)*bins/2))); systems with a zero or non-finite norm are
 * counted in n_skipped[h] instead.  counts[3][bins]; optional dots[n][3] receives d (NaN if skipped). */
void pn_oracle_histogram(const double *final_states, long long n, int bins, unsigned long long *counts,
                         unsigned long long *n_skipped, double *dots)
{
    for (int i = 0; i < 3 * bins; ++i) counts[i] = 0;
    unsigned long long skipped[3] = {0, 0, 0};
    for (long long i = 0; i < n; ++i) {
        const double *y = final_states + 10 * i;
        const double *S1 = y + 1, *S2 = y + 4, *L = y + 7;
        const double n1 = sqrt(dot3(S1, S1)), n2 = sqrt(dot3(S2, S2)), nl = sqrt(dot3(L, L));
        const double d[3] = {dot3(S1, S2) / (n1 * n2), dot3(S1, L) / (n1 * nl), dot3(S2, L) / (n2 * nl)};
        const int ok[3] = {n1 > 0 && n2 > 0, n1 > 0 && nl > 0, n2 > 0 && nl > 0};
        for (int hh = 0; hh < 3; ++hh) {
            if (!ok[hh] || !isfinite(d[hh])) {
                ++skipped[hh];
                if (dots) dots[3 * i + hh] = NAN;
                continue;
            }
            if (dots) dots[3 * i + hh] = d[hh];
            double b = floor((d[hh] + 1.0) * (double)bins / 2.0);
            int ib = (int)b;
            if (ib < 0) ib = 0;
            if (ib > bins - 1) ib = bins - 1;
            ++counts[(long long)hh * bins + ib];
        }
    }
    if (n_skipped) for (int hh = 0; hh < 3; ++hh) n_skipped[hh] = skipped[hh];
}

#else /* PN_COUNT_OPS: print the operation counts used by DESIGN.md 6 and bench.py */
int main()
{
    /* a generic system (unequal masses, misaligned spins) */
    const double y0[10] = {0.01, 0.324 * 0.8660254037844386, 0.0, 0.162, 0.096, -0.0768, 0.1024, 0.0, 0.0, 1.0};
    real y[10], f[10];
    for (int c = 0; c < 10; ++c) y[c] = real(y0[c], true);
    g_add = g_mul = g_div = g_fun = g_cadd = g_cmul = g_cdiv = g_cfun = 0;
    orc_rhs(y, real(0.6), real(0.4), 0, f);
    long rhs_dyn = g_add + g_mul + g_div + g_fun;
    std::printf("{\"rhs\": {\"add\": %ld, \"mul\": %ld, \"div\": %ld, \"fun\": %ld, \"dynamic_total\": %ld, "
                "\"constant_ops\": %ld},\n",
                g_add, g_mul, g_div, g_fun, rhs_dyn, g_cadd + g_cmul + g_cdiv + g_cfun);
    /* one whole trial step incl. norm and controller: run the adaptive loop with max_steps = 1 */
    orc_opts o; o.fixed_steps = 0; o.h0 = 0; o.max_steps = 1; o.term_mask = 0; o.tau_land = 0;
    double yout[10], tf; int nrej;
    g_add = g_mul = g_div = g_fun = g_cadd = g_cmul = g_cdiv = g_cfun = 0;
    orc_integrate_one(y0, 0.6, 0.4, 0.05, 1e-10, 1e-12, &o, yout, &tf, &nrej);
    long total = g_add + g_mul + g_div + g_fun;
    /* the loop evaluated k1 (1 RHS) + one trial (6 RHS + stage sums + error + norm + controller) */
    std::printf(" \"trial_step\": {\"add\": %ld, \"mul\": %ld, \"div\": %ld, \"fun\": %ld, "
                "\"dynamic_total_excl_seed_rhs\": %ld}}\n",
                g_add, g_mul, g_div, g_fun, total - rhs_dyn);
    return 0;
}
#endif
