// pn_gen.cuh -- the per-system arithmetic of the on-device initial-data recipe,
// shared by pn_generate (pn_gen.cu: writes state arrays) and the fused ensemble kernel (pn_integrate.cu: draws a
// system inside the work pull, no arrays), so that both produce the same bits.  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "pn_philox.cuh"

// lo + (hi - lo) u without contraction (the reference recipe rounds the product, then the sum)
__device__ __forceinline__ double gen_lerp(double lo, double hi, double u)
{
    return hi > lo ? __dadd_rn(lo, __dmul_rn(__dsub_rn(hi, lo), u)) : lo;
}
__device__ __forceinline__ void gen_unit(double uz, double uphi, double (&v)[3])
{
    const double z = __dsub_rn(__dmul_rn(2.0, uz), 1.0);
    const double phi = __dmul_rn(2.0 * 3.14159265358979323846, uphi);
    const double r = sqrt(fmax(0.0, __dsub_rn(1.0, __dmul_rn(z, z))));
    double s, c;
    sincos(phi, &s, &c);
    v[0] = __dmul_rn(r, c); v[1] = __dmul_rn(r, s); v[2] = z;
}

struct GenSpec {           // device copy of pn_ensemble
    unsigned long long key0, key1;
    double omega0, q_lo, q_hi, m1_fixed, chi1_lo, chi1_hi, chi2_lo, chi2_hi, s1_tilt_deg;
};


// the seven variates of a system -> its initial state y (omega, S1, S2, L^) and masses.  Every product and sum is an
// individually rounded IEEE operation (no contraction), as in the reference recipe.
__device__ __forceinline__ void gen_system(const GenSpec& sp, const double (&u)[7], double (&y)[10], double& m1, double& m2)
{
    const double q = gen_lerp(sp.q_lo, sp.q_hi, u[0]);
    const double chi1 = gen_lerp(sp.chi1_lo, sp.chi1_hi, u[1]);
    const double chi2 = gen_lerp(sp.chi2_lo, sp.chi2_hi, u[2]);
    double s1[3], s2[3];
    gen_unit(u[3], u[4], s1);
    gen_unit(u[5], u[6], s2);
    if (sp.m1_fixed > 0.0) { m1 = sp.m1_fixed; m2 = __dsub_rn(1.0, m1); }
    else { const double d = __dadd_rn(1.0, q); m1 = __ddiv_rn(1.0, d); m2 = __ddiv_rn(q, d); }
    if (sp.s1_tilt_deg >= 0.0) {
        const double th = __dmul_rn(sp.s1_tilt_deg, 3.14159265358979323846 / 180.0);
        sincos(th, &s1[0], &s1[2]);
        s1[1] = 0.0;
    }
    const double a1 = __dmul_rn(__dmul_rn(chi1, m1), m1), a2 = __dmul_rn(__dmul_rn(chi2, m2), m2);
    y[0] = sp.omega0;
#pragma unroll
    for (int c = 0; c < 3; ++c) { y[1 + c] = __dmul_rn(a1, s1[c]); y[4 + c] = __dmul_rn(a2, s2[c]); }
    y[7] = 0.0; y[8] = 0.0; y[9] = 1.0;
}
// system i of an ensemble of n_total systems, every variate from its own Philox block (any i, any n_total)
__device__ __forceinline__ void gen_system_at(const GenSpec& sp, unsigned long long n_total, unsigned long long i, double (&y)[10],
                                              double& m1, double& m2)
{
    double u[7];
#pragma unroll
    for (int k = 0; k < 7; ++k) u[k] = gen_uniform(sp.key0, sp.key1, (unsigned long long)k * n_total + i);
    gen_system(sp, u, y, m1, m2);
}
