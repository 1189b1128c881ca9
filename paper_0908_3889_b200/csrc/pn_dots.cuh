// pn_dots.cuh -- the unit dot products S1^.S2^, S1^.L^, S2^.L^ of one state (R14):
//     A^.B^ = (A.B) / (|A| |B|),  norms from the state itself,
// ONE routine for every kernel that bins or compares them (pn_histogram, pn_statistics, pn_selfcheck, the fused
// ensemble kernel), so the same state lands in the same bin whatever the layout, alignment or bin count.
// Every operation is an individually rounded IEEE operation (no FMA contraction, correctly rounded sqrt and divide),
// evaluated left to right: a result is a pure function of the nine inputs, reproducible by any IEEE implementation.
#pragma once
#include <cuda_runtime.h>

__device__ __forceinline__ double pn_dot3_rn(double ax, double ay, double az, double bx, double by, double bz)
{
    return __dadd_rn(__dadd_rn(__dmul_rn(ax, bx), __dmul_rn(ay, by)), __dmul_rn(az, bz));
}

// v = (S1x,S1y,S1z, S2x,S2y,S2z, Lx,Ly,Lz).  ok[k] is false where a norm is zero or the quotient is not finite
// (such a system is counted as skipped, not binned).
__device__ __forceinline__ void pn_unit_dots(const double (&v)[9], double (&d)[3], bool (&ok)[3])
{
    const double n1 = __dsqrt_rn(pn_dot3_rn(v[0], v[1], v[2], v[0], v[1], v[2]));
    const double n2 = __dsqrt_rn(pn_dot3_rn(v[3], v[4], v[5], v[3], v[4], v[5]));
    const double nl = __dsqrt_rn(pn_dot3_rn(v[6], v[7], v[8], v[6], v[7], v[8]));
    d[0] = __ddiv_rn(pn_dot3_rn(v[0], v[1], v[2], v[3], v[4], v[5]), __dmul_rn(n1, n2));
    d[1] = __ddiv_rn(pn_dot3_rn(v[0], v[1], v[2], v[6], v[7], v[8]), __dmul_rn(n1, nl));
    d[2] = __ddiv_rn(pn_dot3_rn(v[3], v[4], v[5], v[6], v[7], v[8]), __dmul_rn(n2, nl));
    ok[0] = n1 > 0.0 && n2 > 0.0 && isfinite(d[0]);
    ok[1] = n1 > 0.0 && nl > 0.0 && isfinite(d[1]);
    ok[2] = n2 > 0.0 && nl > 0.0 && isfinite(d[2]);
}

// bin = clamp(floor((d + 1) bins / 2), 0, bins - 1); d = +1 falls in the last bin (R14)
__device__ __forceinline__ int pn_bin_of(double d, int bins)
{
    const int b = (int)floor(__dmul_rn(__dmul_rn(__dadd_rn(d, 1.0), (double)bins), 0.5));
    return max(0, min(bins - 1, b));
}
