// pn_step_common.cuh -- device helpers shared by the integrator kernels (pn_integrate.cu: one system per lane in
// FP64 / FP32 / mixed; pn_integrate_packed.cu: two FP32 systems per lane with packed f32x2 arithmetic): failure
// codes, result store, the seed-record layout and its loader, special-function-unit wrappers.
#pragma once
#include <cfloat>
#include "pn_dp5.cuh"
#include "pn_internal.h"

#define PN_ST_EINVAL 1
#define PN_ST_ENOTCONVERGED 3
#define PN_ST_ENONFINITE 4
#define PN_F_MAXSTEPS (-1)
#define PN_F_HUNDERFLOW (-2)
#define PN_F_NONFINITE (-3)
#define PN_F_LANDING (-4)
#define PN_F_BADINPUT (-5)

template <typename real> struct PnLimits;
template <> struct PnLimits<double> { static __device__ double tiny() { return 1e-300; } static __device__ double huge() { return DBL_MAX; } };
template <> struct PnLimits<float> { static __device__ float tiny() { return 1e-30f; } static __device__ float huge() { return FLT_MAX; } };

template <typename real> struct PnVec;
template <> struct PnVec<double> {
    typedef double2 type;
    static __device__ __forceinline__ double2 make(const double* a) { return make_double2(a[0], a[1]); }
    static __device__ __forceinline__ void unpack(double2 v, double* a) { a[0] = v.x; a[1] = v.y; }
};
template <> struct PnVec<float> {
    typedef float4 type;
    static __device__ __forceinline__ float4 make(const float* a) { return make_float4(a[0], a[1], a[2], a[3]); }
    static __device__ __forceinline__ void unpack(float4 v, float* a) { a[0] = v.x; a[1] = v.y; a[2] = v.z; a[3] = v.w; }
};

// 0.9 * E^{-1/5} (controller, DESIGN.md 3 R8).  Evaluated with the FP32 special-function unit in both
// precisions: the factor only sets the next trial's step size, 1e-6 relative accuracy is ample and
// it keeps ~100 instructions per trial step off the FP64 pipe.
// argument: E^2 = mean_j (err_j/sc_j)^2, so the factor is 0.9 (E^2)^{-1/10}; no square root needed.
__device__ __forceinline__ float pn_ctrl_factor(float E2) { return 0.9f * exp2f(-0.1f * __log2f(E2)); }

// err/sc for the error norm: MUFU reciprocal seed (rcp.approx.ftz.f64, ~2^-23) + one Newton step gives
// ~1.4e-14 relative accuracy with 3 FP64-pipe instructions and no slow-path branch (an IEEE divide is ~10).
__device__ __forceinline__ double pn_ratio(double a, double b)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));
    r = fma(fma(-b, r, 1.0), r, r);
    return a * r;
}
__device__ __forceinline__ float pn_ratio(float a, float b) { return __fdividef(a, b); }

template <typename real>
__device__ __forceinline__ void pn_store_result(const PnKernelParams& p, int idx, const real (&y)[10], int code,
                                                double t, int nrej)
{
#pragma unroll
    for (int i = 0; i < 10; ++i) p.yf[(size_t)i * p.n + idx] = (double)y[i];
    p.steps[idx] = code;
    if (p.time) p.time[idx] = t;
    if (p.rejected) p.rejected[idx] = nrej;
}

// FP32 helpers without the denormal-range fix-up code the CUDA intrinsics carry (inputs are clamped).
__device__ __forceinline__ float pn_rcp_f(float a) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
__device__ __forceinline__ float pn_lg2_f(float a) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }
__device__ __forceinline__ float pn_ex2_f(float a) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a)); return r; }

// Seed record of one system (written by pn_seed_kernel, pn_integrate.cu): PN_REC reals of the launch precision
//   [0..9] y0   [10..19] K1 = h0 f(y0)   [20..34] PnConsts   [35..37] PnBase   [38] atol |S1|   [39] atol |S2|
// A record with [38] < 0 marks a system the seed kernel has already failed (bad input).
#define PN_REC 40
template <typename real>
__device__ __forceinline__ void pn_load_record(const void* seed, int i, real (&out)[PN_REC])
{
    using vec = typename PnVec<real>::type;
    constexpr int W = 16 / (int)sizeof(real);
    const vec* src = (const vec*)((const real*)seed + (size_t)i * PN_REC);
#pragma unroll
    for (int j = 0; j < PN_REC / W; ++j) PnVec<real>::unpack(__ldg(src + j), &out[j * W]);
}

