// pn_f2.cuh -- two FP32 values in one 64-bit register pair, with the packed arithmetic of sm_100a
// (PTX add/mul/fma.rn.f32x2 -> SASS FADD2 / FMUL2 / FFMA2: one issue slot for two FP32 operations per lane).
// The RHS (pn_rhs.cuh) and the Dormand-Prince step (pn_dp5.cuh) are templates on the scalar type; instantiated
// with `f2` they integrate TWO independent inspirals per lane, component x of every value belonging to the lane's
// first system and component y to its second.  A scalar (a tableau coefficient, a tolerance) broadcasts: FFMA2
// takes a 32-bit register or uniform register as a splat operand, so constants cost no packing.
// Only +, -, * and fma are packed in hardware; abs / min / max and the special-function unit stay per component.
#pragma once
#include <cuda_runtime.h>

struct __align__(8) f2 {
    float2 v;
    __device__ __forceinline__ f2() {}
    __device__ __forceinline__ f2(float a, float b) { v.x = a; v.y = b; }
    __device__ __forceinline__ explicit f2(float a) { v.x = a; v.y = a; }
    __device__ __forceinline__ explicit f2(double a) { v.x = v.y = (float)a; }
    __device__ __forceinline__ explicit f2(int a) { v.x = v.y = (float)a; }
};
__device__ __forceinline__ f2 operator*(f2 a, f2 b) { f2 r; r.v = __fmul2_rn(a.v, b.v); return r; }
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { f2 r; r.v = __fadd2_rn(a.v, b.v); return r; }
__device__ __forceinline__ f2 operator-(f2 a) { return f2(-a.v.x, -a.v.y); }
__device__ __forceinline__ f2 operator-(f2 a, f2 b) { f2 r; r.v = __fadd2_rn(a.v, make_float2(-b.v.x, -b.v.y)); return r; }
__device__ __forceinline__ f2 pn_fma(f2 a, f2 b, f2 c) { f2 r; r.v = __ffma2_rn(a.v, b.v, c.v); return r; }
__device__ __forceinline__ f2 pn_abs(f2 a) { return f2(fabsf(a.v.x), fabsf(a.v.y)); }
__device__ __forceinline__ f2 pn_max(f2 a, f2 b) { return f2(fmaxf(a.v.x, b.v.x), fmaxf(a.v.y, b.v.y)); }
__device__ __forceinline__ f2 pn_min(f2 a, f2 b) { return f2(fminf(a.v.x, b.v.x), fminf(a.v.y, b.v.y)); }
// component S (0 or 1) of a packed value
template <int S> __device__ __forceinline__ float f2_get(const f2& a) { return S ? a.v.y : a.v.x; }
template <int S> __device__ __forceinline__ void f2_set(f2& a, float x) { if (S) a.v.y = x; else a.v.x = x; }
