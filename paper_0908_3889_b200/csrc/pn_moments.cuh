// pn_moments.cuh -- bivariate sample moments (n, xbar, ybar, M2x, M2y, Cxy) and their pairwise merge, shared by
// pn_statistics (pn_stats.cu) and the fused ensemble kernel (pn_integrate.cu).  r = Cxy / sqrt(M2x M2y) (R18).
#pragma once
#include <cuda_runtime.h>

// ---- moments ----------------------------------------------------------------------------------------------
struct StMom { double n, mx, my, m2x, m2y, cxy; };

// Chan et al. pairwise update: merge b into a
__device__ __forceinline__ void st_merge(StMom& a, const StMom& b)
{
    const double n = a.n + b.n;
    if (n == 0.0) return;
    const double dx = b.mx - a.mx, dy = b.my - a.my;
    const double w = a.n * b.n / n, f = b.n / n;
    a.m2x += b.m2x + dx * dx * w;
    a.m2y += b.m2y + dy * dy * w;
    a.cxy += b.cxy + dx * dy * w;
    a.mx = (b.n == 0.0) ? a.mx : ((a.n == 0.0) ? b.mx : a.mx + dx * f);
    a.my = (b.n == 0.0) ? a.my : ((a.n == 0.0) ? b.my : a.my + dy * f);
    a.n = n;
}
__device__ __forceinline__ StMom st_shfl_xor(const StMom& a, int o)
{
    StMom r;
    r.n = __shfl_xor_sync(0xffffffffu, a.n, o);
    r.mx = __shfl_xor_sync(0xffffffffu, a.mx, o);
    r.my = __shfl_xor_sync(0xffffffffu, a.my, o);
    r.m2x = __shfl_xor_sync(0xffffffffu, a.m2x, o);
    r.m2y = __shfl_xor_sync(0xffffffffu, a.m2y, o);
    r.cxy = __shfl_xor_sync(0xffffffffu, a.cxy, o);
    return r;
}

// one more sample (Welford's update): exact zero variance for constant data
__device__ __forceinline__ void st_add(StMom& a, double x, double y)
{
    a.n += 1.0;
    const double dx = x - a.mx, dy = y - a.my;
    a.mx += dx / a.n; a.my += dy / a.n;
    a.m2x += dx * (x - a.mx);
    a.m2y += dy * (y - a.my);
    a.cxy += dx * (y - a.my);
}
