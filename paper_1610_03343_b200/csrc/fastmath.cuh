// fastmath.cuh -- branch-free FP64 elementary functions for the pair kernels.
//
// The pair kernels are bound by the FP64 pipe and by the latency of dependent DFMA chains.  The CUDA
// library's exp/log carry range checks and slow-path branches that split basic blocks and stop ptxas
// from interleaving the independent chains of an atom's neighbours.  These versions are straight-line
// code valid on the ranges the potentials produce (stated per function); accuracy ~1-2 ulp, checked in
// tests/test_gpu_math.py against mpmath.  The float overloads forward to the CUDA float functions.
#pragma once
#include <cuda_runtime.h>

namespace fm {

// 1/a: MUFU.RCP64H seed + two Newton steps.  a normal, nonzero.
__device__ __forceinline__ double rcp(double a) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double e = __fma_rn(-a, y, 1.0);
    y = __fma_rn(y, e, y);
    e = __fma_rn(-a, y, 1.0);
    return __fma_rn(y, e, y);
}
__device__ __forceinline__ float rcp(float a) { return __frcp_rn(a); }

// 1/sqrt(a): MUFU.RSQ64H seed + two Newton steps.  a normal, positive.
__device__ __forceinline__ double rsqrt(double a) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double h = 0.5 * y;
    double e = __fma_rn(-a * y, y, 1.0);
    y = __fma_rn(h, e, y);
    h = 0.5 * y;
    e = __fma_rn(-a * y, y, 1.0);
    return __fma_rn(h, e, y);
}
__device__ __forceinline__ float rsqrt(float a) { return ::rsqrtf(a); }

// exp(x) for x clamped to [-700, 700]: k = round(x/ln2), r = x - k ln2 (two-part), degree-13 Taylor
// (|r| <= 0.3466: truncation 4e-18), scaled by adding k to the exponent field.
__device__ __forceinline__ double exp(double x) {
    x = fmin(fmax(x, -700.0), 700.0);
    const double kd = __fma_rn(x, 1.4426950408889634, 6755399441055744.0);       // 1.5 * 2^52 trick
    const int k = __double2loint(kd);
    const double kf = kd - 6755399441055744.0;
    double r = __fma_rn(-kf, 0.6931471803691238, x);
    r = __fma_rn(-kf, 1.9082149292705877e-10, r);
    double p = 1.6059043836821613e-10;
    p = __fma_rn(p, r, 2.08767569878681e-09);
    p = __fma_rn(p, r, 2.505210838544172e-08);
    p = __fma_rn(p, r, 2.755731922398589e-07);
    p = __fma_rn(p, r, 2.7557319223985893e-06);
    p = __fma_rn(p, r, 2.48015873015873e-05);
    p = __fma_rn(p, r, 0.0001984126984126984);
    p = __fma_rn(p, r, 0.001388888888888889);
    p = __fma_rn(p, r, 0.008333333333333333);
    p = __fma_rn(p, r, 0.041666666666666664);
    p = __fma_rn(p, r, 0.16666666666666666);
    p = __fma_rn(p, r, 0.5);
    p = __fma_rn(p, r, 1.0);
    p = __fma_rn(p, r, 1.0);
    // p in [0.70, 1.42]; 2^k with |k| <= 1010 split in two exact power-of-two multiplies
    const int k1 = k >> 1, k2 = k - k1;
    const double s1 = __hiloint2double((k1 + 1023) << 20, 0);
    const double s2 = __hiloint2double((k2 + 1023) << 20, 0);
    return p * s1 * s2;
}
__device__ __forceinline__ float exp(float x) { return ::expf(x); }

// log(a) for a positive and normal: a = 2^e m, m in [sqrt(1/2), sqrt(2)); f = (m-1)/(m+1);
// log m = 2 atanh f = 2f (1 + f^2/3 + ... + f^22/23), |f| <= 0.1716 (truncation 2e-19 relative).
__device__ __forceinline__ double log(double a) {
    int hi = __double2hiint(a);
    const int lo = __double2loint(a);
    int e = (hi >> 20) - 1023;
    hi = (hi & 0x000fffff) | 0x3ff00000;                  // m in [1, 2)
    double m = __hiloint2double(hi, lo);
    if (m > 1.4142135623730951) { m *= 0.5; e += 1; }     // select, not a branch
    const double f = (m - 1.0) * rcp(m + 1.0);
    const double f2 = f * f;
    double p = 0.08695652173913043;
    p = __fma_rn(p, f2, 0.09523809523809523);
    p = __fma_rn(p, f2, 0.10526315789473684);
    p = __fma_rn(p, f2, 0.11764705882352941);
    p = __fma_rn(p, f2, 0.13333333333333333);
    p = __fma_rn(p, f2, 0.15384615384615385);
    p = __fma_rn(p, f2, 0.18181818181818182);
    p = __fma_rn(p, f2, 0.2222222222222222);
    p = __fma_rn(p, f2, 0.2857142857142857);
    p = __fma_rn(p, f2, 0.4);
    p = __fma_rn(p, f2, 0.6666666666666666);
    // log m = 2f + f * f2 * p
    const double ed = (double)e;
    const double t = __fma_rn(f * f2, p, ed * 1.9082149292705877e-10);
    return __fma_rn(ed, 0.6931471803691238, __fma_rn(2.0, f, t));
}
__device__ __forceinline__ float log(float a) { return ::logf(a); }

// log(1 + t) for t >= 0 (and 1 + t normal): log(u) + (t - (u - 1))/u with u = fl(1 + t).
__device__ __forceinline__ double log1p(double t) {
    const double u = 1.0 + t;
    const double c = (t - (u - 1.0)) * rcp(u);
    return log(u) + c;
}
__device__ __forceinline__ float log1p(float t) { return ::log1pf(t); }

}  // namespace fm
