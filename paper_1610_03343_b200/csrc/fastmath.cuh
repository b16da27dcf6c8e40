// fastmath.cuh -- branch-free FP64 elementary functions for the pair kernels.
//
// The pair kernels are bound by the FP64 pipe (64 lanes per SM: a warp-wide FP64 instruction holds the
// pipe of its SM sub-partition for two cycles), so what counts is the number of FP64 instructions and
// that the code stays one straight basic block which ptxas can interleave across an atom's neighbours.
// The CUDA library's exp/log spend 25-40 FP64 instructions each and carry range checks and slow-path
// branches.  These versions use small tables (staged in shared memory, 1.5 KB) to shorten the
// polynomials: exp 10 FP64 instructions, log 11.  Accuracy: |relative error| < 4e-16 (exp), absolute
// error < 4e-16 * max(1, |log a|) (log) -- checked on the GPU against long-double references through
// md_math_probe (tests/test_gpu_math.py).  The force tolerance is 1e-10, the energy tolerance 1e-12.
// The float overloads forward to the CUDA float functions (FP32 mode is not FP64-pipe bound).
#pragma once
#include <cuda_runtime.h>

namespace fm {

constexpr int EXP_N = 64;                        // T[j] = 2^(j/64)
constexpr int LOG_N = 64;                        // {c_j, -log c_j}, c_j ~ 1/(1 + (j + 1/2)/64)
constexpr int TAB_DOUBLES = EXP_N + 2 * LOG_N;   // layout of md_neighbors::math_tab

struct Tab {                                     // pointers into the shared-memory copy
    const double* e;
    const double2* l;
};

// Copies the tables from global to shared memory; the caller synchronises the block afterwards.
__device__ __forceinline__ Tab stage_tables(double* smem /*[TAB_DOUBLES], 16-byte aligned*/,
                                            const double* __restrict__ gtab) {
    for (int k = threadIdx.x; k < TAB_DOUBLES; k += blockDim.x) smem[k] = gtab[k];
    Tab t;
    t.e = smem;
    t.l = reinterpret_cast<const double2*>(smem + EXP_N);
    return t;
}

// 1/a: MUFU.RCP64H seed, then one cubic step y (1 + e + e^2), e = 1 - a y.  a normal, nonzero.
__device__ __forceinline__ double rcp(double a) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    const double e = __fma_rn(-a, y, 1.0);
    const double e2 = __fma_rn(e, e, e);
    return __fma_rn(y, e2, y);
}
__device__ __forceinline__ float rcp(float a) { return __frcp_rn(a); }

// 1/sqrt(a): MUFU.RSQ64H seed, then one cubic step y (1 + e/2 + 3 e^2/8), e = 1 - a y^2.
__device__ __forceinline__ double rsqrt(double a) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    const double ay = a * y;
    const double e = __fma_rn(-ay, y, 1.0);
    const double t = __fma_rn(e, 0.375, 0.5) * e;
    return __fma_rn(y, t, y);
}
__device__ __forceinline__ float rsqrt(float a) { return ::rsqrtf(a); }

// exp(x): k = round(64 x / ln 2), r = x - k ln2/64 (two parts, |r| <= 0.00542), degree-5 Taylor
// (truncation 3.5e-17), times 2^(j/64) from the table with k >> 6 added to its exponent field.
// Saturates instead of overflowing: the exponent shift is clamped to +-1020.  Domain |x| < 2e7
// (k must fit an int32); callers with unbounded arguments clamp them first.
__device__ __forceinline__ double exp(double x, const Tab& tb) {
    const double kd = __fma_rn(x, 92.33248261689366, 6755399441055744.0);     // 1.5 * 2^52
    const int k = __double2loint(kd);
    const double kf = kd - 6755399441055744.0;
    double r = __fma_rn(kf, -0.01083042469326756, x);
    r = __fma_rn(kf, -2.9815858269852933e-12, r);
    double p = __fma_rn(r, 0.008333333333333333, 0.041666666666666664);
    p = __fma_rn(p, r, 0.16666666666666666);
    p = __fma_rn(p, r, 0.5);
    p = __fma_rn(p, r, 1.0);
    p = __fma_rn(p, r, 1.0);
    const double t = tb.e[k & (EXP_N - 1)];
    const int sh = max(-1020, min(1020, k >> 6));
    const double s = __hiloint2double(__double2hiint(t) + (sh << 20), __double2loint(t));
    return s * p;
}
__device__ __forceinline__ float exp(float x, const Tab&) { return ::expf(x); }

// log(a), a positive and normal: a = 2^e m, m in [1,2), j = top 6 mantissa bits,
// r = m c_j - 1 (one FMA, |r| <= 1/128), log a = e ln2 - log c_j + log1p(r), degree-7 series.
__device__ __forceinline__ double log(double a, const Tab& tb) {
    const int hi = __double2hiint(a), lo = __double2loint(a);
    const int e = (hi >> 20) - 1023;
    const int j = (hi >> 14) & (LOG_N - 1);
    const double m = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, lo);
    const double2 cl = tb.l[j];
    const double r = __fma_rn(m, cl.x, -1.0);
    double p = __fma_rn(r, 0.14285714285714285, -0.16666666666666666);
    p = __fma_rn(p, r, 0.2);
    p = __fma_rn(p, r, -0.25);
    p = __fma_rn(p, r, 0.3333333333333333);
    p = __fma_rn(p, r, -0.5);
    // (double)e without I2F: 2^52 + 2^31 + e as a bit pattern, minus the bias
    const double ed = __hiloint2double(0x43300000, e ^ 0x80000000) - 4503601774854144.0;
    const double s = __fma_rn(ed, 0.6931471805599453, cl.y);
    return s + __fma_rn(p, r * r, r);
}
__device__ __forceinline__ float log(float a, const Tab&) { return ::logf(a); }

// sin and cos of a in [0, pi] (the cut-off window's argument): q = round(2a/pi) in {0,1,2},
// y = a - q pi/2 (two parts, |y| <= pi/4), Taylor series to y^15 / y^16.
__device__ __forceinline__ void sincos_0_pi(double a, double* sn, double* cs) {
    const double qd = __fma_rn(a, 0.6366197723675814, 6755399441055744.0);
    const int q = __double2loint(qd);
    const double qf = qd - 6755399441055744.0;
    double y = __fma_rn(qf, -1.5707963109016418, a);
    y = __fma_rn(qf, -1.5893254773528196e-08, y);
    const double y2 = y * y;
    double s = -7.647163731819816e-13;               // -1/15!
    s = __fma_rn(s, y2, 1.6059043836821613e-10);     //  1/13!
    s = __fma_rn(s, y2, -2.505210838544172e-08);     // -1/11!
    s = __fma_rn(s, y2, 2.7557319223985893e-06);     //  1/9!
    s = __fma_rn(s, y2, -0.0001984126984126984);     // -1/7!
    s = __fma_rn(s, y2, 0.008333333333333333);       //  1/5!
    s = __fma_rn(s, y2, -0.16666666666666666);       // -1/3!
    s = __fma_rn(s * y2, y, y);
    double c = 4.779477332387385e-14;                //  1/16!
    c = __fma_rn(c, y2, -1.1470745597729725e-11);    // -1/14!
    c = __fma_rn(c, y2, 2.08767569878681e-09);       //  1/12!
    c = __fma_rn(c, y2, -2.755731922398589e-07);     // -1/10!
    c = __fma_rn(c, y2, 2.48015873015873e-05);       //  1/8!
    c = __fma_rn(c, y2, -0.001388888888888889);      // -1/6!
    c = __fma_rn(c, y2, 0.041666666666666664);       //  1/4!
    c = __fma_rn(c, y2, -0.5);
    c = __fma_rn(c, y2, 1.0);
    // q = 0: (s, c); q = 1: (c, -s); q = 2: (-s, -c)
    *sn = q == 1 ? c : (q == 2 ? -s : s);
    *cs = q == 1 ? -s : (q == 2 ? -c : c);
}
__device__ __forceinline__ void sincos_0_pi(float a, float* sn, float* cs) { ::sincosf(a, sn, cs); }

// ---- N independent evaluations, written stage by stage ---------------------------------------------------
// ptxas schedules a chain of dependent FP64 instructions back to back if the source presents it that way
// (a dependent DFMA issues every 8 cycles, an independent one every 2: measured).  The thread-per-atom
// kernel has N = 4..8 independent evaluations at every step of its arithmetic (one per neighbour slot);
// these versions advance all N together, one polynomial step at a time, so consecutive instructions in
// the emitted order are independent.
template <int N>
__device__ __forceinline__ void exp_v(const double (&x)[N], double (&out)[N], const Tab& tb) {
    double kd[N], kf[N], r[N], p[N], t[N];
    int k[N];
#pragma unroll
    for (int m = 0; m < N; ++m) kd[m] = __fma_rn(x[m], 92.33248261689366, 6755399441055744.0);
#pragma unroll
    for (int m = 0; m < N; ++m) { k[m] = __double2loint(kd[m]); t[m] = tb.e[k[m] & (EXP_N - 1)]; }
#pragma unroll
    for (int m = 0; m < N; ++m) kf[m] = kd[m] - 6755399441055744.0;
#pragma unroll
    for (int m = 0; m < N; ++m) r[m] = __fma_rn(kf[m], -0.01083042469326756, x[m]);
#pragma unroll
    for (int m = 0; m < N; ++m) r[m] = __fma_rn(kf[m], -2.9815858269852933e-12, r[m]);
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = __fma_rn(r[m], 0.008333333333333333, 0.041666666666666664);
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = __fma_rn(p[m], r[m], 0.16666666666666666);
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = __fma_rn(p[m], r[m], 0.5);
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = __fma_rn(p[m], r[m], 1.0);
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = __fma_rn(p[m], r[m], 1.0);
#pragma unroll
    for (int m = 0; m < N; ++m) {
        const int sh = max(-1020, min(1020, k[m] >> 6));
        out[m] = __hiloint2double(__double2hiint(t[m]) + (sh << 20), __double2loint(t[m])) * p[m];
    }
}
template <int N>
__device__ __forceinline__ void exp_v(const float (&x)[N], float (&out)[N], const Tab&) {
#pragma unroll
    for (int m = 0; m < N; ++m) out[m] = ::expf(x[m]);
}

template <int N>
__device__ __forceinline__ void log_v(const double (&a)[N], double (&out)[N], const Tab& tb) {
    double mm[N], r[N], p[N], ed[N], cy[N];
#pragma unroll
    for (int m = 0; m < N; ++m) {
        const int hi = __double2hiint(a[m]), lo = __double2loint(a[m]);
        const int e = (hi >> 20) - 1023;
        const double2 cl = tb.l[(hi >> 14) & (LOG_N - 1)];
        mm[m] = __hiloint2double((hi & 0x000fffff) | 0x3ff00000, lo);
        ed[m] = __hiloint2double(0x43300000, e ^ 0x80000000);
        r[m] = cl.x; cy[m] = cl.y;
    }
#pragma unroll
    for (int m = 0; m < N; ++m) r[m] = __fma_rn(mm[m], r[m], -1.0);
#pragma unroll
    for (int m = 0; m < N; ++m) ed[m] = ed[m] - 4503601774854144.0;
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = __fma_rn(r[m], 0.14285714285714285, -0.16666666666666666);
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = __fma_rn(p[m], r[m], 0.2);
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = __fma_rn(p[m], r[m], -0.25);
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = __fma_rn(p[m], r[m], 0.3333333333333333);
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = __fma_rn(p[m], r[m], -0.5);
#pragma unroll
    for (int m = 0; m < N; ++m) cy[m] = __fma_rn(ed[m], 0.6931471805599453, cy[m]);
#pragma unroll
    for (int m = 0; m < N; ++m) mm[m] = r[m] * r[m];
#pragma unroll
    for (int m = 0; m < N; ++m) p[m] = __fma_rn(p[m], mm[m], r[m]);
#pragma unroll
    for (int m = 0; m < N; ++m) out[m] = cy[m] + p[m];
}
template <int N>
__device__ __forceinline__ void log_v(const float (&a)[N], float (&out)[N], const Tab&) {
#pragma unroll
    for (int m = 0; m < N; ++m) out[m] = ::logf(a[m]);
}

template <int N>
__device__ __forceinline__ void rcp_v(const double (&a)[N], double (&out)[N]) {
    double y[N], e[N];
#pragma unroll
    for (int m = 0; m < N; ++m) asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y[m]) : "d"(a[m]));
#pragma unroll
    for (int m = 0; m < N; ++m) e[m] = __fma_rn(-a[m], y[m], 1.0);
#pragma unroll
    for (int m = 0; m < N; ++m) e[m] = __fma_rn(e[m], e[m], e[m]);
#pragma unroll
    for (int m = 0; m < N; ++m) out[m] = __fma_rn(y[m], e[m], y[m]);
}
template <int N>
__device__ __forceinline__ void rcp_v(const float (&a)[N], float (&out)[N]) {
#pragma unroll
    for (int m = 0; m < N; ++m) out[m] = __frcp_rn(a[m]);
}

template <int N>
__device__ __forceinline__ void rsqrt_v(const double (&a)[N], double (&out)[N]) {
    double y[N], e[N], ay[N];
#pragma unroll
    for (int m = 0; m < N; ++m) asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y[m]) : "d"(a[m]));
#pragma unroll
    for (int m = 0; m < N; ++m) ay[m] = a[m] * y[m];
#pragma unroll
    for (int m = 0; m < N; ++m) e[m] = __fma_rn(-ay[m], y[m], 1.0);
#pragma unroll
    for (int m = 0; m < N; ++m) ay[m] = __fma_rn(e[m], 0.375, 0.5);
#pragma unroll
    for (int m = 0; m < N; ++m) e[m] = ay[m] * e[m];
#pragma unroll
    for (int m = 0; m < N; ++m) out[m] = __fma_rn(y[m], e[m], y[m]);
}
template <int N>
__device__ __forceinline__ void rsqrt_v(const float (&a)[N], float (&out)[N]) {
#pragma unroll
    for (int m = 0; m < N; ++m) out[m] = ::rsqrtf(a[m]);
}

}  // namespace fm
