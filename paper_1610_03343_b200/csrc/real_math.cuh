// real_math.cuh -- overloads that let the force kernels be written once for double and float.
#pragma once
#include "common.cuh"

namespace rm {
__device__ __forceinline__ double rsqrt(double a) { return ::rsqrt(a); }
__device__ __forceinline__ float rsqrt(float a) { return ::rsqrtf(a); }
__device__ __forceinline__ double exp(double a) { return ::exp(a); }
__device__ __forceinline__ float exp(float a) { return ::expf(a); }
__device__ __forceinline__ double log(double a) { return ::log(a); }
__device__ __forceinline__ float log(float a) { return ::logf(a); }
__device__ __forceinline__ double log1p(double a) { return ::log1p(a); }
__device__ __forceinline__ float log1p(float a) { return ::log1pf(a); }
__device__ __forceinline__ double pow(double a, double b) { return ::pow(a, b); }
__device__ __forceinline__ float pow(float a, float b) { return ::powf(a, b); }
__device__ __forceinline__ void sincos(double a, double* s, double* c) { ::sincos(a, s, c); }
__device__ __forceinline__ void sincos(float a, float* s, float* c) { ::sincosf(a, s, c); }

// one 32-byte (FP64) or 16-byte (FP32) record per directed pair.  The FP64 record moves as a single
// 256-bit access (sm_100: STG.E.ENL2.256): one DRAM sector, one instruction; the coalesced row reads of the
// gather measured faster as two 128-bit loads.
__device__ __forceinline__ void store_rec(PairRec64* q, double px, double py, double pz) {
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(q), "d"(px), "d"(py), "d"(pz), "d"(0.0) : "memory");
}
// The same record as two 128-bit stores, for code inside a non-inlined device function: ptxas 12.9 turned the
// 256-bit store above into a single 64-bit one (only Px reached memory) when the per-thread general path of round 1
// was compiled as a callee of the 128-register kernel k_tersoff_lean (seen in the SASS and as stale records on
// the GPU).  tersoff_warp_atom, today's non-inlined callee, uses this form.
__device__ __forceinline__ void store_rec_2x128(PairRec64* q, double px, double py, double pz) {
    double2* d = reinterpret_cast<double2*>(q);
    d[0] = make_double2(px, py);
    d[1] = make_double2(pz, 0.0);
}
__device__ __forceinline__ void store_rec_2x128(float4* q, float px, float py, float pz) {
    *q = make_float4(px, py, pz, 0.f);
}
__device__ __forceinline__ void store_rec(float4* q, float px, float py, float pz) {
    *q = make_float4(px, py, pz, 0.f);
}
__device__ __forceinline__ void load_rec(const PairRec64* q, double* px, double* py, double* pz) {
    const double2* d = reinterpret_cast<const double2*>(q);
    const double2 a = d[0], b = d[1];
    *px = a.x; *py = a.y; *pz = b.x;
}
__device__ __forceinline__ void load_rec(const float4* q, float* px, float* py, float* pz) {
    const float4 a = *q;
    *px = a.x; *py = a.y; *pz = a.z;
}
}  // namespace rm
