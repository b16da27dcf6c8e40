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
// The gather is the only reader of a record (and, in the NVE loop, of MASK and of the own-half force), once:
// evict-first loads (ld.global.cs), so that the 65 MB of records streaming through do not push the positions,
// velocities and list rows of the next pair kernel out of the 126 MB L2 (config 2: 0.0687 -> 0.0650 ms per step,
// the fused gather 22.7 -> 19.2 us; SW 0.1895 -> 0.1821).
__device__ __forceinline__ void load_rec_once(const PairRec64* q, double* px, double* py, double* pz) {
    double a, b, c;
    [[maybe_unused]] double d;
    asm volatile("ld.global.cs.v2.f64 {%0,%1}, [%2];" : "=d"(a), "=d"(b) : "l"(q));
    asm volatile("ld.global.cs.v2.f64 {%0,%1}, [%2];" : "=d"(c), "=d"(d) : "l"(reinterpret_cast<const double2*>(q) + 1));
    *px = a; *py = b; *pz = c;
}
__device__ __forceinline__ void load_rec_once(const float4* q, float* px, float* py, float* pz) {
    float a, b, c;
    [[maybe_unused]] float d;
    asm volatile("ld.global.cs.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(a), "=f"(b), "=f"(c), "=f"(d) : "l"(q));
    *px = a; *py = b; *pz = c;
}
__device__ __forceinline__ double load_once(const double* p) {
    double v;
    asm volatile("ld.global.cs.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ unsigned long long load_once(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.global.cs.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void load_rec(const float4* q, float* px, float* py, float* pz) {
    const float4 a = *q;
    *px = a.x; *py = a.y; *pz = a.z;
}
}  // namespace rm
