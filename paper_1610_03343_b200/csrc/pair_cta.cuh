// pair_cta.cuh -- "lanes = pairs" skeleton shared by the Tersoff and SW pair kernels.
//
// A CTA owns TA consecutive atoms.  Stage A compacts the in-range directed pairs of those atoms into a
// dense list in shared memory (per-atom bit masks -> prefix sum -> dense slots), so that the expensive
// per-pair arithmetic and the triplet loops run with one thread per in-range pair: no idle lanes for
// listed-but-out-of-range neighbours (SW: 16 listed, 6 in range) and no warp divergence from rows of
// different length beyond the trip count of the inner loop.
#pragma once
#include "common.cuh"
#include "real_math.cuh"

namespace pc {

constexpr int NT = 256;          // threads per CTA

template <class T, int TA, int PC>
struct Dense {                   // shared-memory image of the CTA's in-range pairs
    unsigned long long mask[TA]; // bit m: slot m of the atom's list row is inside the force range
    int off[TA + 1];             // dense range of atom t: [off[t], off[t+1])
    int nn[TA];
    int j[PC];                   // neighbour index
    unsigned short tm[PC];       // t * 64 + m
    T ex[PC], ey[PC], ez[PC];    // first r_ij (raw), then the unit vector e_ij
    int scan_tmp[32];
    int np;                      // number of dense pairs
};

// Stage A.  Returns after a __syncthreads(); d.np = number of dense pairs (clamped to PC).
template <class T, int TA, int PC>
__device__ __forceinline__ void
compact_in_range(Dense<T, TA, PC>& d, int64_t A0, int na, int64_t n, int K,
                 const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
                 double Lx, double Ly, double Lz, const int32_t* __restrict__ NN,
                 const int32_t* __restrict__ NL, T range2, int* __restrict__ status) {
    const int tid = threadIdx.x;
    const double hx = 0.5 * Lx, hy = 0.5 * Ly, hz = 0.5 * Lz;
    for (int t = tid; t < TA; t += NT) {
        d.mask[t] = 0ull;
        d.nn[t] = t < na ? NN[A0 + t] : 0;
    }
    __syncthreads();
    // A1: one task per (slot m, atom t); consecutive threads -> consecutive atoms (coalesced NL rows)
    int kmax = 0;
    for (int t = 0; t < TA; ++t) kmax = max(kmax, d.nn[t]);          // smem broadcast reads
    for (int q = tid; q < kmax * TA; q += NT) {
        const int m = q / TA, t = q - m * TA;
        if (m < d.nn[t]) {
            const int64_t i = A0 + t;
            const int jj = NL[(int64_t)m * n + i];
            const T tx = (T)md_min_image(x[jj] - x[i], Lx, hx);
            const T ty = (T)md_min_image(y[jj] - y[i], Ly, hy);
            const T tz = (T)md_min_image(z[jj] - z[i], Lz, hz);
            if (tx * tx + ty * ty + tz * tz < range2) atomicOr(&d.mask[t], 1ull << m);
        }
    }
    __syncthreads();
    // A2: exclusive scan of the per-atom counts (TA <= NT)
    {
        const int c = tid < TA ? __popcll(d.mask[tid]) : 0;
        int inc = c;
        const int lane = tid & 31, wid = tid >> 5;
#pragma unroll
        for (int s = 1; s < 32; s <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, inc, s);
            if (lane >= s) inc += v;
        }
        if (lane == 31) d.scan_tmp[wid] = inc;
        __syncthreads();
        if (wid == 0) {
            int s2 = lane < NT / 32 ? d.scan_tmp[lane] : 0;
#pragma unroll
            for (int s = 1; s < 32; s <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, s2, s);
                if (lane >= s) s2 += v;
            }
            d.scan_tmp[lane] = s2;
        }
        __syncthreads();
        const int base = wid ? d.scan_tmp[wid - 1] : 0;
        if (tid < TA) d.off[tid] = base + inc - c;
        if (tid == TA - 1) {
            int total = base + inc;
            if (total > PC) { atomicOr(&status[0], MD_DEV_INRANGE_OVERFLOW); total = PC; }
            d.off[TA] = total;
            d.np = total;
        }
    }
    __syncthreads();
    // A3: write the dense entries (geometry recomputed: L1-resident)
    for (int q = tid; q < kmax * TA; q += NT) {
        const int m = q / TA, t = q - m * TA;
        const unsigned long long mk = d.mask[t];
        if (mk >> m & 1ull) {
            const int k = d.off[t] + __popcll(mk & ((1ull << m) - 1ull));
            if (k < PC) {
                const int64_t i = A0 + t;
                const int jj = NL[(int64_t)m * n + i];
                d.j[k] = jj;
                d.tm[k] = (unsigned short)(t * 64 + m);
                d.ex[k] = (T)md_min_image(x[jj] - x[i], Lx, hx);
                d.ey[k] = (T)md_min_image(y[jj] - y[i], Ly, hy);
                d.ez[k] = (T)md_min_image(z[jj] - z[i], Lz, hz);
            }
        }
    }
    __syncthreads();
}

// 1/a by MUFU.RCP64H + two Newton steps (4 DFMA): full double accuracy for normal a.
__device__ __forceinline__ double fast_rcp(double a) {
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double e = __fma_rn(-a, y, 1.0);
    y = __fma_rn(y, e, y);
    e = __fma_rn(-a, y, 1.0);
    return __fma_rn(y, e, y);
}
__device__ __forceinline__ float fast_rcp(float a) { return __frcp_rn(a); }

}  // namespace pc
