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
// A task is one (slot m, atom t) of the CTA's list rows; consecutive threads take consecutive atoms, so a
// warp reads 128 contiguous bytes of a list row.  Each thread owns up to TPT tasks and keeps their geometry
// in registers: all its list entries are fetched first, then all neighbour coordinates (two dependent
// memory levels for the whole stage, not two per task), and the dense entries are written from registers
// once the prefix sum has placed them.  KL = longest list row the CTA can hold (rows beyond it latch
// MD_DEV_INRANGE_OVERFLOW).
template <class T, int TA, int PC, int KL>
__device__ __forceinline__ void
compact_in_range(Dense<T, TA, PC>& d, int64_t A0, int na, int64_t n, int K,
                 const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
                 double Lx, double Ly, double Lz, const int32_t* __restrict__ NN,
                 const int32_t* __restrict__ NL, T range2, int* __restrict__ status) {
    constexpr int TPT = (KL * TA + NT - 1) / NT;
    const int tid = threadIdx.x;
    const double hx = 0.5 * Lx, hy = 0.5 * Ly, hz = 0.5 * Lz;
    for (int t = tid; t < TA; t += NT) {
        d.mask[t] = 0ull;
        const int nn = t < na ? NN[A0 + t] : 0;
        if (nn > KL) atomicOr(&status[0], MD_DEV_INRANGE_OVERFLOW);
        d.nn[t] = nn < KL ? nn : KL;
    }
    __syncthreads();
    int jj[TPT];
    T tx[TPT], ty[TPT], tz[TPT];
    bool in[TPT];
#pragma unroll
    for (int u = 0; u < TPT; ++u) {                          // level 1: list entries
        const int q = tid + u * NT;
        const int m = q / TA, t = q - m * TA;
        in[u] = m < KL && m < d.nn[t];
        jj[u] = in[u] ? NL[(int64_t)m * n + A0 + t] : (int)(A0 + (t < na ? t : 0));   // always a valid atom
    }
#pragma unroll
    for (int u = 0; u < TPT; ++u) {                          // level 2: coordinates
        const int q = tid + u * NT;
        const int t = q % TA;
        const int64_t i = A0 + (t < na ? t : 0);
        tx[u] = (T)md_min_image(x[jj[u]] - x[i], Lx, hx);
        ty[u] = (T)md_min_image(y[jj[u]] - y[i], Ly, hy);
        tz[u] = (T)md_min_image(z[jj[u]] - z[i], Lz, hz);
    }
#pragma unroll
    for (int u = 0; u < TPT; ++u) {
        const int q = tid + u * NT;
        const int m = q / TA, t = q - m * TA;
        in[u] = in[u] && tx[u] * tx[u] + ty[u] * ty[u] + tz[u] * tz[u] < range2;
        if (in[u]) atomicOr(&d.mask[t], 1ull << m);
    }
    __syncthreads();
    // exclusive scan of the per-atom counts (TA <= NT)
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
    // dense entries, from registers
#pragma unroll
    for (int u = 0; u < TPT; ++u) {
        if (!in[u]) continue;
        const int q = tid + u * NT;
        const int m = q / TA, t = q - m * TA;
        const int k = d.off[t] + __popcll(d.mask[t] & ((1ull << m) - 1ull));
        if (k < PC) {
            d.j[k] = jj[u];
            d.tm[k] = (unsigned short)(t * 64 + m);
            d.ex[k] = tx[u]; d.ey[k] = ty[u]; d.ez[k] = tz[u];
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
