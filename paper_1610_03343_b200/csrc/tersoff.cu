// tersoff.cu -- per-pair kernel for the Tersoff potential (steps B1 + B2 of DESIGN.md).
//
// One thread per atom i.  For every listed neighbour inside the force range S it computes the
// bond order zeta_ij, b_ij, b'_ij (Eqs. 3-6; Algorithm 3) and the
// partial derivative P_ij = dU_i/dr_ij (Eq. 14; explicit form: DESIGN.md T5), then
//   * pushes P_ij into the record slot of atom j that the gather kernel of j reads
//     (Q[rev(i,m)*n + j]; exactly one writer per slot, no atomics),
//   * accumulates the "own" halves  sum_j P_ij  and  -1/2 sum_j r_ij (x) P_ij  and U_i.
// T = double (MD_FP64) or float (MD_FP32: r_ij formed in double, then rounded; reading A10).
#include <algorithm>
#include <cstdlib>

#include "common.cuh"
#include "real_math.cuh"
#include "pair_sort.cuh"
#include "fastmath.cuh"

namespace {

template <class T>
struct TersoffDev {
    T A, B, lambda, mu, beta, n, h, R, S2;
    T c2, d2, c2_over_d2;     // c^2, d^2, c^2/d^2
    T w;                      // pi / (S - R)
    T minus_half_over_n;      // -1/(2n)
};

// Multi-element form (reading A17): per-pair mixed parameters and per-centre parameters.  NT = 1 is the
// single-element potential (every index folds to 0 at compile time).
template <class T> struct TsPair { T A, B, lambda, mu, R, w, chi; };     // w = pi / (S - R); B carries no chi
template <class T> struct TsCenter { T beta, n, h, c2, d2, c2_over_d2, minus_half_over_n; };
template <class T, int NT> struct TersoffTab { TsCenter<T> c[NT]; TsPair<T> p[NT * NT]; };

// Validation build (-DMD_TERSOFF_ALL_GENERAL=true through MD_NVCC_EXTRA): every atom of the crystal kernels takes
// the warp-per-atom general path, so the full-size parity tests exercise it on all 512 000 atoms, not on the
// handful that need it (done once per change of that path; profiles/r02_general_path_validation.md).
#ifndef MD_TERSOFF_ALL_GENERAL
#define MD_TERSOFF_ALL_GENERAL false
#endif
#ifndef MD_TERSOFF_LEAN_BT
#define MD_TERSOFF_LEAN_BT 128
#endif
#ifndef MD_TERSOFF_LEAN_MAXREG
#define MD_TERSOFF_LEAN_MAXREG 128   // 4 CTAs of 128 threads per SM
#endif

// General path, one WARP per atom: list rows of any length (up to 64 listed, 32 in range) and pairs inside the
// cut-off window.  The register kernels hand it the few atoms their straight-line bodies do not cover.  Such an
// atom used to be finished by its own thread alone (per-thread arrays in local memory, ~2500 dependent
// instructions: one 8 us straggler held an SM long after the other 147 had finished a 35 us kernel -- ncu
// l1tex__cycles_active min/avg/max, profiles/r02b).  Here the lanes of a warp are the atom's in-range slots:
//   screen   lane l tests list entries l and l + 32; the in-range ones are compacted to lanes 0..M-1 through a
//            per-warp shared-memory scratch (ballot + popc ranks);
//   pass 1   lane a: e_a, 1/r_a, f_C, f_C', f_R, f_A of its slot;
//   pass 2   lane a: zeta_a = sum_{b != a} f_C(r_b) g_ab with slot b's data fetched by shuffles; b, b', D_a, h_a;
//   pass 3   lane a: P_a (T5) likewise, stored to Q[rev(i,a) * n + j_a]; U_i and the own halves by a shuffle tree.
// Called by all 32 lanes of a warp (converged).  Records are stored as 2 x 128 bit (real_math.cuh).
struct WarpSlots { double dx[32], dy[32], dz[32]; int j[32], m[32]; };

template <class T>
__device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

template <class T, class Rec>
__device__ __noinline__ void
tersoff_warp_atom(int64_t i, int64_t n, const double* x, const double* y, const double* z, double Lx, double Ly,
                  double Lz, const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
                  const uint8_t* __restrict__ REV, const TersoffDev<T>& p, const double* tab_smem, Rec* __restrict__ Q,
                  unsigned long long* __restrict__ MASK, double* __restrict__ pe, double* __restrict__ f,
                  double* __restrict__ virial, int* __restrict__ status, WarpSlots& ws) {
    fm::Tab tb;
    tb.e = tab_smem;
    tb.l = reinterpret_cast<const double2*>(tab_smem + fm::EXP_N);
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    const ps::MinImage mi = ps::make_min_image(Lx, Ly, Lz);
    const int nn = min(NN[i], 64);
    const double xi = x[i], yi = y[i], zi = z[i];
    // screen and compaction
    bool in[2];
    double qx[2], qy[2], qz[2];
    int jj[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int m = lane + 32 * h;
        const bool valid = m < nn;
        jj[h] = valid ? NL[(int64_t)m * n + i] : (int)i;
        qx[h] = x[jj[h]] - xi; qy[h] = y[jj[h]] - yi; qz[h] = z[jj[h]] - zi;
        mi.wrap(qx[h], qy[h], qz[h]);
        in[h] = valid && ps::in_range_d2((T)qx[h], (T)qy[h], (T)qz[h]) < p.S2;
    }
    const unsigned lo = __ballot_sync(0xffffffffu, in[0]), hi = __ballot_sync(0xffffffffu, in[1]);
    int M = __popc(lo) + __popc(hi);
    if (M > 32) { if (lane == 0) atomicOr(&status[0], MD_DEV_INRANGE_OVERFLOW); M = 32; }
    __syncwarp();
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int rank = h == 0 ? __popc(lo & lt) : __popc(lo) + __popc(hi & lt);
        if (in[h] && rank < 32) {
            ws.dx[rank] = qx[h]; ws.dy[rank] = qy[h]; ws.dz[rank] = qz[h];
            ws.j[rank] = jj[h]; ws.m[rank] = lane + 32 * h;
        }
    }
    __syncwarp();
    const bool act = lane < M;
    // pass 1 (an idle lane computes on a unit vector and carries f_C = f_R = f_A = 0)
    const T tx = act ? (T)ws.dx[lane] : T(1), ty = act ? (T)ws.dy[lane] : T(0), tz = act ? (T)ws.dz[lane] : T(0);
    const int ja = act ? ws.j[lane] : 0, ma = act ? ws.m[lane] : 0;
    const T d2 = ps::in_range_d2(tx, ty, tz);
    const T rinv = fm::rsqrt(d2);
    const T r = d2 * rinv;
    const T ex = tx * rinv, ey = ty * rinv, ez = tz * rinv;
    T fc = act ? T(1) : T(0), fcp = T(0);
    if (act && r > p.R) {                                    // f_C window R < r < S (reading A1)
        T sn, cs;
        fm::sincos_0_pi((r - p.R) * p.w, &sn, &cs);
        fc = T(0.5) + T(0.5) * cs;
        fcp = T(-0.5) * p.w * sn;
    }
    const T fR = act ? p.A * fm::exp(-p.lambda * r, tb) : T(0);
    const T fA = act ? p.B * fm::exp(-p.mu * r, tb) : T(0);
    // pass 2: zeta (Eq. 4), g = 1 + (c/d)^2 x^2/(d^2 + x^2), x = h - cos (Eq. 5 without its cancellation)
    T zt = T(0);
    for (int b = 0; b < M; ++b) {
        const T bx = __shfl_sync(0xffffffffu, ex, b), by = __shfl_sync(0xffffffffu, ey, b),
                bz = __shfl_sync(0xffffffffu, ez, b), fcb = __shfl_sync(0xffffffffu, fc, b);
        const T xx = p.h - (ex * bx + ey * by + ez * bz);
        const T x2 = xx * xx;
        const T g = T(1) + p.c2_over_d2 * x2 * fm::rcp(p.d2 + x2);
        zt += b != lane ? fcb * g : T(0);
    }
    T bo = T(1), bp = T(0);
    if (zt > T(0)) {                                         // zeta = 0: b = 1, b' = 0 (reading A8)
        const T tt = fm::exp(p.n * fm::log(p.beta * zt, tb), tb);                 // (beta zeta)^n
        bo = fm::exp(p.minus_half_over_n * fm::log(T(1) + tt, tb), tb);           // Eq. (3)
        bp = T(-0.5) * bo * tt * fm::rcp(zt * (T(1) + tt));
    }
    const T bfA = bo * fA;
    T U = T(0.5) * fc * (fR - bfA);                                               // U_ia / 2
    const T D = T(0.5) * (fcp * (fR - bfA) + fc * (p.mu * bfA - p.lambda * fR));
    const T hh = T(-0.5) * fc * fA * bp;
    // pass 3: P_a = D_a e_a + sum_{b != a} [ (h_a fc_b + h_b fc_a) g' (e_b - cos e_a)/r_a + h_b fc'_a g e_a ]
    T ce = D, sx = T(0), sy = T(0), sz = T(0);
    for (int b = 0; b < M; ++b) {
        const T bx = __shfl_sync(0xffffffffu, ex, b), by = __shfl_sync(0xffffffffu, ey, b),
                bz = __shfl_sync(0xffffffffu, ez, b), fcb = __shfl_sync(0xffffffffu, fc, b),
                hb = __shfl_sync(0xffffffffu, hh, b);
        const T cs = ex * bx + ey * by + ez * bz;
        const T xx = p.h - cs;
        const T x2 = xx * xx;
        const T q = fm::rcp(p.d2 + x2);
        const T gp = T(-2) * p.c2 * xx * q * q;              // dg/dcos
        const T ta = b != lane ? (hh * fcb + hb * fc) * gp * rinv : T(0);
        ce += b != lane ? hb * fcp * (T(1) + p.c2_over_d2 * x2 * q) - ta * cs : T(0);
        sx += ta * bx; sy += ta * by; sz += ta * bz;
    }
    T px = sx + ce * ex, py = sy + ce * ey, pz = sz + ce * ez;
    if (act) {
        const int rev = (int)REV[(int64_t)ma * n + i];
        rm::store_rec_2x128(&Q[(int64_t)rev * n + ja], px, py, pz);
    } else {
        px = T(0); py = T(0); pz = T(0); U = T(0);
    }
    // U_i and the own halves: shuffle tree (fixed order)
    const T Us = warp_sum(U), Fx = warp_sum(px), Fy = warp_sum(py), Fz = warp_sum(pz);
    if (virial) {
        const T rr = fm::rcp(rinv);
        const T rx = ex * rr, ry = ey * rr, rz = ez * rr;
        const T w[9] = {rx * px, rx * py, rx * pz, ry * px, ry * py, ry * pz, rz * px, rz * py, rz * pz};
#pragma unroll
        for (int k = 0; k < 9; ++k) {
            const T ws9 = warp_sum(w[k]);
            if (lane == 0) virial[(int64_t)k * n + i] = (double)(T(-0.5) * ws9);
        }
    }
    if (lane == 0) {
        MASK[i] = (unsigned long long)lo | ((unsigned long long)hi << 32);
        if (pe) pe[i] = (double)Us;
        if (f) { f[i] = (double)Fx; f[n + i] = (double)Fy; f[2 * n + i] = (double)Fz; }
    }
    __syncwarp();                                            // the scratch may be reused by the caller's next atom
}

// The CTA's atoms that need the general path are queued (a shared-memory counter; the order in the queue does
// not influence any result) and, after a barrier, taken one per warp.
template <class T, int BT>
struct SlowQueue {
    WarpSlots ws[BT / 32];
    TersoffDev<T> p;          // the kernel's parameter block: handed to the non-inlined general path by address (as a
    int atom[BT];             // by-value or by-reference argument every thread spilled its 112 bytes to local memory
    int count;                // before the call, whether or not the queue held anything)
};

template <class T, class Rec, int BT>
__device__ __forceinline__ void
tersoff_drain_queue(SlowQueue<T, BT>& sq, int64_t n, const double* x, const double* y, const double* z, double Lx,
                    double Ly, double Lz, const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
                    const uint8_t* __restrict__ REV, const fm::Tab& tb, Rec* __restrict__ Q,
                    unsigned long long* __restrict__ MASK, double* __restrict__ pe, double* __restrict__ f,
                    double* __restrict__ virial, int* __restrict__ status) {
    __syncthreads();
    const int ns = sq.count, w = threadIdx.x >> 5;
    for (int k = w; k < ns; k += BT / 32)
        tersoff_warp_atom<T, Rec>(sq.atom[k], n, x, y, z, Lx, Ly, Lz, NN, NL, REV, sq.p, tb.e, Q, MASK, pe, f, virial,
                                  status, sq.ws[w]);
}

// Register body: up to MR neighbour slots, every per-neighbour quantity in registers (all array indices are
// compile-time constants after unrolling).  The arithmetic is one straight basic block over all MR slots, so
// ptxas interleaves the slots' independent FP64 chains; a slot that is empty or outside the force range
// (bit clear in `mask`) carries f_C = f_C' = f_R = f_A = 0 and drops out of every sum.  The only branch is
// the (rare) cut-off window R < r < S.  Inputs: raw r_ij of the slots (minimum image applied), the partner
// index jd and the reverse slot rv of each.  Every phase advances all MR slots (or all MR(MR-1)/2 unordered
// slot pairs) together, one arithmetic step at a time (fastmath.cuh, *_v): consecutive instructions are
// independent.
template <class T, class Rec, int MR>
__device__ __forceinline__ void
tersoff_reg_body(int64_t i, int64_t n, T (&ex)[MR], T (&ey)[MR], T (&ez)[MR], unsigned mask,
                 const int (&jd)[MR], const int (&rv)[MR], const TersoffDev<T>& p, const fm::Tab& tb,
                 Rec* __restrict__ Q, double* __restrict__ pe, double* __restrict__ f,
                 double* __restrict__ virial) {
    constexpr int NP = MR * (MR - 1) / 2;
    T rinv[MR], rr[MR], fc[MR], fcp[MR], fR[MR], fA[MR], zeta[MR];
    unsigned window = 0u;
    {
        T d2s[MR], aR[MR], aA[MR];
#pragma unroll
        for (int m = 0; m < MR; ++m) {
            const T d2 = ps::in_range_d2(ex[m], ey[m], ez[m]);
            d2s[m] = (mask >> m & 1u) ? d2 : T(1);           // keeps the empty slot's arithmetic finite
        }
        fm::rsqrt_v<MR>(d2s, rinv);
#pragma unroll
        for (int m = 0; m < MR; ++m) {
            rr[m] = d2s[m] * rinv[m];
            ex[m] *= rinv[m]; ey[m] *= rinv[m]; ez[m] *= rinv[m];
            aR[m] = -p.lambda * rr[m]; aA[m] = -p.mu * rr[m];
        }
        fm::exp_v<MR>(aR, fR, tb);
        fm::exp_v<MR>(aA, fA, tb);
#pragma unroll
        for (int m = 0; m < MR; ++m) {
            const bool in = mask >> m & 1u;
            window |= (in && rr[m] > p.R) ? 1u << m : 0u;
            fc[m] = in ? T(1) : T(0);
            fcp[m] = T(0);
            fR[m] = in ? p.A * fR[m] : T(0);
            fA[m] = in ? p.B * fA[m] : T(0);
            zeta[m] = T(0);
        }
    }
    if (window) {                                            // f_C window R < r < S (reading A1)
#pragma unroll
        for (int m = 0; m < MR; ++m)
            if (window >> m & 1u) {
                T sn, cs;
                fm::sincos_0_pi((rr[m] - p.R) * p.w, &sn, &cs);
                fc[m] = T(0.5) + T(0.5) * cs;
                fcp[m] = T(-0.5) * p.w * sn;
            }
    }

    // zeta (Eq. 4), unordered neighbour pairs visited once (g_ijk = g_ikj for one element);
    // g = 1 + (c/d)^2 x^2/(d^2 + x^2), x = h - cos (Eq. 5 without its cancellation)
    {
        T x2[NP], den[NP], q[NP];
        int c = 0;
#pragma unroll
        for (int a = 0; a < MR; ++a)
#pragma unroll
            for (int b = a + 1; b < MR; ++b, ++c) {
                const T xx = p.h - (ex[a] * ex[b] + ey[a] * ey[b] + ez[a] * ez[b]);
                x2[c] = xx * xx;
                den[c] = p.d2 + x2[c];
            }
        fm::rcp_v<NP>(den, q);
        c = 0;
#pragma unroll
        for (int a = 0; a < MR; ++a)
#pragma unroll
            for (int b = a + 1; b < MR; ++b, ++c) {
                const T g = T(1) + p.c2_over_d2 * x2[c] * q[c];
                zeta[a] += fc[b] * g;
                zeta[b] += fc[a] * g;
            }
    }

    // b_ij, b'_ij (Eq. 3); zeta = 0: b = 1, b' = 0 (reading A8)
    T U = T(0);
    T Px[MR], Py[MR], Pz[MR], hh[MR];
    {
        T zt[MR], w1[MR], w2[MR], t[MR], u[MR], bb[MR], rc[MR];
#pragma unroll
        for (int a = 0; a < MR; ++a) { zt[a] = zeta[a] > T(0) ? zeta[a] : T(1); w1[a] = p.beta * zt[a]; }
        fm::log_v<MR>(w1, w2, tb);
#pragma unroll
        for (int a = 0; a < MR; ++a) w2[a] *= p.n;
        fm::exp_v<MR>(w2, t, tb);                                        // (beta zeta)^n
#pragma unroll
        for (int a = 0; a < MR; ++a) { u[a] = T(1) + t[a]; w1[a] = zt[a] * u[a]; }
        fm::log_v<MR>(u, w2, tb);
#pragma unroll
        for (int a = 0; a < MR; ++a) w2[a] *= p.minus_half_over_n;
        fm::exp_v<MR>(w2, bb, tb);                                       // (1 + t)^(-1/2n)
        fm::rcp_v<MR>(w1, rc);
#pragma unroll
        for (int a = 0; a < MR; ++a) {
            const T posf = zeta[a] > T(0) ? T(1) : T(0);                 // a factor, not a branch
            const T b = zeta[a] > T(0) ? bb[a] : T(1);
            const T bp = T(-0.5) * bb[a] * t[a] * rc[a] * posf;
            const T bfA = b * fA[a];
            U += T(0.5) * fc[a] * (fR[a] - bfA);
            const T D = T(0.5) * (fcp[a] * (fR[a] - bfA) + fc[a] * (p.mu * bfA - p.lambda * fR[a]));
            hh[a] = T(-0.5) * fc[a] * fA[a] * bp;
            Px[a] = D * ex[a]; Py[a] = D * ey[a]; Pz[a] = D * ez[a];
        }
    }

    // P_a = D_a e_a + sum_{b != a} [ (h_a fc_b + h_b fc_a) g'_ab (e_b - cos e_a)/r_a + h_b fc'_a g_ab e_a ]
    {
        T cs[NP], xx[NP], den[NP], q[NP];
        int c = 0;
#pragma unroll
        for (int a = 0; a < MR; ++a)
#pragma unroll
            for (int b = a + 1; b < MR; ++b, ++c) {
                cs[c] = ex[a] * ex[b] + ey[a] * ey[b] + ez[a] * ez[b];
                xx[c] = p.h - cs[c];
                den[c] = p.d2 + xx[c] * xx[c];
            }
        fm::rcp_v<NP>(den, q);
        c = 0;
#pragma unroll
        for (int a = 0; a < MR; ++a)
#pragma unroll
            for (int b = a + 1; b < MR; ++b, ++c) {
                const T g = T(1) + p.c2_over_d2 * xx[c] * xx[c] * q[c];
                const T gp = T(-2) * p.c2 * xx[c] * q[c] * q[c];         // dg/dcos
                const T tab = (hh[a] * fc[b] + hh[b] * fc[a]) * gp;
                const T ta = tab * rinv[a], tb2 = tab * rinv[b];
                const T ua = hh[b] * fcp[a] * g - ta * cs[c];
                const T ub = hh[a] * fcp[b] * g - tb2 * cs[c];
                Px[a] += ta * ex[b] + ua * ex[a]; Py[a] += ta * ey[b] + ua * ey[a]; Pz[a] += ta * ez[b] + ua * ez[a];
                Px[b] += tb2 * ex[a] + ub * ex[b]; Py[b] += tb2 * ey[a] + ub * ey[b]; Pz[b] += tb2 * ez[a] + ub * ez[b];
            }
    }

    T Fx = T(0), Fy = T(0), Fz = T(0);
    T W[9] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
#pragma unroll
    for (int a = 0; a < MR; ++a)
        if (mask >> a & 1u) {
            rm::store_rec(&Q[(int64_t)rv[a] * n + jd[a]], Px[a], Py[a], Pz[a]);
            Fx += Px[a]; Fy += Py[a]; Fz += Pz[a];
            if (virial) {
                const T rx = ex[a] * rr[a], ry = ey[a] * rr[a], rz = ez[a] * rr[a];
                W[0] += rx * Px[a]; W[1] += rx * Py[a]; W[2] += rx * Pz[a];
                W[3] += ry * Px[a]; W[4] += ry * Py[a]; W[5] += ry * Pz[a];
                W[6] += rz * Px[a]; W[7] += rz * Py[a]; W[8] += rz * Pz[a];
            }
        }
    if (pe) pe[i] = (double)U;
    if (f) { f[i] = (double)Fx; f[n + i] = (double)Fy; f[2 * n + i] = (double)Fz; }
    if (virial) {
#pragma unroll
        for (int q = 0; q < 9; ++q) virial[(int64_t)q * n + i] = (double)(T(-0.5) * W[q]);
    }
}


// ---------------------------------------------------------------------------------------------------
// Lean register body: the crystal case of the NVE loop and of force-only calls (no virial asked for, no pair
// inside the cut-off window R < r < S).  Then f_C is 1 or 0 and f_C' = 0 for every slot, so f_C, f_C', r and
// every term that carries f_C' drop out (in the force pass g itself is no longer needed, only g'), the partner
// index and reverse slot fold into ONE 32-bit record index per slot, and the body fits 128 registers: 4 CTAs
// of 128 threads per SM instead of 3 (the kernel is bound by latency, not by the FP64 pipe: ncu r02a).  An
// atom with a pair inside the window is handed to the general per-thread path before any arithmetic.
template <class T, class Rec, int MR, bool WITH_W>
__device__ __forceinline__ void
tersoff_lean_body(int64_t i, int64_t n, T (&ex)[MR], T (&ey)[MR], T (&ez)[MR], const T (&d2in)[MR], unsigned mask,
                  const unsigned (&qi)[MR], const TersoffDev<T>& p, const fm::Tab& tb,
                  Rec* __restrict__ Q, double* __restrict__ pe, double* __restrict__ f, double* __restrict__ virial) {
    constexpr int NP = MR * (MR - 1) / 2;
    T rinv[MR], fR[MR], fA[MR], zeta[MR];
    {
        T d2s[MR], rr[MR], aR[MR], aA[MR];
#pragma unroll
        for (int m = 0; m < MR; ++m) d2s[m] = (mask >> m & 1u) ? d2in[m] : T(1);   // keeps an empty slot finite
        fm::rsqrt_v<MR>(d2s, rinv);
#pragma unroll
        for (int m = 0; m < MR; ++m) {
            rr[m] = d2s[m] * rinv[m];
            ex[m] *= rinv[m]; ey[m] *= rinv[m]; ez[m] *= rinv[m];
            aR[m] = -p.lambda * rr[m]; aA[m] = -p.mu * rr[m];
        }
        fm::exp_v<MR>(aR, fR, tb);
        fm::exp_v<MR>(aA, fA, tb);
#pragma unroll
        for (int m = 0; m < MR; ++m) {
            const bool in = mask >> m & 1u;
            fR[m] = in ? p.A * fR[m] : T(0);
            fA[m] = in ? p.B * fA[m] : T(0);
            zeta[m] = T(0);
        }
    }
    // zeta (Eq. 4) with f_C = 1 inside the range: unordered slot pairs once (g_ijk = g_ikj for one element)
    {
        T x2[NP], den[NP], q[NP];
        int c = 0;
#pragma unroll
        for (int a = 0; a < MR; ++a)
#pragma unroll
            for (int b = a + 1; b < MR; ++b, ++c) {
                const T xx = p.h - (ex[a] * ex[b] + ey[a] * ey[b] + ez[a] * ez[b]);
                x2[c] = xx * xx;
                den[c] = p.d2 + x2[c];
            }
        fm::rcp_v<NP>(den, q);
        c = 0;
#pragma unroll
        for (int a = 0; a < MR; ++a)
#pragma unroll
            for (int b = a + 1; b < MR; ++b, ++c) {
                const T g = T(1) + p.c2_over_d2 * x2[c] * q[c];
                zeta[a] += (mask >> b & 1u) ? g : T(0);
                zeta[b] += (mask >> a & 1u) ? g : T(0);
            }
    }
    // b, b' (Eq. 3); U_i; D_a = (mu b f_A - lambda f_R)/2; h_a = -f_A b'/2  (all zero for a slot out of range)
    T U = T(0);
    T Px[MR], Py[MR], Pz[MR], hh[MR];
    {
        T zt[MR], w1[MR], w2[MR], t[MR], u[MR], bb[MR], rc[MR];
#pragma unroll
        for (int a = 0; a < MR; ++a) { zt[a] = zeta[a] > T(0) ? zeta[a] : T(1); w1[a] = p.beta * zt[a]; }
        fm::log_v<MR>(w1, w2, tb);
#pragma unroll
        for (int a = 0; a < MR; ++a) w2[a] *= p.n;
        fm::exp_v<MR>(w2, t, tb);                                        // (beta zeta)^n
#pragma unroll
        for (int a = 0; a < MR; ++a) { u[a] = T(1) + t[a]; w1[a] = zt[a] * u[a]; }
        fm::log_v<MR>(u, w2, tb);
#pragma unroll
        for (int a = 0; a < MR; ++a) w2[a] *= p.minus_half_over_n;
        fm::exp_v<MR>(w2, bb, tb);                                       // (1 + t)^(-1/2n)
        fm::rcp_v<MR>(w1, rc);
#pragma unroll
        for (int a = 0; a < MR; ++a) {
            const bool pos = zeta[a] > T(0);                             // zeta = 0: b = 1, b' = 0 (reading A8)
            const T b = pos ? bb[a] : T(1);
            const T bp = pos ? T(-0.5) * bb[a] * t[a] * rc[a] : T(0);
            const T bfA = b * fA[a];
            U += T(0.5) * (fR[a] - bfA);
            const T D = T(0.5) * (p.mu * bfA - p.lambda * fR[a]);
            hh[a] = T(-0.5) * fA[a] * bp;
            Px[a] = D * ex[a]; Py[a] = D * ey[a]; Pz[a] = D * ez[a];
        }
    }
    // P_a = D_a e_a + sum_{b != a} (h_a [b in range] + h_b [a in range]) g'_ab (e_b - cos e_a)/r_a
    {
        T cs[NP], xx[NP], den[NP], q[NP];
        int c = 0;
#pragma unroll
        for (int a = 0; a < MR; ++a)
#pragma unroll
            for (int b = a + 1; b < MR; ++b, ++c) {
                cs[c] = ex[a] * ex[b] + ey[a] * ey[b] + ez[a] * ez[b];
                xx[c] = p.h - cs[c];
                den[c] = p.d2 + xx[c] * xx[c];
            }
        fm::rcp_v<NP>(den, q);
        c = 0;
#pragma unroll
        for (int a = 0; a < MR; ++a)
#pragma unroll
            for (int b = a + 1; b < MR; ++b, ++c) {
                const T gp = T(-2) * p.c2 * xx[c] * q[c] * q[c];         // dg/dcos
                const T tab = (((mask >> b & 1u) ? hh[a] : T(0)) + ((mask >> a & 1u) ? hh[b] : T(0))) * gp;
                const T ta = tab * rinv[a], tb2 = tab * rinv[b];
                const T ua = -ta * cs[c], ub = -tb2 * cs[c];
                Px[a] += ta * ex[b] + ua * ex[a]; Py[a] += ta * ey[b] + ua * ey[a]; Pz[a] += ta * ez[b] + ua * ez[a];
                Px[b] += tb2 * ex[a] + ub * ex[b]; Py[b] += tb2 * ey[a] + ub * ey[b]; Pz[b] += tb2 * ez[a] + ub * ez[b];
            }
    }
    T Fx = T(0), Fy = T(0), Fz = T(0);
#pragma unroll
    for (int a = 0; a < MR; ++a)
        if (mask >> a & 1u) {
            rm::store_rec(&Q[qi[a]], Px[a], Py[a], Pz[a]);
            Fx += Px[a]; Fy += Py[a]; Fz += Pz[a];
        }
    if (pe) pe[i] = (double)U;
    if (f) { f[i] = (double)Fx; f[n + i] = (double)Fy; f[2 * n + i] = (double)Fz; }
    if (WITH_W) {                                            // own half -1/2 sum_a r_a (x) P_a; r_a = e_a d2_a / r_a
        T W[9] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
#pragma unroll
        for (int a = 0; a < MR; ++a)
            if (mask >> a & 1u) {
                const T rr = d2in[a] * rinv[a];
                const T rx = ex[a] * rr, ry = ey[a] * rr, rz = ez[a] * rr;
                W[0] += rx * Px[a]; W[1] += rx * Py[a]; W[2] += rx * Pz[a];
                W[3] += ry * Px[a]; W[4] += ry * Py[a]; W[5] += ry * Pz[a];
                W[6] += rz * Px[a]; W[7] += rz * Py[a]; W[8] += rz * Pz[a];
            }
#pragma unroll
        for (int q = 0; q < 9; ++q) virial[(int64_t)q * n + i] = (double)(T(-0.5) * W[q]);
    }
}

template <class T, class Rec, int MR, int BT, int MAXREG, bool WITH_W>
__global__ void __launch_bounds__(BT) __maxnreg__(MAXREG)
k_tersoff_lean(int64_t n, int K, const double* x, const double* y, const double* z,   // no __restrict__ (see the wait below)
               double Lx, double Ly, double Lz,
               const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
               const uint8_t* __restrict__ REV, const MdRowHead* __restrict__ HEAD, TersoffDev<T> p,
               const double* __restrict__ gtab, Rec* __restrict__ Q, unsigned long long* __restrict__ MASK,
               double* __restrict__ pe, double* __restrict__ f, double* __restrict__ virial, int* __restrict__ status) {
    static_assert(MR == 4, "the row head record holds four entries");
    __shared__ __align__(16) double s_tab[fm::TAB_DOUBLES];
    __shared__ SlowQueue<T, BT> s_slow;
    if (threadIdx.x == 0) { s_slow.count = 0; s_slow.p = p; }
    const int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t i = i0 < n ? i0 : n - 1;
    // the row's first four entries, their reverse slots and its length: one 32-byte record (k_reverse wrote it)
    int4 h0; unsigned hrev; int nn;
    asm volatile("ld.global.nc.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(h0.x), "=r"(h0.y), "=r"(h0.z), "=r"(h0.w) : "l"(HEAD + i));
    asm volatile("ld.global.nc.v2.b32 {%0,%1}, [%2];" : "=r"(hrev), "=r"(nn) : "l"(reinterpret_cast<const int*>(HEAD + i) + 4));
    const int hj[4] = {h0.x, h0.y, h0.z, h0.w};
    int jd[MR];
    unsigned qi[MR];
#pragma unroll
    for (int m = 0; m < MR; ++m) {
        const int jr = hj[m];
        jd[m] = (unsigned)jr < (unsigned long long)n ? jr : (int)i;
        qi[m] = (hrev >> (8 * m) & 255u) * (unsigned)n + (unsigned)jd[m];   // n * K <= 2e9 (md_neighbors_create)
    }
    const fm::Tab tb = fm::stage_tables(s_tab, gtab);
    // Inside md_nve_run this kernel is launched as a programmatic dependent of the fused gather kernel that
    // wrote x, y, z (common.cuh, md_launch_pdl): the list loads above overlap with that kernel's tail; the
    // coordinates are read only from here on, through plain (coherent, non-.nc) loads.
    md_grid_wait();
    md_grid_release();
    const double xi = x[i], yi = y[i], zi = z[i];
    double dx[MR], dy[MR], dz[MR];
#pragma unroll
    for (int m = 0; m < MR; ++m) { dx[m] = x[jd[m]]; dy[m] = y[jd[m]]; dz[m] = z[jd[m]]; }
    __syncthreads();
    if (i0 < n) {
    const ps::MinImage mi = ps::make_min_image(Lx, Ly, Lz);
    T ex[MR], ey[MR], ez[MR], d2[MR];
    unsigned mask = 0u;
    bool slow = nn > MR || MD_TERSOFF_ALL_GENERAL;
    {
        bool far = false;
#pragma unroll
        for (int m = 0; m < MR; ++m) {
            dx[m] -= xi; dy[m] -= yi; dz[m] -= zi;
            d2[m] = ps::in_range_d2((T)dx[m], (T)dy[m], (T)dz[m]);       // the one in-range decision (pair_sort.cuh)
            far = far || mi.far(d2[m]);
        }
        if (__any_sync(__activemask(), far)) {               // warp-uniform: interior warps never shift
#pragma unroll
            for (int m = 0; m < MR; ++m) {
                mi.wrap(dx[m], dy[m], dz[m]);
                d2[m] = ps::in_range_d2((T)dx[m], (T)dy[m], (T)dz[m]);
            }
        }
        const T R2 = p.R * p.R;
#pragma unroll
        for (int m = 0; m < MR; ++m) {
            ex[m] = (T)dx[m]; ey[m] = (T)dy[m]; ez[m] = (T)dz[m];
            const bool in = m < nn && d2[m] < p.S2;
            mask |= in ? 1u << m : 0u;
            slow = slow || (in && d2[m] > R2);               // a pair inside the cut-off window
        }
    }
    if (slow) {                                              // rows longer than MR, or f_C not 0/1: the general path
        s_slow.atom[atomicAdd(&s_slow.count, 1)] = (int)i;
    } else {
        MASK[i] = (unsigned long long)mask;
        tersoff_lean_body<T, Rec, MR, WITH_W>(i, n, ex, ey, ez, d2, mask, qi, p, tb, Q, pe, f, virial);
    }
    }
    tersoff_drain_queue<T, Rec, BT>(s_slow, n, x, y, z, Lx, Ly, Lz, NN, NL, REV, tb, Q, MASK, pe, f, WITH_W ? virial : nullptr,
                                    status);
}

// Register path for a bin of atoms with at most MR in-range neighbours (pair_sort.cuh, Bins): thread t of CTA
// `cta` takes atom list[cta * BT + t], compacts its in-range list entries (bits of MASK) into MR register slots
// and runs the straight-line body.  Records go to the dense slots (every MASK is known: k_screen ran before).
// The math tables are staged by the calling kernel.
template <class T, class Rec, int MR, int BT>
__device__ __forceinline__ void
tersoff_binned_cta(int64_t cta, int64_t n, const double* __restrict__ x, const double* __restrict__ y,
                   const double* __restrict__ z, double Lx, double Ly, double Lz,
                   const int32_t* __restrict__ NL, const uint8_t* __restrict__ REV,
                   const int32_t* list, const int32_t* count, const TersoffDev<T>& p,
                   const fm::Tab& tb, Rec* __restrict__ Q, const unsigned long long* MASK,
                   double* __restrict__ pe, double* __restrict__ f, double* __restrict__ virial) {
    const int64_t cnt = *count;
    const int64_t t0 = cta * BT + threadIdx.x;
    if (t0 >= cnt) return;                                   // no barrier follows (the caller may still wait on the grid)
    const int64_t i = list[t0];
    unsigned long long run = MASK[i];
    const int M = min(__popcll(run), MR);
    int jd[MR], rv[MR];
#pragma unroll
    for (int k = 0; k < MR; ++k) {
        const int m = run ? __ffsll((long long)run) - 1 : 0;
        const unsigned q = (unsigned)m * (unsigned)n + (unsigned)i;
        jd[k] = run ? NL[q] : (int)i;                        // an empty slot points at the atom itself
        rv[k] = (int)REV[q];
        run &= run - 1;
    }
    const double xi = x[i], yi = y[i], zi = z[i];
    double qx[MR], qy[MR], qz[MR];
    unsigned long long mj[MR];
#pragma unroll
    for (int k = 0; k < MR; ++k) { qx[k] = x[jd[k]]; qy[k] = y[jd[k]]; qz[k] = z[jd[k]]; mj[k] = MASK[jd[k]]; }
    const ps::MinImage mi = ps::make_min_image(Lx, Ly, Lz);
    bool far = false;
#pragma unroll
    for (int k = 0; k < MR; ++k) {
        qx[k] -= xi; qy[k] -= yi; qz[k] -= zi;
        far = far || mi.far(ps::in_range_d2((T)qx[k], (T)qy[k], (T)qz[k]));
        rv[k] = (int)ps::dense_slot(mj[k], rv[k]);           // dense record layout
    }
    if (__any_sync(__activemask(), far)) {
#pragma unroll
        for (int k = 0; k < MR; ++k) mi.wrap(qx[k], qy[k], qz[k]);
    }
    T ex[MR], ey[MR], ez[MR];
#pragma unroll
    for (int k = 0; k < MR; ++k) { ex[k] = (T)qx[k]; ey[k] = (T)qy[k]; ez[k] = (T)qz[k]; }
    tersoff_reg_body<T, Rec, MR>(i, n, ex, ey, ez, (1u << M) - 1u, jd, rv, p, tb, Q, pe, f, virial);
}

// ---------------------------------------------------------------------------------------------------
// Loop kernel for list rows of any length (config 5: 4-9 listed, 3-6 in range; rows longer than 4 are what
// the register kernel cannot hold).  One thread per atom; the CTA first screens its atoms and reassigns them
// to threads in order of their in-range count M (pair_sort.cuh), so the loops below have warp-uniform trip
// counts.  Per-slot data live in the thread's shared-memory columns.
//   pass 1  per slot: e_ij, 1/r, f_C, f_C', f_R, f_A
//   pass 2  per slot a: zeta_ia over the other slots, b, b', U_ia/2; D_a and h_a replace f_R, f_A
//   pass 3  per slot a: P_ia (T5), pushed to Q[rev(i,a)*n + j_a]; own halves in registers
// Ordered pairs (a,b) and (b,a) are both visited: nothing here relies on g_ijk = g_ikj.
// With one element it only sees the atoms of the long-row bin (k_tersoff_binned takes the others).
template <class T, int BT, int PCA>
struct TersoffSortSmem {
    ps::SortScratch<2 * BT> ss;                              // two rounds per tile with several elements
    T ex[PCA * BT], ey[PCA * BT], ez[PCA * BT], rinv[PCA * BT];
    T fc[PCA * BT], fcp[PCA * BT], fRD[PCA * BT], fAh[PCA * BT];   // fRD: f_R then D; fAh: f_A then h
    int jj[PCA * BT];
    __align__(16) double tab[fm::TAB_DOUBLES];
};

// CTA `cta` of `nctas` CTAs that share the tiles; tables staged (and the block synchronised) by the caller.
template <class T, class Rec, int BT, int PCA, int NT>
__device__ __forceinline__ void
tersoff_sorted_ctas(int64_t cta, int64_t nctas, TersoffSortSmem<T, BT, PCA>& s, const fm::Tab& tb, int64_t n,
                    const double* __restrict__ x, const double* __restrict__ y,
                    const double* __restrict__ z, double Lx, double Ly, double Lz,
                    const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
                    const uint8_t* __restrict__ REV, const TersoffDev<T>& p, const TersoffTab<T, NT>& tab,
                    const int32_t* __restrict__ types, const int32_t* list,
                    const int32_t* count,
                    Rec* __restrict__ Q, const unsigned long long* MASK,
                    double* __restrict__ pe, double* __restrict__ f, double* __restrict__ virial,
                    int* __restrict__ status) {
    const int tid = threadIdx.x, lane = tid & 31;
    const ps::MinImage mi = ps::make_min_image(Lx, Ly, Lz);

    // a tile: BT consecutive atoms, or BT consecutive entries of a bin's index list (pair_sort.cuh, Bins); the
    // grid strides over the tiles (a bin may hold few atoms: a grid sized for "all atoms" would mostly launch
    // CTAs that exit at once, 25 us of nothing at 512 000 atoms)
    const int64_t cnt = list ? (int64_t)*count : n;
    // Several elements: tiles of 2 BT atoms in two rounds per thread (ps::sort_by_count_x2: every warp takes a block
    // of small and a block of large in-range counts); one element (the tail bin of config 5): BT atoms, one round.
    constexpr int RT = NT > 1 ? 2 : 1;
    for (int64_t A0 = cta * (RT * BT); A0 < cnt; A0 += nctas * (RT * BT)) {
    __syncthreads();                                         // the previous tile is done with the scratch
    unsigned long long mask0[RT];
#pragma unroll
    for (int r = 0; r < RT; ++r) {
        const int64_t e = A0 + r * BT + tid;
        const int64_t a0 = e < cnt ? (list ? (int64_t)list[e] : e) : -1;
        s.ss.atom[r * BT + tid] = (int)a0;
        mask0[r] = a0 >= 0 ? MASK[a0] : 0ull;                // in-range mask (k_screen wrote it)
    }
    int tv[2], basev[2], Mwv[2];
    unsigned long long mkv[2];
    bool sync_between = false;
    if constexpr (RT == 1) {
        ps::sort_by_count<BT>(s.ss, mask0[0], PCA * BT, status, &tv[0], &mkv[0], &basev[0], &Mwv[0]);
    } else {
        ps::sort_by_count_x2<BT>(s.ss, mask0, PCA * BT, status, tv, mkv, basev, Mwv, &sync_between);
    }
#pragma unroll 1
    for (int rd = 0; rd < RT; ++rd) {
    if (rd > 0 && sync_between) __syncthreads();             // the pool is divided anew for this round (CTA-uniform)
    // (selects, not tv[rd]: a dynamic index would put the four small arrays into local memory)
    const int col = (rd == 0 ? basev[0] : basev[1]) + lane;  // slot k of this thread: col + 32 k
    const unsigned long long mk = rd == 0 ? mkv[0] : mkv[1];
    const int M = min(__popcll(mk), rd == 0 ? Mwv[0] : Mwv[1]);
    const int64_t i = s.ss.atom[rd == 0 ? tv[0] : tv[1]];
    if (i < 0) continue;                                     // tile tail (M = 0); the barriers are reached by all

    const int ti = NT > 1 ? types[i] : 0;
    const TsCenter<T> pc = tab.c[ti];
    // pass 1
    {
        const double xi = x[i], yi = y[i], zi = z[i];
        unsigned long long run = mk;
        for (int k0 = 0; k0 < M; k0 += 2) {
            int j[2];
            double dx[2], dy[2], dz[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int m = __ffsll((long long)run) - 1;
                if (k0 + u < M) run &= run - 1;
                j[u] = NL[(unsigned)(m < 0 ? 0 : m) * (unsigned)n + (unsigned)i];
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) { dx[u] = x[j[u]] - xi; dy[u] = y[j[u]] - yi; dz[u] = z[j[u]] - zi; }
            T d2s[2];
            bool far = false;
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                d2s[u] = ps::in_range_d2((T)dx[u], (T)dy[u], (T)dz[u]);
                far = far || mi.far(d2s[u]);
            }
            if (__any_sync(__activemask(), far)) {           // warp-uniform: interior warps never shift
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    mi.wrap(dx[u], dy[u], dz[u]);
                    d2s[u] = ps::in_range_d2((T)dx[u], (T)dy[u], (T)dz[u]);
                }
            }
            // both slots step by step, branch-free (a slot past the last one computes on d2 = 1 and is not stored)
            bool val[2], win[2];
            int tj[2];
            T ri[2], r[2], ea[2], eb[2], fr[2], fa[2], c[2], cp[2];
            TsPair<T> pp[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) { val[u] = k0 + u < M; d2s[u] = val[u] ? d2s[u] : T(1); }
            fm::rsqrt_v<2>(d2s, ri);
            bool anywin = false;
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                r[u] = d2s[u] * ri[u];
                tj[u] = NT > 1 ? types[j[u]] : 0;
                pp[u] = tab.p[ti * NT + tj[u]];              // mixed parameters of the pair (reading A17)
                ea[u] = -pp[u].lambda * r[u]; eb[u] = -pp[u].mu * r[u];
                win[u] = val[u] && r[u] > pp[u].R;           // f_C window R < r < S (reading A1)
                anywin = anywin || win[u];
                c[u] = T(1); cp[u] = T(0);
            }
            fm::exp_v<2>(ea, fr, tb);
            fm::exp_v<2>(eb, fa, tb);
            if (anywin) {
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    if (!win[u]) continue;
                    T sn, cs;
                    fm::sincos_0_pi((r[u] - pp[u].R) * pp[u].w, &sn, &cs);
                    c[u] = T(0.5) + T(0.5) * cs;
                    cp[u] = T(-0.5) * pp[u].w * sn;
                }
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                if (!val[u]) continue;
                const int q = col + 32 * (k0 + u);
                s.ex[q] = (T)dx[u] * ri[u]; s.ey[q] = (T)dy[u] * ri[u]; s.ez[q] = (T)dz[u] * ri[u]; s.rinv[q] = ri[u];
                s.fc[q] = c[u]; s.fcp[q] = cp[u];
                s.fRD[q] = pp[u].A * fr[u];
                s.fAh[q] = pp[u].chi * pp[u].B * fa[u];      // chi_ij f_A: b_ij only ever multiplies it
                s.jj[q] = j[u] | (tj[u] << 28);              // element of the neighbour in the top bits (n < 2^28)
            }
        }
    }

    // pass 2: zeta_a = sum_{b != a} f_C(r_b) g_ab (Eq. 4), g in the cancellation-free form; b, b' (Eq. 3)
    // Two slots a per iteration, every arithmetic step written for both (independent chains for the FP64 pipe;
    // one slot at a time the kernel ran its dependent chains at ~17 cycles per instruction).  The loop over b
    // covers all M slots and masks b == a, so both chains walk the same b; the sums keep the order b = 0..M-1.
    T U = T(0);
    // (this pass reads only e and f_C of the other slots, so D and h can replace f_R and f_A of slot a at once)
    for (int a0 = 0; a0 < M; a0 += 2) {
        int av[2], ca[2];
        bool val[2];
        T ax[2], ay[2], az[2], zt[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            val[u] = a0 + u < M;
            av[u] = val[u] ? a0 + u : a0;
            ca[u] = col + 32 * av[u];
            ax[u] = s.ex[ca[u]]; ay[u] = s.ey[ca[u]]; az[u] = s.ez[ca[u]];
            zt[u] = T(0);
        }
#pragma unroll 2
        for (int b = 0; b < M; ++b) {
            const int cb = col + 32 * b;
            const T bx = s.ex[cb], by = s.ey[cb], bz = s.ez[cb], fcb = s.fc[cb];
            T x2[2], den[2], q[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const T cs = ax[u] * bx + ay[u] * by + az[u] * bz;
                const T xx = pc.h - cs;
                x2[u] = xx * xx;
                den[u] = pc.d2 + x2[u];
            }
            fm::rcp_v<2>(den, q);
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const T term = fcb * (T(1) + pc.c2_over_d2 * x2[u] * q[u]);
                zt[u] += b != av[u] ? term : T(0);
            }
        }
        // zeta = 0: b = 1, b' = 0 (reading A8); the chain runs on a harmless argument and is dropped
        bool pos[2];
        T arg[2], lg[2], tt[2], l1[2], bo[2], den2[2], rq[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) { pos[u] = zt[u] > T(0); arg[u] = pos[u] ? pc.beta * zt[u] : T(1); }
        fm::log_v<2>(arg, lg, tb);
#pragma unroll
        for (int u = 0; u < 2; ++u) arg[u] = pc.n * lg[u];
        fm::exp_v<2>(arg, tt, tb);                                                   // (beta zeta)^n
#pragma unroll
        for (int u = 0; u < 2; ++u) arg[u] = T(1) + tt[u];
        fm::log_v<2>(arg, l1, tb);
#pragma unroll
        for (int u = 0; u < 2; ++u) { den2[u] = (pos[u] ? zt[u] : T(1)) * arg[u]; arg[u] = pc.minus_half_over_n * l1[u]; }
        fm::exp_v<2>(arg, bo, tb);                                                   // Eq. (3)
        fm::rcp_v<2>(den2, rq);
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (!val[u]) continue;
            const T bov = pos[u] ? bo[u] : T(1);
            const T bp = pos[u] ? T(-0.5) * bo[u] * tt[u] * rq[u] : T(0);
            const T c = s.fc[ca[u]], cp = s.fcp[ca[u]], fR = s.fRD[ca[u]], fA = s.fAh[ca[u]];
            const TsPair<T> pp = tab.p[ti * NT + (NT > 1 ? (int)((unsigned)s.jj[ca[u]] >> 28) : 0)];
            const T bfA = bov * fA;
            U += T(0.5) * c * (fR - bfA);                                                  // U_ia / 2
            s.fRD[ca[u]] = T(0.5) * (cp * (fR - bfA) + c * (pp.mu * bfA - pp.lambda * fR));   // D
            s.fAh[ca[u]] = T(-0.5) * c * fA * bp;                                          // h
        }
    }

    // pass 3: P_a = D_a e_a + sum_{b != a} [ (h_a fc_b + h_b fc_a) g' (e_b - cos e_a)/r_a + h_b fc'_a g e_a ]
    // (two slots a per iteration as in pass 2; b == a is masked)
    T Fx = T(0), Fy = T(0), Fz = T(0);
    T W[9] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
    unsigned long long run = mk;
    for (int a0 = 0; a0 < M; a0 += 2) {
        int av[2], ca[2], ja[2], rv[2];
        bool val[2];
        T ax[2], ay[2], az[2], ha[2], fca[2], cpa[2], ria[2], ce[2], sx[2], sy[2], sz[2];
        unsigned long long mj[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            val[u] = a0 + u < M;
            av[u] = val[u] ? a0 + u : a0;
            ca[u] = col + 32 * av[u];
            const int m = run ? __ffsll((long long)run) - 1 : 0;
            if (val[u]) run &= run - 1;
            ja[u] = s.jj[ca[u]] & 0x0fffffff;
            rv[u] = (int)REV[(int64_t)m * n + i];
            mj[u] = MASK[ja[u]];
            ax[u] = s.ex[ca[u]]; ay[u] = s.ey[ca[u]]; az[u] = s.ez[ca[u]];
            ha[u] = s.fAh[ca[u]]; fca[u] = s.fc[ca[u]]; cpa[u] = s.fcp[ca[u]]; ria[u] = s.rinv[ca[u]];
            ce[u] = s.fRD[ca[u]];                            // coefficient of e_a
            sx[u] = T(0); sy[u] = T(0); sz[u] = T(0);        // sum of ta * e_b
        }
#pragma unroll 2
        for (int b = 0; b < M; ++b) {
            const int cb = col + 32 * b;
            const T bx = s.ex[cb], by = s.ey[cb], bz = s.ez[cb], hb = s.fAh[cb], fcb = s.fc[cb];
            T cs[2], xx[2], x2[2], den[2], q[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                cs[u] = ax[u] * bx + ay[u] * by + az[u] * bz;
                xx[u] = pc.h - cs[u];
                x2[u] = xx[u] * xx[u];
                den[u] = pc.d2 + x2[u];
            }
            fm::rcp_v<2>(den, q);
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const bool on = b != av[u];
                const T gp = T(-2) * pc.c2 * xx[u] * q[u] * q[u];                    // dg/dcos
                const T ta = on ? (ha[u] * fcb + hb * fca[u]) * gp * ria[u] : T(0);
                const T cterm = hb * cpa[u] * (T(1) + pc.c2_over_d2 * x2[u] * q[u]) - ta * cs[u];
                ce[u] += on ? cterm : T(0);
                sx[u] += ta * bx; sy[u] += ta * by; sz[u] += ta * bz;
            }
        }
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (!val[u]) continue;
            const unsigned slot = ps::dense_slot(mj[u], rv[u]);                      // dense record layout
            const T px = sx[u] + ce[u] * ax[u], py = sy[u] + ce[u] * ay[u], pz = sz[u] + ce[u] * az[u];
            rm::store_rec(&Q[slot * (unsigned)n + (unsigned)ja[u]], px, py, pz);
            Fx += px; Fy += py; Fz += pz;
            if (virial) {
                const T r = fm::rcp(ria[u]);
                const T rx = ax[u] * r, ry = ay[u] * r, rz = az[u] * r;
                W[0] += rx * px; W[1] += rx * py; W[2] += rx * pz;
                W[3] += ry * px; W[4] += ry * py; W[5] += ry * pz;
                W[6] += rz * px; W[7] += rz * py; W[8] += rz * pz;
            }
        }
    }
    if (pe) pe[i] = (double)U;
    if (f) { f[i] = (double)Fx; f[n + i] = (double)Fy; f[2 * n + i] = (double)Fz; }
    if (virial) {
#pragma unroll
        for (int q = 0; q < 9; ++q) virial[(int64_t)q * n + i] = (double)(T(-0.5) * W[q]);
    }
    }   // rounds
    }   // tiles
}

// The loop code on all atoms (several elements) or on one bin's list.
template <class T, class Rec, int BT, int PCA, int NT>
__global__ void __launch_bounds__(BT)
k_tersoff_sorted(int64_t n, const double* __restrict__ x, const double* __restrict__ y,
                 const double* __restrict__ z, double Lx, double Ly, double Lz,
                 const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
                 const uint8_t* __restrict__ REV, TersoffDev<T> p, TersoffTab<T, NT> tab,
                 const int32_t* __restrict__ types, const int32_t* list,
                 const int32_t* count, const double* __restrict__ gtab,
                 Rec* __restrict__ Q, const unsigned long long* MASK,
                 double* __restrict__ pe, double* __restrict__ f, double* __restrict__ virial,
                 int* __restrict__ status) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TersoffSortSmem<T, BT, PCA>& s = *reinterpret_cast<TersoffSortSmem<T, BT, PCA>*>(smem_raw);
    const fm::Tab tb = fm::stage_tables(s.tab, gtab);
    md_grid_wait();                                          // programmatic dependent of k_screen, which wrote MASK and
    md_grid_release();                                       // the bin lists (read below through plain loads)
    __syncthreads();
    tersoff_sorted_ctas<T, Rec, BT, PCA, NT>(blockIdx.x, gridDim.x, s, tb, n, x, y, z, Lx, Ly, Lz, NN, NL, REV, p, tab,
                                             types, list, count, Q, MASK, pe, f, virial, status);
}

// One element, rows of any length (config 5), ONE launch: the first `tail_ctas` CTAs run the loop code on the
// bin of atoms with more than MR in-range neighbours (few atoms, but a tile of them is ~20 us of dependent
// latency: they start first and overlap with everything else), the other CTAs run the register body on the
// bin with at most MR, BT atoms each.  (Measured alternatives: the tail as a kernel of its own after the
// register kernel costs its full latency, 25 us per step; on a second stream, the fork/join events cost more.)
template <class T, class Rec, int MR, int BT, int PCA, int MAXREG>
__global__ void __launch_bounds__(BT) __maxnreg__(MAXREG)
k_tersoff_hot(int64_t n, int tail_ctas, const double* __restrict__ x, const double* __restrict__ y,
              const double* __restrict__ z, double Lx, double Ly, double Lz,
              const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
              const uint8_t* __restrict__ REV, TersoffDev<T> p, TersoffTab<T, 1> tab,
              const int32_t* lists, const int32_t* counts,
              const double* __restrict__ gtab, Rec* __restrict__ Q, const unsigned long long* MASK,
              double* __restrict__ pe, double* __restrict__ f, double* __restrict__ virial,
              int* __restrict__ status) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    TersoffSortSmem<T, BT, PCA>& s = *reinterpret_cast<TersoffSortSmem<T, BT, PCA>*>(smem_raw);
    const fm::Tab tb = fm::stage_tables(s.tab, gtab);
    md_grid_wait();                                          // as k_tersoff_sorted
    md_grid_release();
    __syncthreads();
    if ((int)blockIdx.x < tail_ctas)
        tersoff_sorted_ctas<T, Rec, BT, PCA, 1>(blockIdx.x, tail_ctas, s, tb, n, x, y, z, Lx, Ly, Lz, NN, NL, REV, p, tab,
                                                nullptr, lists + 2 * n, counts + 2, Q, MASK, pe, f, virial, status);
    else
        tersoff_binned_cta<T, Rec, MR, BT>((int64_t)blockIdx.x - tail_ctas, n, x, y, z, Lx, Ly, Lz, NL, REV, lists,
                                           counts, p, tb, Q, MASK, pe, f, virial);
}

// The bin with at most MR in-range neighbours as a kernel of its own (k_tersoff_hot_tail, the loop code on the small
// tail bin, is launched just before it).  It needs nothing from that kernel, so it is launched as its programmatic
// dependent and does NOT wait at its start: both run side by side from the first cycle, the tail's few long-latency
// CTAs with their 52-68 KB of shared memory on some SMs, this kernel -- a few KB of shared memory, the whole L1 for
// its gathers -- everywhere else.  Its last `wait_ctas` CTAs call griddepcontrol.wait when their work is done, so
// that "this grid has completed" implies "the tail kernel has completed" for whatever follows on the stream; they
// are dispatched last, long after the tail kernel has finished, and never actually wait.
template <class T, class Rec, int MR, int BT, int MAXREG>
__global__ void __launch_bounds__(BT) __maxnreg__(MAXREG)
k_tersoff_binned(int64_t n, int wait_ctas, const double* __restrict__ x, const double* __restrict__ y,
                 const double* __restrict__ z, double Lx, double Ly, double Lz,
                 const int32_t* __restrict__ NL, const uint8_t* __restrict__ REV, TersoffDev<T> p,
                 const int32_t* list, const int32_t* count, const double* __restrict__ gtab, Rec* __restrict__ Q,
                 const unsigned long long* MASK, double* __restrict__ pe, double* __restrict__ f,
                 double* __restrict__ virial) {
    __shared__ __align__(16) double s_tab[fm::TAB_DOUBLES];
    const fm::Tab tb = fm::stage_tables(s_tab, gtab);
    md_grid_release();
    __syncthreads();
    tersoff_binned_cta<T, Rec, MR, BT>(blockIdx.x, n, x, y, z, Lx, Ly, Lz, NL, REV, list, count, p, tb, Q, MASK, pe, f, virial);
    if ((int)blockIdx.x >= (int)gridDim.x - wait_ctas) md_grid_wait();
}

template <class T>
TersoffDev<T> make_dev(const md_tersoff_params* hp) {
    TersoffDev<T> p;
    p.A = (T)hp->A; p.B = (T)hp->B; p.lambda = (T)hp->lambda; p.mu = (T)hp->mu; p.beta = (T)hp->beta;
    p.n = (T)hp->n; p.h = (T)hp->h; p.R = (T)hp->R; p.S2 = (T)(hp->S * hp->S);
    p.c2 = (T)(hp->c * hp->c); p.d2 = (T)(hp->d * hp->d); p.c2_over_d2 = (T)((hp->c * hp->c) / (hp->d * hp->d));
    p.w = (T)(3.14159265358979323846 / (hp->S - hp->R));
    p.minus_half_over_n = (T)(-0.5 / hp->n);
    return p;
}

// Mixing rules of reading A17 (lambda, mu: arithmetic means; A, B, R, S: geometric means), computed in double.
template <class T, int NT>
void make_tab(const md_tersoff_multi_params* hp, TersoffTab<T, NT>* tab, ps::RangeTab<T>* rt) {
    rt->nt = NT;
    for (int a = 0; a < NT; ++a) {
        const md_tersoff_params& e = hp->elem[a];
        TsCenter<T>& c = tab->c[a];
        c.beta = (T)e.beta; c.n = (T)e.n; c.h = (T)e.h; c.c2 = (T)(e.c * e.c); c.d2 = (T)(e.d * e.d);
        c.c2_over_d2 = (T)((e.c * e.c) / (e.d * e.d)); c.minus_half_over_n = (T)(-0.5 / e.n);
        for (int b = 0; b < NT; ++b) {
            const md_tersoff_params& g = hp->elem[b];
            const double R = sqrt(e.R * g.R), S = sqrt(e.S * g.S);
            TsPair<T>& q = tab->p[a * NT + b];
            q.A = (T)sqrt(e.A * g.A); q.B = (T)sqrt(e.B * g.B);
            q.lambda = (T)(0.5 * (e.lambda + g.lambda)); q.mu = (T)(0.5 * (e.mu + g.mu));
            q.R = (T)R; q.w = (T)(3.14159265358979323846 / (S - R)); q.chi = (T)hp->chi[a][b];
            rt->r2[a * NT + b] = (T)(S * S);
        }
    }
}

template <class T, class Rec, int NT>
int launch_sorted(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                  const double box[3], const TersoffDev<T>& p, const md_tersoff_multi_params* mp,
                  const int32_t* types, const double* gtab, double* pe, double* f, double* virial, bool pdl,
                  cudaStream_t s) {
    TersoffTab<T, NT> tab;
    ps::RangeTab<T> rt;
    make_tab<T, NT>(mp, &tab, &rt);
    // One element: atoms with at most 4 in-range neighbours (bin 0: four in five of a hot crystal) go to the
    // register kernel, the others (bin 2) to the loop kernel.  Several elements: the loop kernel takes all.
    ps::Bins bins;
    bins.b0 = 4; bins.b1 = 4;
    bins.list = NT == 1 ? nl->bin_list : nullptr;
    nl->bin_phase ^= 1;                                       // two sets of counters: this launch's, and the next one's
    int32_t* const counts = nl->bin_count + 4 * nl->bin_phase;   // (zeroed by this k_screen, see pair_sort.cuh)
    bins.count = counts;
    bins.count_next = NT == 1 ? nl->bin_count + 4 * (nl->bin_phase ^ 1) : nullptr;
    nl->launches[MD_KIND_PAIR] += NT == 1 ? (sizeof(T) == 8 ? 3 : 2) : 1;
    MD_CUDA_TRY(md_launch_pdl(ps::k_screen<T>, dim3((unsigned)((n + 255) / 256)), dim3(256), 0, s, pdl, (unsigned)n, x, y, z,
                              box[0], box[1], box[2], nl->NN, nl->NL, rt, NT > 1 ? types : (const int32_t*)nullptr, nl->MASK, bins));
    nl->q_dense = 1;
    constexpr int BT = 128, PCA = MD_TERSOFF_POOL_PER_ATOM;
    const unsigned grid = (unsigned)((n + BT - 1) / BT);      // sized for "every atom in this bin"; surplus CTAs exit at once
    using Sm = TersoffSortSmem<T, BT, PCA>;
    auto kern = k_tersoff_sorted<T, Rec, BT, PCA, NT>;
    const int rca = md_allow_dynamic_smem((const void*)kern, (int)sizeof(Sm));
    if (rca != MD_OK) return rca;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if constexpr (NT == 1) {
        const int tail = sms;                                // loop-code CTAs for the tail bin, striding over its tiles
        if constexpr (sizeof(T) == 8) {
            // FP64: tail bin first, then the register kernel beside it as a dependent that does not wait
            // (k_tersoff_binned): without the tail's 68 KB shared-memory pool in every CTA the register body has the
            // whole L1 for its gathers and fits 4 CTAs per SM at 128 registers (0.1244 -> 0.1140 ms per step on config 5)
            MD_CUDA_TRY(md_launch_pdl(kern, dim3((unsigned)tail), dim3(BT), sizeof(Sm), s, true, n, x, y, z, box[0], box[1],
                                      box[2], nl->NN, nl->NL, nl->REV, p, tab, (const int32_t*)nullptr,
                                      (const int32_t*)(nl->bin_list + 2 * n), (const int32_t*)(counts + 2), gtab, (Rec*)nl->Q,
                                      (const unsigned long long*)nl->MASK, pe, f, virial, nl->d_status));
            MD_CUDA_TRY(md_launch_pdl(k_tersoff_binned<T, Rec, 4, BT, 128>, dim3(grid), dim3(BT), 0, s, true, n, sms, x, y, z,
                                      box[0], box[1], box[2], nl->NL, nl->REV, p, (const int32_t*)nl->bin_list,
                                      (const int32_t*)counts, gtab, (Rec*)nl->Q, (const unsigned long long*)nl->MASK, pe, f,
                                      virial));
        } else {
            // FP32 mode: one launch, the first CTAs on the tail bin (measured: split 0.1033 / 0.0999 vs 0.0946 ms per
            // step -- the cheap float register body leaves the tail's tiles as the critical path, and they run
            // faster beside 2 than beside 4 register-body CTAs per SM)
            auto hot = k_tersoff_hot<T, Rec, 4, BT, PCA, 168>;
            const int rch = md_allow_dynamic_smem((const void*)hot, (int)sizeof(Sm));
            if (rch != MD_OK) return rch;
            MD_CUDA_TRY(md_launch_pdl(hot, dim3(grid + (unsigned)tail), dim3(BT), sizeof(Sm), s, true, n, tail, x, y, z, box[0],
                                      box[1], box[2], nl->NN, nl->NL, nl->REV, p, tab, (const int32_t*)nl->bin_list,
                                      (const int32_t*)counts, gtab, (Rec*)nl->Q, (const unsigned long long*)nl->MASK, pe, f,
                                      virial, nl->d_status));
        }
    } else {
        MD_CUDA_TRY(md_launch_pdl(kern, dim3(std::min<unsigned>(grid, 3u * (unsigned)sms)), dim3(BT), sizeof(Sm), s, true, n,
                                  x, y, z, box[0], box[1], box[2], nl->NN, nl->NL, nl->REV, p, tab, types,
                                  (const int32_t*)nullptr, (const int32_t*)nullptr, gtab, (Rec*)nl->Q,
                                  (const unsigned long long*)nl->MASK, pe, f, virial, nl->d_status));
    }
    MD_CUDA_TRY(cudaGetLastError());
    return MD_OK;
}

template <class T, class Rec>
int launch(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
           const double box[3], const md_tersoff_params* hp, double* pe, double* f, double* virial,
           bool pdl, cudaStream_t s) {
    const TersoffDev<T> p = make_dev<T>(hp);
    nl->gather_pdl = 0;
    ProfScope prof(nl, MD_KIND_PAIR, 1, s);
    const double* gtab = md_math_tables();
    if (!gtab) return MD_ERR_ALLOC;
    // Kernel selection by the row lengths of the list (known on the host once per build): the register
    // kernel handles rows of up to 4 entries (the crystal) in its fast path and longer ones through a slow
    // per-thread fallback, so it is used while fewer than 1 row in 256 is longer; otherwise the
    // sorted loop kernel (k_tersoff_sorted), which handles rows of any length.
    int max_row = 0, long_rows = 0;
    const int rcs = md_list_row_stats(nl, &max_row, &long_rows, 0);
    if (rcs != MD_OK) return rcs;
    if ((int64_t)long_rows * 256 > n) {
        md_tersoff_multi_params one;
        one.ntypes = 1; one.elem[0] = *hp; one.chi[0][0] = 1.0;
        return launch_sorted<T, Rec, 1>(nl, n, x, y, z, box, p, &one, nullptr, gtab, pe, f, virial, pdl, s);
    }
    nl->q_dense = 0;                                         // slot = reverse position (rows are at most 4 long)
    {   // the lean body; with the virial own half as a second instantiation (both fit 128 registers)
        constexpr int LBT = MD_TERSOFF_LEAN_BT;
        if (virial)
            MD_CUDA_TRY(md_launch_pdl(k_tersoff_lean<T, Rec, 4, LBT, MD_TERSOFF_LEAN_MAXREG, true>, dim3((unsigned)((n + LBT - 1) / LBT)),
                                      dim3(LBT), 0, s, pdl, n, nl->K, x, y, z, box[0], box[1], box[2], nl->NN, nl->NL,
                                      nl->REV, (const MdRowHead*)nl->HEAD, p, gtab, (Rec*)nl->Q, nl->MASK, pe, f, virial, nl->d_status));
        else
            MD_CUDA_TRY(md_launch_pdl(k_tersoff_lean<T, Rec, 4, LBT, MD_TERSOFF_LEAN_MAXREG, false>, dim3((unsigned)((n + LBT - 1) / LBT)),
                                      dim3(LBT), 0, s, pdl, n, nl->K, x, y, z, box[0], box[1], box[2], nl->NN, nl->NL,
                                      nl->REV, (const MdRowHead*)nl->HEAD, p, gtab, (Rec*)nl->Q, nl->MASK, pe, f, virial, nl->d_status));
        nl->gather_pdl = 1;
        return MD_OK;
    }
}

template <class T, class Rec>
int launch_multi(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                 const double box[3], const int32_t* types, const md_tersoff_multi_params* mp, double* pe,
                 double* f, double* virial, cudaStream_t s) {
    nl->gather_pdl = 0;
    const TersoffDev<T> p = make_dev<T>(&mp->elem[0]);       // used by the single-element register body only
    ProfScope prof(nl, MD_KIND_PAIR, 1, s);
    const double* gtab = md_math_tables();
    if (!gtab) return MD_ERR_ALLOC;
    switch (mp->ntypes) {
        case 1: return launch_sorted<T, Rec, 1>(nl, n, x, y, z, box, p, mp, nullptr, gtab, pe, f, virial, false, s);
        case 2: return launch_sorted<T, Rec, 2>(nl, n, x, y, z, box, p, mp, types, gtab, pe, f, virial, false, s);
        case 3: return launch_sorted<T, Rec, 3>(nl, n, x, y, z, box, p, mp, types, gtab, pe, f, virial, false, s);
        default: return launch_sorted<T, Rec, 4>(nl, n, x, y, z, box, p, mp, types, gtab, pe, f, virial, false, s);
    }
}

}  // namespace

int md_launch_tersoff_multi(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                            const double* vx, const double* vy, const double* vz, const double box[3],
                            const int32_t* types, const md_tersoff_multi_params* p, int precision, double* pe,
                            double* f, double* virial, double* heat, cudaStream_t s) {
    if (n == 0) return MD_OK;
    int rc = precision == MD_FP32 ? launch_multi<float, float4>(nl, n, x, y, z, box, types, p, pe, f, virial, s)
                                  : launch_multi<double, PairRec64>(nl, n, x, y, z, box, types, p, pe, f, virial, s);
    if (rc != MD_OK) return rc;
    return md_launch_gather(nl, n, x, y, z, vx, vy, vz, box, precision, f, virial, heat, nullptr, s);
}

int md_launch_tersoff(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                      const double* vx, const double* vy, const double* vz, const double box[3],
                      const md_tersoff_params* p, int precision, double* pe, double* f, double* virial,
                      double* heat, const VVFuse* vv, cudaStream_t s) {
    if (n == 0) return MD_OK;
    const bool pdl = vv && vv->pdl_pair;
    int rc = precision == MD_FP32 ? launch<float, float4>(nl, n, x, y, z, box, p, pe, f, virial, pdl, s)
                                  : launch<double, PairRec64>(nl, n, x, y, z, box, p, pe, f, virial, pdl, s);
    if (rc != MD_OK) return rc;
    return md_launch_gather(nl, n, x, y, z, vx, vy, vz, box, precision, f, virial, heat, vv, s);
}
