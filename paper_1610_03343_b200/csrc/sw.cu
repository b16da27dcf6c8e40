// sw.cu -- per-pair kernel for the Stillinger-Weber potential (second instance of the general
// many-body form, Eqs. 28-30; "only a single kernel" is needed for the bond
// terms).  Formulas: DESIGN.md S1-S3 (the paper prints none; its Ref. [18]).
//
//   U_i  = 1/2 sum_j V2(r_ij) + sum_{j<k} V3(r_ij, r_ik, cos theta_jik)          (reading A6)
//   P_ij = 1/2 V2'(r_ij) e_ij
//        + sum_{k != j} lambda eps s_j s_k [ ds_j delta^2 e_ij + 2 delta (e_ik - cos e_ij)/r_ij ]
//   s_j = exp(gamma sigma/(r_ij - r_c)), ds_j = -gamma sigma/(r_ij - r_c)^2, delta = cos - cos0.
// Same push / own-half scheme as tersoff.cu.
//
// The three-body sum is separable.  With s_j = exp(gamma sigma/(r_ij - r_c)), c0 = cos0 and the moments
//   S = sum_j s_j,  S2 = sum_j s_j^2,  v = sum_j s_j e_j,  T = sum_j s_j e_j (x) e_j      (in-range j)
// one has  sum_{j<k} s_j s_k (e_j.e_k - c0)^2 = 1/2 [ T:T - 2 c0 |v|^2 + c0^2 S^2 - (1 - c0)^2 S2 ],  so
//   U3_i      = lambda eps / 2 [ T:T - 2 c0 |v|^2 + c0^2 S^2 - (1 - c0)^2 S2 ]
//   dU3/ds_j  = lambda eps [ e_j.T e_j - 2 c0 v.e_j + c0^2 S - (1 - c0)^2 s_j ]  =: A_j  (= sum_{k!=j} lambda eps s_k delta_jk^2)
//   dU3/de_j  = 2 lambda eps s_j (T e_j - c0 v) =: g_j   (up to a radial part that the projection removes)
//   P_ij      = [ V2'/2 + A_j s_j ds_j - (e_j.g_j)/r_ij ] e_j + g_j / r_ij
// which is term for term the double sum above, evaluated in O(M) per atom instead of O(M^2).  Every term
// keeps its factor s_j, so a neighbour at the edge of the range still gets full relative accuracy; the
// cancellation inside A_j and g_j (terms O(S), result O(S delta)) costs ~2 digits of 16.
//
// Kernel structure (k_sw_sorted): one thread per atom, loops over the atom's in-range neighbours.  The SW
// list holds the whole second shell (16-18 entries at the 0.5 A skin) but only 4-12 of them (mean 5.9) are
// inside r_c, so
//   screen  every thread tests the listed neighbours of one atom of the CTA's tile (coalesced row reads)
//           and keeps the in-range bits: that is MASK, stored at once;
//   sort    the CTA reassigns its atoms to threads in order of M (pair_sort.cuh): warps become M-uniform;
//   pass 1  per in-range slot: e_ij, r, s_j  -> the thread's shared-memory columns; moments in registers;
//   pass 2  per slot: two-body terms, A_j, g_j, P_ij pushed to Q[rev(i,j)*n + j]; U_i and the own halves
//           sum_j P_ij, -1/2 sum_j r_ij (x) P_ij accumulate in registers.
// Both passes take two slots per iteration (independent chains for the FP64 pipe).
#include "common.cuh"
#include "real_math.cuh"
#include "pair_sort.cuh"
#include "fastmath.cuh"

namespace {

template <class T>
struct SWDev {
    T Aeps, B, sigma, rc, rc2, gs, leps, cos0, p, q;
};

// (sigma/r)^e: E >= 0 is a compile-time integer exponent, E < 0 means "use pow with the real exponent"
template <int E, class T> __device__ __forceinline__ T spow(T a, T e) {
    if (E < 0) return rm::pow(a, e);
    T r = T(1);
#pragma unroll
    for (int k = 0; k < E; ++k) r *= a;
    return r;
}

template <class T, int BT, int PCA>
struct SWSmem {
    ps::SortScratch<BT> ss;
    T ex[PCA * BT], ey[PCA * BT], ez[PCA * BT];   // unit vectors e_ij of the thread's in-range slots
    T sj[PCA * BT], rr[PCA * BT];                 // s_j and r_ij
    __align__(16) double tab[fm::TAB_DOUBLES];
};

template <class T, class Rec, int BT, int PCA, int IP, int IQ>
__global__ void __launch_bounds__(BT)
k_sw_sorted(int64_t n, const double* __restrict__ x, const double* __restrict__ y,
            const double* __restrict__ z, double Lx, double Ly, double Lz,
            const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
            const uint8_t* __restrict__ REV, SWDev<T> p, const double* __restrict__ gtab,
            Rec* __restrict__ Q, unsigned long long* __restrict__ MASK,
            double* __restrict__ pe, double* __restrict__ f, double* __restrict__ virial,
            int* __restrict__ status) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SWSmem<T, BT, PCA>& s = *reinterpret_cast<SWSmem<T, BT, PCA>*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31;
    const int64_t A0 = (int64_t)blockIdx.x * BT;
    const fm::Tab tb = fm::stage_tables(s.tab, gtab);       // visible after the sort's barriers
    const ps::MinImage mi = ps::make_min_image(Lx, Ly, Lz);

    // screen, tile order
    unsigned long long mask0 = 0ull;
    if (A0 + tid < n) {
        const int64_t i0 = A0 + tid;
        int nn = NN[i0];
        if (nn > 64) nn = 64;
        mask0 = ps::screen_row<T>((unsigned)i0, (unsigned)n, nn, x, y, z, mi, NL, p.rc2);
        MASK[i0] = mask0;
    }
    int t, base, Mw;
    unsigned long long mk;
    ps::sort_by_count<BT>(s.ss, mask0, PCA * BT, status, &t, &mk, &base, &Mw);
    const int M = min(__popcll(mk), Mw);
    if (A0 + t >= n) return;                                 // tile tail (M = 0); no barrier follows
    const int64_t i = A0 + t;
    const int col = base + lane;                             // slot k of this thread: col + 32 k

    // pass 1: geometry and s_j of every in-range slot; moments S, S2, v, T
    T S = T(0), S2 = T(0), vx = T(0), vy = T(0), vz = T(0);
    T Txx = T(0), Txy = T(0), Txz = T(0), Tyy = T(0), Tyz = T(0), Tzz = T(0);
    {
        const double xi = x[i], yi = y[i], zi = z[i];
        unsigned long long run = mk;
        for (int k0 = 0; k0 < M; k0 += 2) {
            int j[2];
            double dx[2], dy[2], dz[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int m = __ffsll((long long)run) - 1;   // run != 0 while k0 + u < M; else m = -1 -> slot 0
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
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                if (k0 + u >= M) continue;
                const T tx = (T)dx[u], ty = (T)dy[u], tz = (T)dz[u];
                const T d2 = d2s[u];
                const T ri = fm::rsqrt(d2);
                const T r = d2 * ri;
                // u = 1/(r - r_c) < 0, clamped at -300: beyond that exp(sigma u) < 1e-270 is zero for every
                // purpose, and fm::exp wants |argument| < 2e7; never divide by r - r_c = 0 (reading A8)
                const bool ok = r < p.rc;
                const T uu = ok ? max(fm::rcp(r - p.rc), T(-300)) : T(-1);
                const int c = col + 32 * (k0 + u);
                const T ex = tx * ri, ey = ty * ri, ez = tz * ri;
                const T sj = ok ? fm::exp(p.gs * uu, tb) : T(0);
                s.ex[c] = ex; s.ey[c] = ey; s.ez[c] = ez;
                s.rr[c] = r;
                s.sj[c] = sj;
                const T wx = sj * ex, wy = sj * ey, wz = sj * ez;
                S += sj; S2 += sj * sj;
                vx += wx; vy += wy; vz += wz;
                Txx += wx * ex; Txy += wx * ey; Txz += wx * ez;
                Tyy += wy * ey; Tyz += wy * ez; Tzz += wz * ez;
            }
        }
    }

    // pass 2: P_j = [ V2'/2 + A_j s_j ds_j - (e_j.g_j)/r_j ] e_j + g_j/r_j  (header comment)
    const T c0 = p.cos0, om2 = (T(1) - c0) * (T(1) - c0);
    const T cvx = c0 * vx, cvy = c0 * vy, cvz = c0 * vz, kS = c0 * c0 * S;
    T U = T(0.5) * p.leps * (Txx * Txx + Tyy * Tyy + Tzz * Tzz + T(2) * (Txy * Txy + Txz * Txz + Tyz * Tyz)
                             - T(2) * (cvx * vx + cvy * vy + cvz * vz) + kS * S - om2 * S2);   // V3 of atom i (A6)
    T Fx = T(0), Fy = T(0), Fz = T(0);
    T W[9] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
    unsigned long long run = mk;
    for (int a0 = 0; a0 < M; a0 += 2) {
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            if (a0 + u >= M) continue;
            const int m = __ffsll((long long)run) - 1;
            run &= run - 1;
            const int ca = col + 32 * (a0 + u);
            const T ex = s.ex[ca], ey = s.ey[ca], ez = s.ez[ca], r = s.rr[ca], sj = s.sj[ca];
            const unsigned mi32 = (unsigned)m * (unsigned)n + (unsigned)i;
            const int ja = NL[mi32];                         // L1-hot: read by the screen and by pass 1
            const int mm = REV[mi32];
            // two-body: V2 = A eps [B (sigma/r)^p - (sigma/r)^q] exp(sigma/(r - rc))
            const bool ok = r < p.rc;
            const T ri = fm::rcp(r);
            const T uu = ok ? max(fm::rcp(r - p.rc), T(-300)) : T(-1);
            const T sr = p.sigma * ri;
            const T sp = spow<IP>(sr, p.p), sq = spow<IQ>(sr, p.q);
            const T ev = ok ? p.Aeps * fm::exp(p.sigma * uu, tb) : T(0);
            const T br = p.B * sp - sq;
            const T u2 = uu * uu;
            const T D = T(0.5) * ev * ((p.q * sq - p.p * p.B * sp) * ri - br * p.sigma * u2);   // V2'/2
            // three-body through the moments
            const T wx = Txx * ex + Txy * ey + Txz * ez, wy = Txy * ex + Tyy * ey + Tyz * ez,
                    wz = Txz * ex + Tyz * ey + Tzz * ez;                                          // T e_j
            const T q = ex * wx + ey * wy + ez * wz, ve = vx * ex + vy * ey + vz * ez;
            const T A = p.leps * (q - T(2) * c0 * ve + kS - om2 * sj);
            const T k2 = T(2) * p.leps * sj;
            const T gx = k2 * (wx - cvx), gy = k2 * (wy - cvy), gz = k2 * (wz - cvz);             // g_j
            const T eg = k2 * (q - c0 * ve);                                                      // e_j . g_j
            const T ce = D - A * sj * p.gs * u2 - eg * ri;                                        // ds_j = -gs u^2
            const T px = ce * ex + gx * ri, py = ce * ey + gy * ri, pz = ce * ez + gz * ri;
            rm::store_rec(&Q[(unsigned)mm * (unsigned)n + (unsigned)ja], px, py, pz);
            U += T(0.5) * ev * br;                           // V2/2
            Fx += px; Fy += py; Fz += pz;
            if (virial) {
                const T rx = ex * r, ry = ey * r, rz = ez * r;
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
}

template <class T, class Rec>
int launch(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
           const double box[3], const md_sw_params* hp, double* pe, double* f, double* virial, cudaStream_t s) {
    SWDev<T> p;
    const double rc = hp->a * hp->sigma;
    p.Aeps = (T)(hp->A * hp->epsilon); p.B = (T)hp->B; p.sigma = (T)hp->sigma;
    p.rc = (T)rc; p.rc2 = (T)(rc * rc); p.gs = (T)(hp->gamma * hp->sigma);
    p.leps = (T)(hp->lambda * hp->epsilon); p.cos0 = (T)hp->cos0; p.p = (T)hp->p; p.q = (T)hp->q;
    const double* gtab = md_math_tables();
    if (!gtab) return MD_ERR_ALLOC;
    ProfScope prof(nl, MD_KIND_PAIR, 1, s);
    constexpr int BT = 128, PCA = MD_SW_POOL_PER_ATOM;
    using Sm = SWSmem<T, BT, PCA>;
    // the published exponents (p = 4, q = 0) get compile-time integer powers; anything else goes through pow
    auto kern = (hp->p == 4.0 && hp->q == 0.0) ? k_sw_sorted<T, Rec, BT, PCA, 4, 0> : k_sw_sorted<T, Rec, BT, PCA, -1, -1>;
    const int rcs = md_allow_dynamic_smem((const void*)kern, (int)sizeof(Sm));
    if (rcs != MD_OK) return rcs;
    kern<<<(unsigned)((n + BT - 1) / BT), BT, sizeof(Sm), s>>>(
        n, x, y, z, box[0], box[1], box[2], nl->NN, nl->NL, nl->REV, p, gtab, (Rec*)nl->Q, nl->MASK,
        pe, f, virial, nl->d_status);
    MD_CUDA_TRY(cudaGetLastError());
    return MD_OK;
}

}  // namespace

int md_launch_sw(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                 const double* vx, const double* vy, const double* vz, const double box[3],
                 const md_sw_params* p, int precision, double* pe, double* f, double* virial,
                 double* heat, const VVFuse* vv, cudaStream_t s) {
    if (n == 0) return MD_OK;
    int rc = precision == MD_FP32 ? launch<float, float4>(nl, n, x, y, z, box, p, pe, f, virial, s)
                                  : launch<double, PairRec64>(nl, n, x, y, z, box, p, pe, f, virial, s);
    if (rc != MD_OK) return rc;
    return md_launch_gather(nl, n, x, y, z, vx, vy, vz, box, precision, f, virial, heat, vv, s);
}
