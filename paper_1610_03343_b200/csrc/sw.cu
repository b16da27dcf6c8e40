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

#ifndef MD_SW_MAXREG
#define MD_SW_MAXREG 168     // 3 CTAs of 128 threads per SM; measured: 128 registers (4 CTAs) spills and is 30 % slower
#endif
template <class T, class Rec, int BT, int PCA, int IP, int IQ, int MAXREG>
__global__ void __launch_bounds__(BT) __maxnreg__(MAXREG)
k_sw_sorted(int64_t n, const double* __restrict__ x, const double* __restrict__ y,
            const double* __restrict__ z, double Lx, double Ly, double Lz,
            const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
            const uint8_t* __restrict__ REV, SWDev<T> p, const double* __restrict__ gtab,
            Rec* __restrict__ Q, const unsigned long long* MASK,    // MASK: k_screen, the kernel before, wrote it
            double* __restrict__ pe, double* __restrict__ f, double* __restrict__ virial,
            int* __restrict__ status) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SWSmem<T, BT, PCA>& s = *reinterpret_cast<SWSmem<T, BT, PCA>*>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31;
    const int64_t A0 = (int64_t)blockIdx.x * BT;
    const fm::Tab tb = fm::stage_tables(s.tab, gtab);       // visible after the sort's barriers
    md_grid_wait();                                          // programmatic dependent of k_screen (common.cuh)
    md_grid_release();
    const ps::MinImage mi = ps::make_min_image(Lx, Ly, Lz);

    // in-range masks of the tile (k_screen wrote them), tile order
    const unsigned long long mask0 = A0 + tid < n ? MASK[A0 + tid] : 0ull;
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
        const unsigned n32 = (unsigned)n, i32 = (unsigned)i;
        unsigned long long run = mk;
        // Two-deep software pipeline over chunks of two slots: while chunk c is worked on, the coordinates of
        // chunk c+1 and the list entries of chunk c+2 are in flight (the list entry -> coordinate chain is two
        // dependent loads; ld_early pins the requests where they are written).
        double cx[2], cy[2], cz[2], nx[2], ny[2], nz[2];
        int jq[2];
        auto req_idx = [&](int k0, int (&j)[2]) {
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int m = __ffsll((long long)run) - 1;   // run != 0 while k0 + u < M; else m = -1 -> slot 0
                if (k0 + u < M) run &= run - 1;
                j[u] = ps::ld_early(&NL[(unsigned)(m < 0 ? 0 : m) * n32 + i32]);
            }
        };
        auto req_xyz = [&](const int (&j)[2], double (&fx)[2], double (&fy)[2], double (&fz)[2]) {
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                fx[u] = ps::ld_early(&x[j[u]]); fy[u] = ps::ld_early(&y[j[u]]); fz[u] = ps::ld_early(&z[j[u]]);
            }
        };
        {
            int j0[2];
            req_idx(0, j0);
            req_idx(2, jq);
            req_xyz(j0, cx, cy, cz);
        }
        for (int k0 = 0; k0 < M; k0 += 2) {
            if (k0 + 2 < M) req_xyz(jq, nx, ny, nz);
            if (k0 + 4 < M) req_idx(k0 + 4, jq);
            double dx[2], dy[2], dz[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) { dx[u] = cx[u] - xi; dy[u] = cy[u] - yi; dz[u] = cz[u] - zi; }
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
            // Both slots advance together, one arithmetic step at a time, with no branch between them (a slot
            // past the atom's last one computes on d2 = 1 and contributes s_j = 0), so that consecutive FP64
            // instructions are independent.
            bool val[2], ok[2];
            T ri[2], r[2], um[2], uu[2], arg[2], sj[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) { val[u] = k0 + u < M; d2s[u] = val[u] ? d2s[u] : T(1); }
            fm::rsqrt_v<2>(d2s, ri);
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                r[u] = d2s[u] * ri[u];
                ok[u] = val[u] && r[u] < p.rc;               // never divide by r - r_c = 0 (reading A8)
                um[u] = ok[u] ? r[u] - p.rc : T(-1);
            }
            fm::rcp_v<2>(um, uu);
            // u = 1/(r - r_c) < 0, clamped at -300: beyond that exp(sigma u) < 1e-270 is zero for every purpose,
            // and fm::exp wants |argument| < 2e7
#pragma unroll
            for (int u = 0; u < 2; ++u) { uu[u] = max(uu[u], T(-300)); arg[u] = p.gs * uu[u]; }
            fm::exp_v<2>(arg, sj, tb);
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                sj[u] = ok[u] ? sj[u] : T(0);
                const T ex = (T)dx[u] * ri[u], ey = (T)dy[u] * ri[u], ez = (T)dz[u] * ri[u];
                const int c = col + 32 * (k0 + u);
                if (val[u]) { s.ex[c] = ex; s.ey[c] = ey; s.ez[c] = ez; s.rr[c] = r[u]; s.sj[c] = sj[u]; }
                const T wx = sj[u] * ex, wy = sj[u] * ey, wz = sj[u] * ez;
                S += sj[u]; S2 += sj[u] * sj[u];
                vx += wx; vy += wy; vz += wz;
                Txx += wx * ex; Txy += wx * ey; Txz += wx * ez;
                Tyy += wy * ey; Tyz += wy * ez; Tzz += wz * ez;
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) { cx[u] = nx[u]; cy[u] = ny[u]; cz[u] = nz[u]; }
        }
    }

    // pass 2: P_j = [ V2'/2 + A_j s_j ds_j - (e_j.g_j)/r_j ] e_j + g_j/r_j  (header comment)
    const T c0 = p.cos0, om2 = (T(1) - c0) * (T(1) - c0);
    const T cvx = c0 * vx, cvy = c0 * vy, cvz = c0 * vz, kS = c0 * c0 * S;
    T U = T(0.5) * p.leps * (Txx * Txx + Tyy * Tyy + Tzz * Tzz + T(2) * (Txy * Txy + Txz * Txz + Tyz * Tyz)
                             - T(2) * (cvx * vx + cvy * vy + cvz * vz) + kS * S - om2 * S2);   // V3 of atom i (A6)
    T Fx = T(0), Fy = T(0), Fz = T(0);
    T W[9] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
    // the record slot of pair (i -> j) needs NL -> MASK[j] (two dependent loads): same two-deep pipeline
    const unsigned n32 = (unsigned)n, i32 = (unsigned)i;
    unsigned long long run = mk;
    int qj[2], qr[2], cj[2], cr[2], nj[2], nr[2];            // requested / current / next: partner index, rev
    unsigned long long cm[2], nm[2];                         // MASK of the partner
    auto req_jr = [&](int k0, int (&j)[2], int (&r)[2]) {
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int m = __ffsll((long long)run) - 1;
            if (k0 + u < M) run &= run - 1;
            const unsigned q = (unsigned)(m < 0 ? 0 : m) * n32 + i32;
            j[u] = ps::ld_early(&NL[q]);
            r[u] = ps::ld_early(&REV[q]);
        }
    };
    auto req_mask = [&](const int (&j)[2], unsigned long long (&mj)[2]) {
#pragma unroll
        for (int u = 0; u < 2; ++u) mj[u] = ps::ld_early(&MASK[j[u]]);
    };
    req_jr(0, cj, cr);
    req_jr(2, qj, qr);
    req_mask(cj, cm);
    for (int a0 = 0; a0 < M; a0 += 2) {
        if (a0 + 2 < M) {
#pragma unroll
            for (int u = 0; u < 2; ++u) { nj[u] = qj[u]; nr[u] = qr[u]; }
            req_mask(nj, nm);
        }
        if (a0 + 4 < M) req_jr(a0 + 4, qj, qr);
        // both slots together, stage by stage, branch-free (a slot past the last one re-reads slot M-1 and is
        // masked out of the store and the sums)
        bool val[2], ok[2];
        T ex[2], ey[2], ez[2], r[2], sj[2], um[2], ri[2], uu[2], arg[2], ev[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            val[u] = a0 + u < M;
            const int ca = col + 32 * min(a0 + u, M - 1);
            ex[u] = s.ex[ca]; ey[u] = s.ey[ca]; ez[u] = s.ez[ca]; r[u] = s.rr[ca]; sj[u] = s.sj[ca];
            ok[u] = r[u] < p.rc;
            um[u] = ok[u] ? r[u] - p.rc : T(-1);
        }
        fm::rcp_v<2>(r, ri);
        fm::rcp_v<2>(um, uu);
#pragma unroll
        for (int u = 0; u < 2; ++u) { uu[u] = max(uu[u], T(-300)); arg[u] = p.sigma * uu[u]; }
        fm::exp_v<2>(arg, ev, tb);
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            // two-body: V2 = A eps [B (sigma/r)^p - (sigma/r)^q] exp(sigma/(r - rc))
            const T evu = ok[u] ? p.Aeps * ev[u] : T(0);
            const T sr = p.sigma * ri[u];
            const T sp = spow<IP>(sr, p.p), sq = spow<IQ>(sr, p.q);
            const T br = p.B * sp - sq;
            const T u2 = uu[u] * uu[u];
            const T D = T(0.5) * evu * ((p.q * sq - p.p * p.B * sp) * ri[u] - br * p.sigma * u2);   // V2'/2
            // three-body through the moments
            const T wx = Txx * ex[u] + Txy * ey[u] + Txz * ez[u], wy = Txy * ex[u] + Tyy * ey[u] + Tyz * ez[u],
                    wz = Txz * ex[u] + Tyz * ey[u] + Tzz * ez[u];                                   // T e_j
            const T q = ex[u] * wx + ey[u] * wy + ez[u] * wz, ve = vx * ex[u] + vy * ey[u] + vz * ez[u];
            const T A = p.leps * (q - T(2) * c0 * ve + kS - om2 * sj[u]);
            const T k2 = T(2) * p.leps * sj[u];
            const T gx = k2 * (wx - cvx), gy = k2 * (wy - cvy), gz = k2 * (wz - cvz);               // g_j
            const T eg = k2 * (q - c0 * ve);                                                        // e_j . g_j
            const T ce = D - A * sj[u] * p.gs * u2 - eg * ri[u];                                    // ds_j = -gs u^2
            const T keep = val[u] ? T(1) : T(0);
            const T px = keep * (ce * ex[u] + gx * ri[u]), py = keep * (ce * ey[u] + gy * ri[u]),
                    pz = keep * (ce * ez[u] + gz * ri[u]);
            if (val[u]) rm::store_rec(&Q[ps::dense_slot(cm[u], cr[u]) * n32 + (unsigned)cj[u]], px, py, pz);
            U += keep * T(0.5) * evu * br;                   // V2/2
            Fx += px; Fy += py; Fz += pz;
            if (virial) {
                const T rx = ex[u] * r[u], ry = ey[u] * r[u], rz = ez[u] * r[u];
                W[0] += rx * px; W[1] += rx * py; W[2] += rx * pz;
                W[3] += ry * px; W[4] += ry * py; W[5] += ry * pz;
                W[6] += rz * px; W[7] += rz * py; W[8] += rz * pz;
            }
        }
#pragma unroll
        for (int u = 0; u < 2; ++u) { cj[u] = nj[u]; cr[u] = nr[u]; cm[u] = nm[u]; }
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
           const double box[3], const md_sw_params* hp, double* pe, double* f, double* virial, bool pdl,
           cudaStream_t s) {
    SWDev<T> p;
    const double rc = hp->a * hp->sigma;
    p.Aeps = (T)(hp->A * hp->epsilon); p.B = (T)hp->B; p.sigma = (T)hp->sigma;
    p.rc = (T)rc; p.rc2 = (T)(rc * rc); p.gs = (T)(hp->gamma * hp->sigma);
    p.leps = (T)(hp->lambda * hp->epsilon); p.cos0 = (T)hp->cos0; p.p = (T)hp->p; p.q = (T)hp->q;
    const double* gtab = md_math_tables();
    if (!gtab) return MD_ERR_ALLOC;
    nl->gather_pdl = 0;
    ProfScope prof(nl, MD_KIND_PAIR, 2, s);
    ps::RangeTab<T> rt;
    rt.nt = 1; rt.r2[0] = p.rc2;
    MD_CUDA_TRY(md_launch_pdl(ps::k_screen<T>, dim3((unsigned)((n + 255) / 256)), dim3(256), 0, s, pdl, (unsigned)n, x, y, z,
                              box[0], box[1], box[2], nl->NN, nl->NL, rt, (const int32_t*)nullptr, nl->MASK,
                              ps::Bins{0, 0, nullptr, nullptr, nullptr}));
    nl->q_dense = 1;
    constexpr int BT = 128, PCA = MD_SW_POOL_PER_ATOM;
    using Sm = SWSmem<T, BT, PCA>;
    // the published exponents (p = 4, q = 0) get compile-time integer powers; anything else goes through pow
    auto kern = (hp->p == 4.0 && hp->q == 0.0) ? k_sw_sorted<T, Rec, BT, PCA, 4, 0, MD_SW_MAXREG>
                                                   : k_sw_sorted<T, Rec, BT, PCA, -1, -1, MD_SW_MAXREG>;
    const int rcs = md_allow_dynamic_smem((const void*)kern, (int)sizeof(Sm));
    if (rcs != MD_OK) return rcs;
    MD_CUDA_TRY(md_launch_pdl(kern, dim3((unsigned)((n + BT - 1) / BT)), dim3(BT), sizeof(Sm), s, true, n, x, y, z, box[0],
                              box[1], box[2], nl->NN, nl->NL, nl->REV, p, gtab, (Rec*)nl->Q,
                              (const unsigned long long*)nl->MASK, pe, f, virial, nl->d_status));
    return MD_OK;
}

}  // namespace

int md_launch_sw(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                 const double* vx, const double* vy, const double* vz, const double box[3],
                 const md_sw_params* p, int precision, double* pe, double* f, double* virial,
                 double* heat, const VVFuse* vv, cudaStream_t s) {
    if (n == 0) return MD_OK;
    const bool pdl = vv && vv->pdl_pair;                     // the list is unchanged and the kernel before is the loop's own
    int rc = precision == MD_FP32 ? launch<float, float4>(nl, n, x, y, z, box, p, pe, f, virial, pdl, s)
                                  : launch<double, PairRec64>(nl, n, x, y, z, box, p, pe, f, virial, pdl, s);
    if (rc != MD_OK) return rc;
    return md_launch_gather(nl, n, x, y, z, vx, vy, vz, box, precision, f, virial, heat, vv, s);
}
