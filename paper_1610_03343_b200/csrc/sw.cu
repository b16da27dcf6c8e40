// sw.cu -- per-pair kernel for the Stillinger-Weber potential (second instance of the general
// many-body form, Eqs. 28-30; "only a single kernel" is needed for the bond
// terms).  Formulas: DESIGN.md S1-S3 (the paper prints none; its Ref. [18]).
//
//   U_i  = 1/2 sum_j V2(r_ij) + sum_{j<k} V3(r_ij, r_ik, cos theta_jik)          (reading A6)
//   P_ij = 1/2 V2'(r_ij) e_ij
//        + sum_{k != j} lambda eps s_j s_k [ ds_j delta^2 e_ij + 2 delta (e_ik - cos e_ij)/r_ij ]
//   s_j = exp(gamma sigma/(r_ij - r_c)), ds_j = -gamma sigma/(r_ij - r_c)^2, delta = cos - cos0.
// Same push / own-half scheme as tersoff.cu.
#include "common.cuh"
#include "real_math.cuh"
#include "pair_cta.cuh"
#include "fastmath.cuh"

namespace {

template <class T>
struct SWDev {
    T Aeps, B, sigma, rc, rc2, gs, leps, cos0, p, q;
    int ip, iq;      // integer exponents if p, q are small non-negative integers, else -1
};

template <class T> __device__ __forceinline__ T ipow(T a, int e) {
    T r = T(1);
    for (int k = 0; k < e; ++k) r *= a;
    return r;
}

// "lanes = pairs" kernel.  The SW list holds the whole second shell (16-18 entries at the 0.5 A skin) but
// only ~6 of them are inside r_c, so a thread-per-atom loop would idle most lanes and spill its per-
// neighbour arrays.  A CTA of 256 threads owns TA atoms:
//   stage A  compaction of the in-range pairs into shared memory              (pair_cta.cuh)
//   stage B  per pair: e_ij, 1/r, V2, V2', s_j = exp(gamma sigma/(r - r_c)), ds_j
//   stage C  per pair: three-body sums over the other in-range pairs of the same atom, P_ij pushed
//            to Q[rev(i,m)*n + j]
//   stage D  per atom: U_i, own halves sum_j P_ij and -1/2 sum_j r_ij (x) P_ij, MASK
template <class T, int TA, int PC>
struct SWSmem {
    pc::Dense<T, TA, PC> d;
    T rinv[PC], sj[PC], ds[PC], D[PC], Uh[PC];   // Uh: V2/2, then + the pair's share of the V3 terms
    T Px[PC], Py[PC], Pz[PC];
    __align__(16) double tab[fm::TAB_DOUBLES];
};

template <class T, class Rec, int TA, int PC>
__global__ void __launch_bounds__(pc::NT)
k_sw_pairs_cta(int64_t n, int K, const double* __restrict__ x, const double* __restrict__ y,
               const double* __restrict__ z, double Lx, double Ly, double Lz,
               const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
               const uint8_t* __restrict__ REV, SWDev<T> p, const double* __restrict__ gtab,
               Rec* __restrict__ Q, unsigned long long* __restrict__ MASK,
               double* __restrict__ pe, double* __restrict__ f, double* __restrict__ virial,
               int* __restrict__ status) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SWSmem<T, TA, PC>& s = *reinterpret_cast<SWSmem<T, TA, PC>*>(smem_raw);
    const int tid = threadIdx.x;
    const int64_t A0 = (int64_t)blockIdx.x * TA;
    const int na = (int)min((int64_t)TA, n - A0);
    const fm::Tab tb = fm::stage_tables(s.tab, gtab);       // visible after compact_in_range's barriers
    pc::compact_in_range<T, TA, PC, 32>(s.d, A0, na, n, K, x, y, z, Lx, Ly, Lz, NN, NL, p.rc2, status);
    const int np = s.d.np;

    // stage B
    for (int k = tid; k < np; k += pc::NT) {
        const T tx = s.d.ex[k], ty = s.d.ey[k], tz = s.d.ez[k];
        const T d2 = tx * tx + ty * ty + tz * tz;
        const T ri = fm::rsqrt(d2);
        const T rr = d2 * ri;
        s.d.ex[k] = tx * ri; s.d.ey[k] = ty * ri; s.d.ez[k] = tz * ri; s.rinv[k] = ri;
        const bool ok = rr < p.rc;                          // never divide by r - r_c = 0 (reading A8)
        // u = 1/(r - r_c) < 0, clamped at -300: beyond that exp(sigma u) < 1e-270 is zero for every purpose,
        // and fm::exp wants |argument| < 2e7
        const T u = ok ? max(fm::rcp(rr - p.rc), T(-300)) : T(-1);
        // two-body: V2 = A eps [B (sigma/r)^p - (sigma/r)^q] exp(sigma/(r - rc))
        const T sr = p.sigma * ri;
        const T sp = p.ip >= 0 ? ipow(sr, p.ip) : rm::pow(sr, p.p);
        const T sq = p.iq >= 0 ? ipow(sr, p.iq) : rm::pow(sr, p.q);
        const T ev = ok ? p.Aeps * fm::exp(p.sigma * u, tb) : T(0);
        const T br = p.B * sp - sq;
        s.Uh[k] = T(0.5) * ev * br;
        s.D[k] = T(0.5) * ev * ((p.q * sq - p.p * p.B * sp) * ri - br * p.sigma * u * u);
        s.sj[k] = ok ? fm::exp(p.gs * u, tb) : T(0);
        s.ds[k] = -p.gs * u * u;
    }
    __syncthreads();

    // stage C: P_a = D_a e_a + sum_{b != a} E [ ds_a delta^2 e_a + 2 delta (e_b - cos e_a)/r_a ],
    // E = lambda eps s_a s_b, delta = cos - cos0; V3 of a triplet belongs to the central atom (A6)
    for (int k = tid; k < np; k += pc::NT) {
        const int tmk = s.d.tm[k];
        const int t = tmk >> 6, m = tmk & 63;
        const int b0 = s.d.off[t], b1 = s.d.off[t + 1];
        const T ax = s.d.ex[k], ay = s.d.ey[k], az = s.d.ez[k];
        const T sa = p.leps * s.sj[k], dsa = s.ds[k], two_ria = T(2) * s.rinv[k];
        T ce = s.D[k];                                       // coefficient of e_a
        T sx = T(0), sy = T(0), sz = T(0), u3 = T(0);
        for (int b = b0; b < b1; ++b) {
            if (b == k) continue;
            const T bx = s.d.ex[b], by = s.d.ey[b], bz = s.d.ez[b];
            const T cs = ax * bx + ay * by + az * bz;
            const T dl = cs - p.cos0;
            const T Ed = sa * s.sj[b] * dl;
            const T Edd = Ed * dl;
            u3 += Edd;
            const T ta = Ed * two_ria;
            ce += Edd * dsa - ta * cs;
            sx += ta * bx; sy += ta * by; sz += ta * bz;
        }
        const T px = sx + ce * ax, py = sy + ce * ay, pz = sz + ce * az;
        s.Px[k] = px; s.Py[k] = py; s.Pz[k] = pz;
        s.Uh[k] += T(0.5) * u3;                              // each unordered pair (a,b) is met twice
        const int64_t i = A0 + t;
        const int mm = REV[(int64_t)m * n + i];
        rm::store_rec(&Q[(int64_t)mm * n + s.d.j[k]], px, py, pz);
    }
    __syncthreads();

    // stage D: per-atom sums
    for (int t = tid; t < na; t += pc::NT) {
        const int64_t i = A0 + t;
        T U = T(0), Fx = T(0), Fy = T(0), Fz = T(0);
        T W[9] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
        for (int b = s.d.off[t]; b < s.d.off[t + 1]; ++b) {
            const T px = s.Px[b], py = s.Py[b], pz = s.Pz[b];
            U += s.Uh[b]; Fx += px; Fy += py; Fz += pz;
            if (virial) {
                const T rr = T(1) / s.rinv[b];
                const T rx = s.d.ex[b] * rr, ry = s.d.ey[b] * rr, rz = s.d.ez[b] * rr;
                W[0] += rx * px; W[1] += rx * py; W[2] += rx * pz;
                W[3] += ry * px; W[4] += ry * py; W[5] += ry * pz;
                W[6] += rz * px; W[7] += rz * py; W[8] += rz * pz;
            }
        }
        MASK[i] = s.d.mask[t];
        if (pe) pe[i] = (double)U;
        if (f) { f[i] = (double)Fx; f[n + i] = (double)Fy; f[2 * n + i] = (double)Fz; }
        if (virial) {
#pragma unroll
            for (int q = 0; q < 9; ++q) virial[(int64_t)q * n + i] = (double)(T(-0.5) * W[q]);
        }
    }
}

inline int small_int(double v) {
    const int k = (int)v;
    return ((double)k == v && k >= 0 && k <= 16) ? k : -1;
}

template <class T, class Rec>
int launch(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
           const double box[3], const md_sw_params* hp, double* pe, double* f, double* virial, cudaStream_t s) {
    SWDev<T> p;
    const double rc = hp->a * hp->sigma;
    p.Aeps = (T)(hp->A * hp->epsilon); p.B = (T)hp->B; p.sigma = (T)hp->sigma;
    p.rc = (T)rc; p.rc2 = (T)(rc * rc); p.gs = (T)(hp->gamma * hp->sigma);
    p.leps = (T)(hp->lambda * hp->epsilon); p.cos0 = (T)hp->cos0; p.p = (T)hp->p; p.q = (T)hp->q;
    p.ip = small_int(hp->p); p.iq = small_int(hp->q);
    const double* gtab = md_math_tables();
    if (!gtab) return MD_ERR_ALLOC;
    ProfScope prof(nl, MD_KIND_PAIR, 1, s);
    constexpr int TA = 40, PC = 16 * TA;                     // ~6 in-range pairs per atom: ~240 per CTA
    using Sm = SWSmem<T, TA, PC>;
    auto kern = k_sw_pairs_cta<T, Rec, TA, PC>;
    static bool attr_set = false;
    if (!attr_set) {
        MD_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Sm)));
        attr_set = true;
    }
    kern<<<(unsigned)((n + TA - 1) / TA), pc::NT, sizeof(Sm), s>>>(
        n, nl->K, x, y, z, box[0], box[1], box[2], nl->NN, nl->NL, nl->REV, p, gtab, (Rec*)nl->Q, nl->MASK,
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
