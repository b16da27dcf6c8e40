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

namespace {

template <class T>
struct SWDev {
    T Aeps, B, sigma, rc, rc2, gs, leps, cos0, p, q;
    int ip, iq;      // integer exponents if p, q are small non-negative integers, else -1
};

constexpr int SW_KC = 32;

template <class T> __device__ __forceinline__ T ipow(T a, int e) {
    T r = T(1);
    for (int k = 0; k < e; ++k) r *= a;
    return r;
}

template <class T, class Rec>
__global__ void __launch_bounds__(128)
k_sw_pair(int64_t n, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
          double Lx, double Ly, double Lz, const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
          const uint8_t* __restrict__ REV, SWDev<T> p, Rec* __restrict__ Q,
          unsigned long long* __restrict__ MASK, double* __restrict__ pe, double* __restrict__ f,
          double* __restrict__ virial, int* __restrict__ status) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double xi = x[i], yi = y[i], zi = z[i];
    const double hx = 0.5 * Lx, hy = 0.5 * Ly, hz = 0.5 * Lz;
    const int nn = NN[i];

    T ex[SW_KC], ey[SW_KC], ez[SW_KC], rinv[SW_KC], sj[SW_KC], ds[SW_KC];
    T Px[SW_KC], Py[SW_KC], Pz[SW_KC];
    int jdx[SW_KC];
    unsigned char slot[SW_KC];
    int M = 0;
    unsigned long long mask = 0ull;
    T U = T(0);

    for (int m = 0; m < nn; ++m) {
        const int j = NL[(int64_t)m * n + i];
        const double dx = md_min_image(x[j] - xi, Lx, hx);
        const double dy = md_min_image(y[j] - yi, Ly, hy);
        const double dz = md_min_image(z[j] - zi, Lz, hz);
        const T tx = (T)dx, ty = (T)dy, tz = (T)dz;
        const T d2 = tx * tx + ty * ty + tz * tz;
        if (d2 < p.rc2) {
            const T ri = rm::rsqrt(d2);
            const T rr = d2 * ri;
            if (!(rr < p.rc)) continue;                     // never divide by r - r_c = 0 (reading A8)
            if (M >= SW_KC) { atomicOr(&status[0], MD_DEV_INRANGE_OVERFLOW); continue; }
            const T e0 = tx * ri, e1 = ty * ri, e2 = tz * ri;
            const T u = T(1) / (rr - p.rc);                 // < 0
            // two-body: V2 = A eps [B (sigma/r)^p - (sigma/r)^q] exp(sigma/(r - rc))
            const T sr = p.sigma * ri;
            const T sp = p.ip >= 0 ? ipow(sr, p.ip) : rm::pow(sr, p.p);
            const T sq = p.iq >= 0 ? ipow(sr, p.iq) : rm::pow(sr, p.q);
            const T ev = p.Aeps * rm::exp(p.sigma * u);
            const T br = p.B * sp - sq;
            const T V2 = ev * br;
            const T V2p = ev * ((p.q * sq - p.p * p.B * sp) * ri - br * p.sigma * u * u);
            U += T(0.5) * V2;
            const T D = T(0.5) * V2p;
            ex[M] = e0; ey[M] = e1; ez[M] = e2; rinv[M] = ri;
            Px[M] = D * e0; Py[M] = D * e1; Pz[M] = D * e2;
            sj[M] = rm::exp(p.gs * u);
            ds[M] = -p.gs * u * u;
            jdx[M] = j; slot[M] = (unsigned char)m;
            mask |= 1ull << m;
            ++M;
        }
    }

    for (int a = 0; a < M; ++a)
        for (int b = a + 1; b < M; ++b) {
            const T cs = ex[a] * ex[b] + ey[a] * ey[b] + ez[a] * ez[b];
            const T dl = cs - p.cos0;
            const T E = p.leps * sj[a] * sj[b];
            const T Ed = E * dl;
            U += Ed * dl;                                   // V3 belongs to the central atom i
            const T ta = T(2) * Ed * rinv[a], tb = T(2) * Ed * rinv[b];
            const T ua = Ed * dl * ds[a] - ta * cs;
            const T ub = Ed * dl * ds[b] - tb * cs;
            Px[a] += ta * ex[b] + ua * ex[a]; Py[a] += ta * ey[b] + ua * ey[a]; Pz[a] += ta * ez[b] + ua * ez[a];
            Px[b] += tb * ex[a] + ub * ex[b]; Py[b] += tb * ey[a] + ub * ey[b]; Pz[b] += tb * ez[a] + ub * ez[b];
        }

    T Fx = T(0), Fy = T(0), Fz = T(0);
    T W[9] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
    for (int a = 0; a < M; ++a) {
        const int m = slot[a];
        const int mm = REV[(int64_t)m * n + i];
        rm::store_rec(&Q[(int64_t)mm * n + jdx[a]], Px[a], Py[a], Pz[a]);
        Fx += Px[a]; Fy += Py[a]; Fz += Pz[a];
        if (virial) {
            const T rr = T(1) / rinv[a];
            const T rx = ex[a] * rr, ry = ey[a] * rr, rz = ez[a] * rr;
            W[0] += rx * Px[a]; W[1] += rx * Py[a]; W[2] += rx * Pz[a];
            W[3] += ry * Px[a]; W[4] += ry * Py[a]; W[5] += ry * Pz[a];
            W[6] += rz * Px[a]; W[7] += rz * Py[a]; W[8] += rz * Pz[a];
        }
    }
    MASK[i] = mask;
    if (pe) pe[i] = (double)U;
    if (f) { f[i] = (double)Fx; f[n + i] = (double)Fy; f[2 * n + i] = (double)Fz; }
    if (virial) {
#pragma unroll
        for (int q = 0; q < 9; ++q) virial[(int64_t)q * n + i] = (double)(T(-0.5) * W[q]);
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
    ProfScope prof(nl, MD_KIND_PAIR, 1, s);
    k_sw_pair<T, Rec><<<(unsigned)((n + 127) / 128), 128, 0, s>>>(
        n, x, y, z, box[0], box[1], box[2], nl->NN, nl->NL, nl->REV, p, (Rec*)nl->Q, nl->MASK,
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
