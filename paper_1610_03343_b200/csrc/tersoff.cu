// tersoff.cu -- per-pair kernel for the Tersoff potential (steps B1 + B2 of DESIGN.md).
//
// One thread per atom i.  For every listed neighbour inside the force range S it computes the
// bond order zeta_ij, b_ij, b'_ij (Eqs. 3-6; Algorithm 3) and the
// partial derivative P_ij = dU_i/dr_ij (Eq. 14; explicit form: DESIGN.md T5), then
//   * pushes P_ij into the record slot of atom j that the gather kernel of j reads
//     (Q[rev(i,m)*n + j]; exactly one writer per slot, no atomics),
//   * accumulates the "own" halves  sum_j P_ij  and  -1/2 sum_j r_ij (x) P_ij  and U_i.
// T = double (MD_FP64) or float (MD_FP32: r_ij formed in double, then rounded; reading A10).
#include "common.cuh"
#include "real_math.cuh"

namespace {

template <class T>
struct TersoffDev {
    T A, B, lambda, mu, beta, n, h, R, S2;
    T c2, d2, c2_over_d2;     // c^2, d^2, c^2/d^2
    T w;                      // pi / (S - R)
    T minus_half_over_n;      // -1/(2n)
};

constexpr int TERSOFF_KC = 16;   // cap on in-range neighbours per atom

template <class T, class Rec>
__global__ void __launch_bounds__(128)
k_tersoff_pair(int64_t n, const double* __restrict__ x, const double* __restrict__ y,
               const double* __restrict__ z, double Lx, double Ly, double Lz,
               const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
               const uint8_t* __restrict__ REV, TersoffDev<T> p,
               Rec* __restrict__ Q, unsigned long long* __restrict__ MASK,
               double* __restrict__ pe, double* __restrict__ f, double* __restrict__ virial,
               int* __restrict__ status) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double xi = x[i], yi = y[i], zi = z[i];
    const double hx = 0.5 * Lx, hy = 0.5 * Ly, hz = 0.5 * Lz;
    const int nn = NN[i];

    T ex[TERSOFF_KC], ey[TERSOFF_KC], ez[TERSOFF_KC], r[TERSOFF_KC];
    T fc[TERSOFF_KC], fcp[TERSOFF_KC], fR[TERSOFF_KC], fA[TERSOFF_KC];
    T zeta[TERSOFF_KC];
    int jdx[TERSOFF_KC];
    unsigned char slot[TERSOFF_KC];
    int M = 0;
    unsigned long long mask = 0ull;

    for (int m = 0; m < nn; ++m) {
        const int j = NL[(int64_t)m * n + i];
        const double dx = md_min_image(x[j] - xi, Lx, hx);
        const double dy = md_min_image(y[j] - yi, Ly, hy);
        const double dz = md_min_image(z[j] - zi, Lz, hz);
        const T tx = (T)dx, ty = (T)dy, tz = (T)dz;
        const T d2 = tx * tx + ty * ty + tz * tz;
        if (d2 < p.S2) {
            if (M >= TERSOFF_KC) { atomicOr(&status[0], MD_DEV_INRANGE_OVERFLOW); continue; }
            const T rinv = rm::rsqrt(d2);
            const T rr = d2 * rinv;
            ex[M] = tx * rinv; ey[M] = ty * rinv; ez[M] = tz * rinv; r[M] = rr;
            T c = T(1), cp = T(0);
            if (rr > p.R) {                                  // f_C window R < r < S (reading A1)
                T sn, cs;
                rm::sincos((rr - p.R) * p.w, &sn, &cs);
                c = T(0.5) + T(0.5) * cs;
                cp = T(-0.5) * p.w * sn;
            }
            fc[M] = c; fcp[M] = cp;
            fR[M] = p.A * rm::exp(-p.lambda * rr);
            fA[M] = p.B * rm::exp(-p.mu * rr);
            zeta[M] = T(0);
            jdx[M] = j; slot[M] = (unsigned char)m;
            mask |= 1ull << m;
            ++M;
        }
    }

    // zeta_ij = sum_{k != j} f_C(r_ik) g_ijk (Eq. 4); single element: g_ijk = g_ikj, visit a < b once.
    // g = 1 + (c/d)^2 x^2/(d^2 + x^2), x = h - cos (algebraically Eq. 5, without its cancellation)
    for (int a = 0; a < M; ++a)
        for (int b = a + 1; b < M; ++b) {
            const T cs = ex[a] * ex[b] + ey[a] * ey[b] + ez[a] * ez[b];
            const T xx = p.h - cs;
            const T x2 = xx * xx;
            const T g = T(1) + p.c2_over_d2 * x2 / (p.d2 + x2);
            zeta[a] += fc[b] * g;
            zeta[b] += fc[a] * g;
        }

    // b_ij, b'_ij (Eq. 3) and the two-body coefficients
    T U = T(0);
    T D[TERSOFF_KC], hh[TERSOFF_KC];
    for (int a = 0; a < M; ++a) {
        T b = T(1), bp = T(0);
        const T zt = zeta[a];
        if (zt > T(0)) {                                     // zeta = 0: b = 1, b' = 0 (reading A8)
            const T t = rm::exp(p.n * rm::log(p.beta * zt)); // (beta zeta)^n
            b = rm::exp(p.minus_half_over_n * rm::log1p(t));
            bp = -b * t / (T(2) * zt * (T(1) + t));
        }
        const T bfA = b * fA[a];
        U += T(0.5) * fc[a] * (fR[a] - bfA);
        D[a] = T(0.5) * (fcp[a] * (fR[a] - bfA) + fc[a] * (p.mu * bfA - p.lambda * fR[a]));
        hh[a] = T(-0.5) * fc[a] * fA[a] * bp;
    }

    // P_a = D_a e_a + sum_{b != a} [ (h_a fc_b + h_b fc_a) g'_ab (e_b - cos e_a)/r_a + h_b fc'_a g_ab e_a ]
    T Px[TERSOFF_KC], Py[TERSOFF_KC], Pz[TERSOFF_KC];
    for (int a = 0; a < M; ++a) { Px[a] = D[a] * ex[a]; Py[a] = D[a] * ey[a]; Pz[a] = D[a] * ez[a]; }
    for (int a = 0; a < M; ++a)
        for (int b = a + 1; b < M; ++b) {
            const T cs = ex[a] * ex[b] + ey[a] * ey[b] + ez[a] * ez[b];
            const T xx = p.h - cs;
            const T x2 = xx * xx;
            const T q = T(1) / (p.d2 + x2);
            const T g = T(1) + p.c2_over_d2 * x2 * q;
            const T gp = T(-2) * p.c2 * xx * q * q;          // dg/dcos
            const T tab = (hh[a] * fc[b] + hh[b] * fc[a]) * gp;
            const T ta = tab / r[a], tb = tab / r[b];
            const T ua = hh[b] * fcp[a] * g - ta * cs;       // coefficient of e_a in P_a
            const T ub = hh[a] * fcp[b] * g - tb * cs;       // coefficient of e_b in P_b
            Px[a] += ta * ex[b] + ua * ex[a]; Py[a] += ta * ey[b] + ua * ey[a]; Pz[a] += ta * ez[b] + ua * ez[a];
            Px[b] += tb * ex[a] + ub * ex[b]; Py[b] += tb * ey[a] + ub * ey[b]; Pz[b] += tb * ez[a] + ub * ez[b];
        }

    // push P_ij to atom j's slot, accumulate the own halves
    T Fx = T(0), Fy = T(0), Fz = T(0);
    T W[9] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
    for (int a = 0; a < M; ++a) {
        const int m = slot[a];
        const int mm = REV[(int64_t)m * n + i];
        rm::store_rec(&Q[(int64_t)mm * n + jdx[a]], Px[a], Py[a], Pz[a]);
        Fx += Px[a]; Fy += Py[a]; Fz += Pz[a];
        if (virial) {
            const T rx = ex[a] * r[a], ry = ey[a] * r[a], rz = ez[a] * r[a];
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

template <class T, class Rec>
int launch(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
           const double box[3], const md_tersoff_params* hp, double* pe, double* f, double* virial,
           cudaStream_t s) {
    TersoffDev<T> p;
    p.A = (T)hp->A; p.B = (T)hp->B; p.lambda = (T)hp->lambda; p.mu = (T)hp->mu; p.beta = (T)hp->beta;
    p.n = (T)hp->n; p.h = (T)hp->h; p.R = (T)hp->R; p.S2 = (T)(hp->S * hp->S);
    p.c2 = (T)(hp->c * hp->c); p.d2 = (T)(hp->d * hp->d); p.c2_over_d2 = (T)((hp->c * hp->c) / (hp->d * hp->d));
    p.w = (T)(3.14159265358979323846 / (hp->S - hp->R));
    p.minus_half_over_n = (T)(-0.5 / hp->n);
    ProfScope prof(nl, MD_KIND_PAIR, 1, s);
    k_tersoff_pair<T, Rec><<<(unsigned)((n + 127) / 128), 128, 0, s>>>(
        n, x, y, z, box[0], box[1], box[2], nl->NN, nl->NL, nl->REV, p, (Rec*)nl->Q, nl->MASK,
        pe, f, virial, nl->d_status);
    MD_CUDA_TRY(cudaGetLastError());
    return MD_OK;
}

}  // namespace

int md_launch_tersoff(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                      const double* vx, const double* vy, const double* vz, const double box[3],
                      const md_tersoff_params* p, int precision, double* pe, double* f, double* virial,
                      double* heat, cudaStream_t s) {
    if (n == 0) return MD_OK;
    int rc = precision == MD_FP32 ? launch<float, float4>(nl, n, x, y, z, box, p, pe, f, virial, s)
                                  : launch<double, PairRec64>(nl, n, x, y, z, box, p, pe, f, virial, s);
    if (rc != MD_OK) return rc;
    return md_launch_gather(nl, n, x, y, z, vx, vy, vz, box, precision, f, virial, heat, s);
}
