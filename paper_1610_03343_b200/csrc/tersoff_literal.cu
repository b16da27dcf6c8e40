// tersoff_literal.cu -- the paper's own two-kernel scheme, kept as an A/B against the stored-P design of
// tersoff.cu (measured comparison in DESIGN.md section 4).
//
//   Algorithm 3  k_alg3: one thread per atom i; for every neighbour j: zeta_ij over the other
//       neighbours k, then b_ij and b'_ij = db_ij/dzeta_ij  ->  global memory, 16 bytes per listed pair.
//   Algorithm 2  k_alg2: one thread per atom i; for every neighbour j: dU_i/dr_ij (inner loop
//       over the neighbours of i) AND dU_j/dr_ji (inner loop over the neighbours of j, recomputed here instead of
//       being read from a record), F_ij = dU_i/dr_ij - dU_j/dr_ji (Eq. 14), and U_i, F_i, W_i, J_i accumulated in
//       registers: one store per atom, no per-pair force record, no gather kernel.
// As in the paper the geometry of a neighbour is formed again wherever it is needed (nothing is kept per
// neighbour between the loops), so the flop count is ~M times that of the stored-P kernels while the per-pair
// traffic is 16 bytes instead of 32 + 32.  Same formulas (T5), same fastmath.cuh functions.
#include "common.cuh"
#include "real_math.cuh"
#include "pair_sort.cuh"
#include "fastmath.cuh"

namespace {

template <class T>
struct LitDev { T A, B, lambda, mu, beta, n, h, R, S2, c2, d2, c2_over_d2, w, minus_half_over_n; };

template <class T> struct Geo { T ex, ey, ez, r, rinv, fc, fcp; bool in; };

// r_cq of the q-th listed neighbour of centre c, cut-off function and its derivative
template <class T>
__device__ __forceinline__ Geo<T>
geometry(unsigned c, unsigned q, unsigned n, double xc, double yc, double zc, const double* __restrict__ x,
         const double* __restrict__ y, const double* __restrict__ z, const ps::MinImage& mi,
         const int32_t* __restrict__ NL, const LitDev<T>& p, int* k_out) {
    const int k = NL[q * n + c];
    double dx = x[k] - xc, dy = y[k] - yc, dz = z[k] - zc;
    T d2 = ps::in_range_d2((T)dx, (T)dy, (T)dz);
    if (mi.far(d2)) { mi.wrap(dx, dy, dz); d2 = ps::in_range_d2((T)dx, (T)dy, (T)dz); }
    Geo<T> g;
    g.in = d2 < p.S2;
    const T ds = g.in ? d2 : T(1);
    g.rinv = fm::rsqrt(ds);
    g.r = ds * g.rinv;
    g.ex = (T)dx * g.rinv; g.ey = (T)dy * g.rinv; g.ez = (T)dz * g.rinv;
    g.fc = T(1); g.fcp = T(0);
    if (g.in && g.r > p.R) {                                 // f_C window R < r < S (reading A1)
        T sn, cs;
        fm::sincos_0_pi((g.r - p.R) * p.w, &sn, &cs);
        g.fc = T(0.5) + T(0.5) * cs;
        g.fcp = T(-0.5) * p.w * sn;
    }
    *k_out = k;
    return g;
}

// Algorithm 3: b_ij, b'_ij of every listed pair (zero pair outside the force range)
template <class T>
__global__ void __launch_bounds__(128)
k_alg3(unsigned n, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
       double Lx, double Ly, double Lz, const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
       LitDev<T> p, const double* __restrict__ gtab, double2* __restrict__ Bout) {
    __shared__ __align__(16) double s_tab[fm::TAB_DOUBLES];
    const fm::Tab tb = fm::stage_tables(s_tab, gtab);
    __syncthreads();
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const ps::MinImage mi = ps::make_min_image(Lx, Ly, Lz);
    const double xi = x[i], yi = y[i], zi = z[i];
    const int nn = NN[i];
    for (int m = 0; m < nn; ++m) {
        int j;
        const Geo<T> a = geometry<T>(i, m, n, xi, yi, zi, x, y, z, mi, NL, p, &j);
        T b = T(1), bp = T(0);
        if (a.in) {
            T zeta = T(0);
            for (int q = 0; q < nn; ++q) {                   // zeta_ij = sum_{k != j} f_C(r_ik) g_ijk  (Eq. 4)
                if (q == m) continue;
                int k;
                const Geo<T> c = geometry<T>(i, q, n, xi, yi, zi, x, y, z, mi, NL, p, &k);
                if (!c.in) continue;
                const T xx = p.h - (a.ex * c.ex + a.ey * c.ey + a.ez * c.ez);
                const T x2 = xx * xx;
                zeta += c.fc * (T(1) + p.c2_over_d2 * x2 * fm::rcp(p.d2 + x2));
            }
            if (zeta > T(0)) {                               // zeta = 0: b = 1, b' = 0 (reading A8)
                const T tt = fm::exp(p.n * fm::log(p.beta * zeta, tb), tb);
                b = fm::exp(p.minus_half_over_n * fm::log(T(1) + tt, tb), tb);       // Eq. (3)
                bp = T(-0.5) * b * tt * fm::rcp(zeta * (T(1) + tt));
            }
        }
        Bout[m * n + i] = make_double2((double)b, (double)bp);
    }
}

// P = dU_c/dr_ca for the a-th listed neighbour of centre c (T5), and U_ca / 2.  Reads b, b' of row c.
template <class T>
__device__ __forceinline__ bool
partial(unsigned c, unsigned a, unsigned n, const double* __restrict__ x, const double* __restrict__ y,
        const double* __restrict__ z, const ps::MinImage& mi, const int32_t* __restrict__ NN,
        const int32_t* __restrict__ NL, const double2* __restrict__ Bin, const LitDev<T>& p, const fm::Tab& tb,
        T* Px, T* Py, T* Pz, T* Uhalf, T* rx, T* ry, T* rz) {
    const double xc = x[c], yc = y[c], zc = z[c];
    int j;
    const Geo<T> ga = geometry<T>(c, a, n, xc, yc, zc, x, y, z, mi, NL, p, &j);
    if (!ga.in) return false;
    const double2 ba = Bin[a * n + c];
    const T fR = p.A * fm::exp(-p.lambda * ga.r, tb), fA = p.B * fm::exp(-p.mu * ga.r, tb);
    const T bfA = (T)ba.x * fA;
    const T ha = T(-0.5) * ga.fc * fA * (T)ba.y;
    T ce = T(0.5) * (ga.fcp * (fR - bfA) + ga.fc * (p.mu * bfA - p.lambda * fR));      // D
    T sx = T(0), sy = T(0), sz = T(0);
    const int nn = NN[c];
    for (int q = 0; q < nn; ++q) {
        if (q == (int)a) continue;
        int k;
        const Geo<T> gq = geometry<T>(c, q, n, xc, yc, zc, x, y, z, mi, NL, p, &k);
        if (!gq.in) continue;
        const T hq = T(-0.5) * gq.fc * p.B * fm::exp(-p.mu * gq.r, tb) * (T)Bin[q * n + c].y;
        const T cs = ga.ex * gq.ex + ga.ey * gq.ey + ga.ez * gq.ez;
        const T xx = p.h - cs;
        const T x2 = xx * xx;
        const T qq = fm::rcp(p.d2 + x2);
        const T gp = T(-2) * p.c2 * xx * qq * qq;            // dg/dcos
        const T ta = (ha * gq.fc + hq * ga.fc) * gp * ga.rinv;
        ce += hq * ga.fcp * (T(1) + p.c2_over_d2 * x2 * qq) - ta * cs;
        sx += ta * gq.ex; sy += ta * gq.ey; sz += ta * gq.ez;
    }
    *Px = sx + ce * ga.ex; *Py = sy + ce * ga.ey; *Pz = sz + ce * ga.ez;
    *Uhalf = T(0.5) * ga.fc * (fR - bfA);
    *rx = ga.ex * ga.r; *ry = ga.ey * ga.r; *rz = ga.ez * ga.r;
    return true;
}

// Algorithm 2: everything of atom i in one thread, one store per output
template <class T>
__global__ void __launch_bounds__(128)
k_alg2(unsigned n, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
       const double* __restrict__ vx, const double* __restrict__ vy, const double* __restrict__ vz,
       double Lx, double Ly, double Lz, const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
       const uint8_t* __restrict__ REV, LitDev<T> p, const double* __restrict__ gtab,
       const double2* __restrict__ Bin, double* __restrict__ pe, double* __restrict__ f,
       double* __restrict__ virial, double* __restrict__ heat) {
    __shared__ __align__(16) double s_tab[fm::TAB_DOUBLES];
    const fm::Tab tb = fm::stage_tables(s_tab, gtab);
    __syncthreads();
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const ps::MinImage mi = ps::make_min_image(Lx, Ly, Lz);
    T vxi = T(0), vyi = T(0), vzi = T(0);
    if (heat) { vxi = (T)vx[i]; vyi = (T)vy[i]; vzi = (T)vz[i]; }
    T U = T(0), Fx = T(0), Fy = T(0), Fz = T(0), Jx = T(0), Jy = T(0), Jz = T(0);
    T W[9] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
    const int nn = NN[i];
    for (int m = 0; m < nn; ++m) {
        T px, py, pz, uh, rx, ry, rz;
        if (!partial<T>(i, m, n, x, y, z, mi, NN, NL, Bin, p, tb, &px, &py, &pz, &uh, &rx, &ry, &rz)) continue;
        const unsigned j = (unsigned)NL[m * n + i];
        T qx, qy, qz, uj, sx, sy, sz;                        // dU_j/dr_ji, recomputed in this thread (Alg. 2 l.11)
        partial<T>(j, (unsigned)REV[m * n + i], n, x, y, z, mi, NN, NL, Bin, p, tb, &qx, &qy, &qz, &uj, &sx, &sy, &sz);
        const T fx = px - qx, fy = py - qy, fz = pz - qz;    // F_ij, Eq. (14)
        U += uh;
        Fx += fx; Fy += fy; Fz += fz;
        W[0] += rx * fx; W[1] += rx * fy; W[2] += rx * fz;
        W[3] += ry * fx; W[4] += ry * fy; W[5] += ry * fz;
        W[6] += rz * fx; W[7] += rz * fy; W[8] += rz * fz;
        const T dot = qx * vxi + qy * vyi + qz * vzi;
        Jx += rx * dot; Jy += ry * dot; Jz += rz * dot;
    }
    if (pe) pe[i] = (double)U;
    if (f) { f[i] = (double)Fx; f[n + i] = (double)Fy; f[2 * n + i] = (double)Fz; }
    if (virial) {
#pragma unroll
        for (int q = 0; q < 9; ++q) virial[(size_t)q * n + i] = (double)(T(-0.5) * W[q]);
    }
    if (heat) { heat[i] = (double)Jx; heat[n + i] = (double)Jy; heat[2 * n + i] = (double)Jz; }
}

template <class T>
int launch(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z, const double* vx,
           const double* vy, const double* vz, const double box[3], const md_tersoff_params* hp, double* pe,
           double* f, double* virial, double* heat, cudaStream_t s) {
    LitDev<T> p;
    p.A = (T)hp->A; p.B = (T)hp->B; p.lambda = (T)hp->lambda; p.mu = (T)hp->mu; p.beta = (T)hp->beta;
    p.n = (T)hp->n; p.h = (T)hp->h; p.R = (T)hp->R; p.S2 = (T)(hp->S * hp->S);
    p.c2 = (T)(hp->c * hp->c); p.d2 = (T)(hp->d * hp->d); p.c2_over_d2 = (T)((hp->c * hp->c) / (hp->d * hp->d));
    p.w = (T)(3.14159265358979323846 / (hp->S - hp->R));
    p.minus_half_over_n = (T)(-0.5 / hp->n);
    const double* gtab = md_math_tables();
    if (!gtab) return MD_ERR_ALLOC;
    const unsigned gb = (unsigned)((n + 127) / 128);
    {
        ProfScope prof(nl, MD_KIND_PAIR, 1, s);              // Algorithm 3
        k_alg3<T><<<gb, 128, 0, s>>>((unsigned)n, x, y, z, box[0], box[1], box[2], nl->NN, nl->NL, p, gtab,
                                     (double2*)nl->Q);
    }
    {
        ProfScope prof(nl, MD_KIND_GATHER, 1, s);            // Algorithm 2
        k_alg2<T><<<gb, 128, 0, s>>>((unsigned)n, x, y, z, vx, vy, vz, box[0], box[1], box[2], nl->NN, nl->NL, nl->REV,
                                     p, gtab, (const double2*)nl->Q, pe, f, virial, heat);
    }
    MD_CUDA_TRY(cudaGetLastError());
    return MD_OK;
}

}  // namespace

int md_launch_tersoff_literal(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                              const double* vx, const double* vy, const double* vz, const double box[3],
                              const md_tersoff_params* p, int precision, double* pe, double* f, double* virial,
                              double* heat, cudaStream_t s) {
    if (n == 0) return MD_OK;
    return precision == MD_FP32 ? launch<float>(nl, n, x, y, z, vx, vy, vz, box, p, pe, f, virial, heat, s)
                                : launch<double>(nl, n, x, y, z, vx, vy, vz, box, p, pe, f, virial, heat, s);
}
