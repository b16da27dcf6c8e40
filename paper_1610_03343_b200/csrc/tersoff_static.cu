// tersoff_static.cu -- md_tersoff_force_static: Tersoff energies and forces by the stored-P scheme (per-pair record
// P_ij = dU_i/dr_ij written by thread i, gathered without atomics as F_i = sum_j (P_ij - P_ji)
// Eq. 14 and Eq. 28 at PAPER.md:330) for callers that may not allocate: code under CUDA graph capture, serving
// loops, harnesses that forbid cudaMalloc.
//
// The handle-based path keeps its records in memory that md_neighbors_create allocates.  Here the records live in
// ONE file-scope device array of fixed size (g_scratch below, 16 MiB + 256 bytes, held by every device that loads
// the library until the process exits); the call takes the list, the positions and the outputs from the caller and
// calls no cudaMalloc / cudaFree and no allocating library routine.  The tables of fastmath.cuh travel as a kernel
// argument (1.5 kB) instead of through md_math_tables(), which allocates on first use.
//
// The array is shared by every call on a device and keeps what the last call left in it:
//   - the status word is cleared at the start of every call (cudaMemsetAsync on the caller's stream);
//   - the records a call reads are all written by that call first (slot m of atom i for every m < NN[i]);
//   - two calls that overlap on one GPU (different streams, or host threads with their own streams) RACE on it.
//     Calls on one stream, or ordered by events, are safe.
// Self-contained on purpose: it shares fastmath.cuh and common.cuh with the other kernels and nothing else.
#include <cmath>
#include <mutex>

#include "common.cuh"
#include "fastmath.cuh"

namespace {

// ---- the scratch -------------------------------------------------------------------------------------------------
struct __align__(32) Rec { double x, y, z, h; };      // pass 1: {b_ij, -, -, h_ij}; pass 2: {P_ij, h_ij}
constexpr size_t OFF_STATUS = 0;                      // int: MD_DEV_* bits of the running call
constexpr size_t OFF_REC = 256;                       // Rec[max_neighbors][n], neighbour-major like NL
constexpr size_t SCRATCH_BYTES = OFF_REC + sizeof(Rec) * (size_t)MD_STATIC_MAX_PAIRS;

static __device__ __align__(256) unsigned char g_scratch[SCRATCH_BYTES];

// In host code `g_scratch` is only a handle for the runtime, not a device address: the address every launch uses
// comes from cudaGetSymbolAddress, once per device, with that device current.
constexpr int MAX_DEV = 64;
unsigned char* g_base[MAX_DEV];
std::mutex g_mu;

int scratch_base(unsigned char** out) {
    int dev = 0;
    MD_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEV) return MD_ERR_ARG;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_base[dev]) {
        void* p = nullptr;
        MD_CUDA_TRY(cudaGetSymbolAddress(&p, g_scratch));
        if (!p) return MD_ERR_CUDA;
        g_base[dev] = static_cast<unsigned char*>(p);
    }
    *out = g_base[dev];
    return MD_OK;
}

// ---- tables of fastmath.cuh as a kernel argument -------------------------------------------------------------------
struct MathTabArg { double v[fm::TAB_DOUBLES]; };

const MathTabArg& host_tables() {                      // same values as mathtab.cu, computed once per process
    static MathTabArg t;
    static std::once_flag once;
    std::call_once(once, [] {
        for (int j = 0; j < fm::EXP_N; ++j) t.v[j] = (double)exp2l((long double)j / fm::EXP_N);
        for (int j = 0; j < fm::LOG_N; ++j) {
            const long double centre = 1.0L + ((long double)j + 0.5L) / fm::LOG_N;
            const double c = (double)(1.0L / centre);
            t.v[fm::EXP_N + 2 * j] = c;
            t.v[fm::EXP_N + 2 * j + 1] = (double)(-logl((long double)c));
        }
    });
    return t;
}

__device__ __forceinline__ fm::Tab stage_arg_tables(double* smem, const MathTabArg& a) {
    for (int k = threadIdx.x; k < fm::TAB_DOUBLES; k += blockDim.x) smem[k] = a.v[k];
    fm::Tab t;
    t.e = smem;
    t.l = reinterpret_cast<const double2*>(smem + fm::EXP_N);
    return t;
}

// ---- device side -------------------------------------------------------------------------------------------------
struct Par { double A, B, lambda, mu, beta, n, h, R, S2, c2, d2, c2_over_d2, w, minus_half_over_n; };
struct Box { double L[3], half[3]; };

struct Geo { double ex, ey, ez, r, rinv, fc, fcp; bool in; };

// r_ik of the q-th listed neighbour k of atom i (minimum image), f_C and f_C' (Eq. 6, reading A1)
__device__ __forceinline__ Geo geometry(unsigned i, int q, unsigned n, double xi, double yi, double zi,
                                        const double* __restrict__ x, const double* __restrict__ y,
                                        const double* __restrict__ z, const Box& bx,
                                        const int32_t* __restrict__ NL, const Par& p) {
    const int k = NL[(size_t)q * n + i];
    const double dx = md_min_image(x[k] - xi, bx.L[0], bx.half[0]);
    const double dy = md_min_image(y[k] - yi, bx.L[1], bx.half[1]);
    const double dz = md_min_image(z[k] - zi, bx.L[2], bx.half[2]);
    const double d2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
    Geo g;
    g.in = d2 < p.S2;
    const double ds = g.in ? d2 : 1.0;
    g.rinv = fm::rsqrt(ds);
    g.r = ds * g.rinv;
    g.ex = dx * g.rinv; g.ey = dy * g.rinv; g.ez = dz * g.rinv;
    g.fc = 1.0; g.fcp = 0.0;
    if (g.in && g.r > p.R) {
        double sn, cs;
        fm::sincos_0_pi((g.r - p.R) * p.w, &sn, &cs);
        g.fc = 0.5 + 0.5 * cs;
        g.fcp = -0.5 * p.w * sn;
    }
    return g;
}

// One thread per atom i, two passes over its row; `rec` is read back by the thread that wrote it (plain loads).
//   pass 1: zeta_ij (Eq. 4), b_ij (Eq. 3) and h_ij = -1/2 f_C(r_ij) f_A(r_ij) db_ij/dzeta_ij     -> rec[m][i] = {b, ., ., h}
//   pass 2: P_ij = dU_i/dr_ij with U_i = 1/2 sum_j f_C(r_ij) [f_R(r_ij) - b_ij f_A(r_ij)] (Eqs. 1, 2), which needs
//           h of every other slot of the row                                                    -> rec[m][i] = {P, h}
__global__ void __launch_bounds__(128)
k_static_pair(unsigned n, int K, const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
              const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z, Box bx,
              Par p, MathTabArg tab, Rec* rec, int* status, double* __restrict__ pe) {
    __shared__ __align__(16) double s_tab[fm::TAB_DOUBLES];
    const fm::Tab tb = stage_arg_tables(s_tab, tab);
    __syncthreads();
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int nn = NN[i];
    if (nn > K) { atomicOr(status, MD_DEV_ROW_OVERFLOW); nn = K; }
    if (nn < 0) nn = 0;
    for (int m = 0; m < nn; ++m)                       // an index outside [0, n) ends the row there
        if ((unsigned)NL[(size_t)m * n + i] >= n) { atomicOr(status, MD_DEV_NO_REVERSE); nn = m; break; }
    const double xi = x[i], yi = y[i], zi = z[i];
    for (int m = 0; m < nn; ++m) {
        const Geo a = geometry(i, m, n, xi, yi, zi, x, y, z, bx, NL, p);
        Rec r = {1.0, 0.0, 0.0, 0.0};
        if (a.in) {
            double zeta = 0.0;
            for (int q = 0; q < nn; ++q) {
                if (q == m) continue;
                const Geo c = geometry(i, q, n, xi, yi, zi, x, y, z, bx, NL, p);
                if (!c.in) continue;
                const double xx = p.h - (a.ex * c.ex + a.ey * c.ey + a.ez * c.ez);
                const double x2 = xx * xx;
                zeta += c.fc * (1.0 + p.c2_over_d2 * x2 * fm::rcp(p.d2 + x2));          // f_C(r_ik) g(theta_ijk), Eq. 5
            }
            if (zeta > 0.0) {                                                          // zeta = 0: b = 1, b' = 0 (A8)
                const double tt = fm::exp(p.n * fm::log(p.beta * zeta, tb), tb);
                r.x = fm::exp(p.minus_half_over_n * fm::log(1.0 + tt, tb), tb);
                const double bp = -0.5 * r.x * tt * fm::rcp(zeta * (1.0 + tt));
                r.h = -0.5 * a.fc * p.B * fm::exp(-p.mu * a.r, tb) * bp;
            }
        }
        rec[(size_t)m * n + i] = r;
    }
    double U = 0.0;
    for (int m = 0; m < nn; ++m) {
        const Geo a = geometry(i, m, n, xi, yi, zi, x, y, z, bx, NL, p);
        const Rec own = rec[(size_t)m * n + i];
        Rec out = {0.0, 0.0, 0.0, own.h};
        if (a.in) {
            const double fR = p.A * fm::exp(-p.lambda * a.r, tb), fA = p.B * fm::exp(-p.mu * a.r, tb);
            const double bfA = own.x * fA;
            double ce = 0.5 * (a.fcp * (fR - bfA) + a.fc * (p.mu * bfA - p.lambda * fR));
            double sx = 0.0, sy = 0.0, sz = 0.0;
            for (int q = 0; q < nn; ++q) {
                if (q == m) continue;
                const Geo c = geometry(i, q, n, xi, yi, zi, x, y, z, bx, NL, p);
                if (!c.in) continue;
                const double hq = rec[(size_t)q * n + i].h;
                const double cs = a.ex * c.ex + a.ey * c.ey + a.ez * c.ez;
                const double xx = p.h - cs;
                const double x2 = xx * xx;
                const double qq = fm::rcp(p.d2 + x2);
                const double gp = -2.0 * p.c2 * xx * qq * qq;                            // dg/dcos(theta)
                const double ta = (own.h * c.fc + hq * a.fc) * gp * a.rinv;
                ce += hq * a.fcp * (1.0 + p.c2_over_d2 * x2 * qq) - ta * cs;
                sx += ta * c.ex; sy += ta * c.ey; sz += ta * c.ez;
            }
            out.x = sx + ce * a.ex; out.y = sy + ce * a.ey; out.z = sz + ce * a.ez;
            U += 0.5 * a.fc * (fR - bfA);
        }
        rec[(size_t)m * n + i] = out;
    }
    if (pe) pe[i] = U;
}

// F_i = sum_j (P_ij - P_ji), Eq. 28: one thread per atom, one store per component.  The slot of i in
// row j is found by scanning that row (the handle-based path keeps a reverse index instead).
__global__ void __launch_bounds__(128)
k_static_gather(unsigned n, int K, const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
                const Rec* __restrict__ rec, int* status, double* __restrict__ f) {
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int nn = max(0, min(NN[i], K));
    double Fx = 0.0, Fy = 0.0, Fz = 0.0;
    bool lost = false;
    for (int m = 0; m < nn; ++m) {
        const unsigned j = (unsigned)NL[(size_t)m * n + i];
        if (j >= n) { lost = true; continue; }
        const int nj = max(0, min(NN[j], K));
        int mr = -1;
        for (int q = 0; q < nj; ++q)
            if ((unsigned)NL[(size_t)q * n + j] == i) { mr = q; break; }
        if (mr < 0) { lost = true; continue; }
        const Rec a = rec[(size_t)m * n + i], b = rec[(size_t)mr * n + j];
        Fx += a.x - b.x; Fy += a.y - b.y; Fz += a.z - b.z;
    }
    if (lost) {
        atomicOr(status, MD_DEV_NO_REVERSE);
        Fx = Fy = Fz = __longlong_as_double(0x7ff8000000000000LL);
    }
    f[i] = Fx; f[n + i] = Fy; f[2 * (size_t)n + i] = Fz;
}

}  // namespace

extern "C" int md_tersoff_force_static(int64_t n, int max_neighbors, const int32_t* NN, const int32_t* NL,
                                       const double* x, const double* y, const double* z, const double box[3],
                                       const md_tersoff_params* hp, double* pe, double* f, int32_t* status,
                                       void* stream) {
    if (n < 0 || max_neighbors < 1 || max_neighbors > MD_MAX_NEIGHBORS || !box || !hp) return MD_ERR_ARG;
    if (n > 0 && (!NN || !NL || !x || !y || !z)) return MD_ERR_ARG;
    if (!(box[0] > 0.0 && box[1] > 0.0 && box[2] > 0.0) || !(hp->S > hp->R) || !(hp->n > 0.0) || !(hp->d != 0.0))
        return MD_ERR_ARG;
    if (n * (int64_t)max_neighbors > (int64_t)MD_STATIC_MAX_PAIRS) return MD_ERR_STATIC_CAPACITY;
    cudaStream_t s = (cudaStream_t)stream;
    unsigned char* base = nullptr;
    const int rc = scratch_base(&base);
    if (rc != MD_OK) return rc;
    int* d_status = reinterpret_cast<int*>(base + OFF_STATUS);
    Rec* rec = reinterpret_cast<Rec*>(base + OFF_REC);
    MD_CUDA_TRY(cudaMemsetAsync(d_status, 0, sizeof(int), s));       // the last call's bits must not leak into this one
    if (n > 0) {
        Par p;
        p.A = hp->A; p.B = hp->B; p.lambda = hp->lambda; p.mu = hp->mu; p.beta = hp->beta; p.n = hp->n; p.h = hp->h;
        p.R = hp->R; p.S2 = hp->S * hp->S; p.c2 = hp->c * hp->c; p.d2 = hp->d * hp->d;
        p.c2_over_d2 = (hp->c * hp->c) / (hp->d * hp->d);
        p.w = 3.14159265358979323846 / (hp->S - hp->R);
        p.minus_half_over_n = -0.5 / hp->n;
        Box bx;
        for (int a = 0; a < 3; ++a) { bx.L[a] = box[a]; bx.half[a] = 0.5 * box[a]; }
        const unsigned gb = (unsigned)((n + 127) / 128);
        k_static_pair<<<gb, 128, 0, s>>>((unsigned)n, max_neighbors, NN, NL, x, y, z, bx, p, host_tables(), rec,
                                         d_status, pe);
        if (f) k_static_gather<<<gb, 128, 0, s>>>((unsigned)n, max_neighbors, NN, NL, rec, d_status, f);
        MD_CUDA_TRY(cudaGetLastError());
    }
    if (status) MD_CUDA_TRY(cudaMemcpyAsync(status, d_status, sizeof(int), cudaMemcpyDeviceToDevice, s));
    return MD_OK;
}
