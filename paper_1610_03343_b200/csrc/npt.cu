// npt.cu -- Berendsen weak coupling (thermostat + barostat), the paper's benchmark ensemble (PAPER.md:355:
// "NPT ensemble ... Berendsen"), reading A18.  Consumes sum_i W_i.
//   k_npt_partial / k_npt_final  sum_i |v_i|^2 and sum_i (W_xx + W_yy + W_zz): fixed grid, fixed order, no
//                                atomics -> the same bits run to run
//   k_npt_scale                  v *= lambda;  x *= mu
#include "common.cuh"

namespace {
constexpr int RED_BLOCKS = 296, RED_BT = 256;

__global__ void __launch_bounds__(RED_BT)
k_npt_partial(int64_t n, double* __restrict__ vx, double* __restrict__ vy, double* __restrict__ vz,
              const double* __restrict__ W, const double* __restrict__ f, double hk, double* __restrict__ part) {
    __shared__ double s_a[RED_BT / 32], s_b[RED_BT / 32];
    double a = 0.0, b = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * RED_BT + threadIdx.x; i < n; i += (int64_t)RED_BLOCKS * RED_BT) {
        double ux = vx[i], uy = vy[i], uz = vz[i];
        if (f) {                                             // the step's second half-kick, fused (as k_kick, bit for bit)
            ux = __fma_rn(hk, f[i], ux); uy = __fma_rn(hk, f[n + i], uy); uz = __fma_rn(hk, f[2 * n + i], uz);
            vx[i] = ux; vy[i] = uy; vz[i] = uz;
        }
        a += ux * ux + uy * uy + uz * uz;
        b += W[i] + W[4 * n + i] + W[8 * n + i];
    }
    for (int d = 16; d > 0; d >>= 1) { a += __shfl_down_sync(0xffffffffu, a, d); b += __shfl_down_sync(0xffffffffu, b, d); }
    if ((threadIdx.x & 31) == 0) { s_a[threadIdx.x >> 5] = a; s_b[threadIdx.x >> 5] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double ta = 0.0, tb = 0.0;
        for (int w = 0; w < RED_BT / 32; ++w) { ta += s_a[w]; tb += s_b[w]; }
        part[2 * blockIdx.x] = ta; part[2 * blockIdx.x + 1] = tb;
    }
}
// out = {sum v^2, tr sum W^own, lam, mu, Lx mu, Ly mu, Lz mu} (reading A18; the total virial is twice the
// sum of the own halves, api.cu md_npt_run).  The factors are formed here so that the next step's kick + drift
// (k_kick_drift_dev) can start without the host; the host takes lam, mu and the box from this record, not from a
// computation of its own, so both sides hold the same bits.
__global__ void k_npt_final(const double* __restrict__ part, double* __restrict__ out, double n_atoms, double mass_over_kappa,
                            double dt, double bx, double by, double bz, md_berendsen_params b) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    double ta = 0.0, tb = 0.0;
    for (int k = 0; k < RED_BLOCKS; ++k) { ta += part[2 * k]; tb += part[2 * k + 1]; }
    out[0] = ta; out[1] = tb;
    const double ke2 = ta * mass_over_kappa;                                      // 2 KE
    const double V = bx * by * bz;
    const double T = ke2 / (3.0 * n_atoms * MD_KB), P = (ke2 + 2.0 * tb) / (3.0 * V);
    const double lam = T > 0 ? sqrt(1.0 + dt / b.tau_T * (b.T0 / T - 1.0)) : 1.0;
    const double mu = cbrt(1.0 - b.beta * dt / b.tau_P * (b.P0 - P));
    out[2] = lam; out[3] = mu; out[4] = bx * mu; out[5] = by * mu; out[6] = bz * mu;
}
__global__ void k_npt_scale(int64_t n, double* __restrict__ x, double* __restrict__ y, double* __restrict__ z,
                            double* __restrict__ vx, double* __restrict__ vy, double* __restrict__ vz,
                            double lam, double mu) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    vx[i] *= lam; vy[i] *= lam; vz[i] *= lam;
    x[i] *= mu; y[i] *= mu; z[i] *= mu;
}
}  // namespace

// f != nullptr: v += hk f first (the velocity-Verlet kick that ends the step), in the same pass
int md_launch_npt_sums(md_neighbors* nl, int64_t n, double* vx, double* vy, double* vz,
                       const double* W, const double* f, double hk, double mass, double dt, const double box[3],
                       const md_berendsen_params* b, cudaStream_t s) {
    ProfScope prof(nl, MD_KIND_INTEGRATE, 2, s);
    if (!nl->npt_event) MD_CUDA_TRY(cudaEventCreateWithFlags(&nl->npt_event, cudaEventDisableTiming));
    double* out = nl->npt_part + 2 * RED_BLOCKS;
    k_npt_partial<<<RED_BLOCKS, RED_BT, 0, s>>>(n, vx, vy, vz, W, f, hk, nl->npt_part);
    k_npt_final<<<1, 32, 0, s>>>(nl->npt_part, out, (double)n, mass / MD_KAPPA, dt, box[0], box[1], box[2], *b);
    MD_CUDA_TRY(cudaMemcpyAsync(nl->h_npt, out, 7 * sizeof(double), cudaMemcpyDeviceToHost, s));
    MD_CUDA_TRY(cudaEventRecord(nl->npt_event, s));
    return MD_OK;
}
int md_npt_sums_wait(md_neighbors* nl, double out[7]) {
    MD_CUDA_TRY(cudaEventSynchronize(nl->npt_event));
    for (int q = 0; q < 7; ++q) out[q] = nl->h_npt[q];
    return MD_OK;
}
const double* md_npt_scal(md_neighbors* nl) { return nl->npt_part + 2 * RED_BLOCKS; }
int md_launch_npt_scale(md_neighbors* nl, int64_t n, double* x, double* y, double* z, double* vx, double* vy,
                        double* vz, double lam, double mu, cudaStream_t s) {
    ProfScope prof(nl, MD_KIND_INTEGRATE, 1, s);
    k_npt_scale<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, x, y, z, vx, vy, vz, lam, mu);
    MD_CUDA_TRY(cudaGetLastError());
    return MD_OK;
}

// ---- Green-Kubo workload: J_pot = sum_i J_i and J_kin = sum_i (m v_i^2 / 2 + U_i) v_i, same fixed-order scheme
namespace {
__global__ void __launch_bounds__(RED_BT)
k_heat_partial(int64_t n, const double* __restrict__ vx, const double* __restrict__ vy, const double* __restrict__ vz,
               const double* __restrict__ pe, const double* __restrict__ J, double half_m, double* __restrict__ part) {
    __shared__ double s_v[6][RED_BT / 32];
    double a[6] = {0, 0, 0, 0, 0, 0};
    for (int64_t i = (int64_t)blockIdx.x * RED_BT + threadIdx.x; i < n; i += (int64_t)RED_BLOCKS * RED_BT) {
        const double ux = vx[i], uy = vy[i], uz = vz[i];
        const double e = half_m * (ux * ux + uy * uy + uz * uz) + pe[i];
        a[0] += J[i]; a[1] += J[n + i]; a[2] += J[2 * n + i];
        a[3] += e * ux; a[4] += e * uy; a[5] += e * uz;
    }
#pragma unroll
    for (int q = 0; q < 6; ++q) {
        for (int d = 16; d > 0; d >>= 1) a[q] += __shfl_down_sync(0xffffffffu, a[q], d);
        if ((threadIdx.x & 31) == 0) s_v[q][threadIdx.x >> 5] = a[q];
    }
    __syncthreads();
    if (threadIdx.x < 6) {
        double t = 0.0;
        for (int w = 0; w < RED_BT / 32; ++w) t += s_v[threadIdx.x][w];
        part[6 * blockIdx.x + threadIdx.x] = t;
    }
}
__global__ void k_heat_final(const double* __restrict__ part, double* __restrict__ out) {
    if (blockIdx.x != 0 || threadIdx.x >= 6) return;
    double t = 0.0;
    for (int k = 0; k < RED_BLOCKS; ++k) t += part[6 * k + threadIdx.x];
    out[threadIdx.x] = t;
}
}  // namespace

// HOST out[6] = J_pot (3), J_kin (3); synchronises the stream
int md_launch_heat_sums(md_neighbors* nl, int64_t n, const double* vx, const double* vy, const double* vz,
                        const double* pe, const double* J, double mass, double out[6], cudaStream_t s) {
    ProfScope prof(nl, MD_KIND_INTEGRATE, 2, s);
    k_heat_partial<<<RED_BLOCKS, RED_BT, 0, s>>>(n, vx, vy, vz, pe, J, 0.5 * mass / MD_KAPPA, nl->npt_part);
    k_heat_final<<<1, 32, 0, s>>>(nl->npt_part, nl->npt_part + 6 * RED_BLOCKS);
    MD_CUDA_TRY(cudaMemcpyAsync(nl->h_npt, nl->npt_part + 6 * RED_BLOCKS, 6 * sizeof(double), cudaMemcpyDeviceToHost, s));
    MD_CUDA_TRY(cudaStreamSynchronize(s));
    for (int q = 0; q < 6; ++q) out[q] = nl->h_npt[q];
    return MD_OK;
}
int md_npt_scratch_doubles() { return 6 * RED_BLOCKS + 6; }
