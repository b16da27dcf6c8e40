// integrate.cu -- velocity-Verlet half steps, pure streaming.
#include "common.cuh"

namespace {

__global__ void k_kick_drift(int64_t n, double* __restrict__ x, double* __restrict__ y, double* __restrict__ z,
                             double* __restrict__ vx, double* __restrict__ vy, double* __restrict__ vz,
                             const double* __restrict__ f, double hk, double dt, double Lx, double Ly, double Lz,
                             double lam, double mu) {
    // lam, mu: the weak-coupling scaling of the step before (md_npt_run), applied first; 1.0 (exact) otherwise
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double ux = __fma_rn(hk, f[i], __dmul_rn(vx[i], lam)), uy = __fma_rn(hk, f[n + i], __dmul_rn(vy[i], lam)),
                 uz = __fma_rn(hk, f[2 * n + i], __dmul_rn(vz[i], lam));
    vx[i] = ux; vy[i] = uy; vz[i] = uz;
    x[i] = md_wrap(__fma_rn(dt, ux, __dmul_rn(x[i], mu)), Lx);
    y[i] = md_wrap(__fma_rn(dt, uy, __dmul_rn(y[i], mu)), Ly);
    z[i] = md_wrap(__fma_rn(dt, uz, __dmul_rn(z[i], mu)), Lz);
}

// The same pass with lam, mu and the box taken from device memory: scal = {.., .., lam, mu, Lx, Ly, Lz} as
// k_npt_final (npt.cu) leaves them, so that md_npt_run can enqueue the next step's kick + drift before the host
// has read the step's temperature and pressure.
__global__ void k_kick_drift_dev(int64_t n, double* __restrict__ x, double* __restrict__ y, double* __restrict__ z,
                                 double* __restrict__ vx, double* __restrict__ vy, double* __restrict__ vz,
                                 const double* __restrict__ f, double hk, double dt, const double* scal) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double lam = scal[2], mu = scal[3], Lx = scal[4], Ly = scal[5], Lz = scal[6];
    const double ux = __fma_rn(hk, f[i], __dmul_rn(vx[i], lam)), uy = __fma_rn(hk, f[n + i], __dmul_rn(vy[i], lam)),
                 uz = __fma_rn(hk, f[2 * n + i], __dmul_rn(vz[i], lam));
    vx[i] = ux; vy[i] = uy; vz[i] = uz;
    x[i] = md_wrap(__fma_rn(dt, ux, __dmul_rn(x[i], mu)), Lx);
    y[i] = md_wrap(__fma_rn(dt, uy, __dmul_rn(y[i], mu)), Ly);
    z[i] = md_wrap(__fma_rn(dt, uz, __dmul_rn(z[i], mu)), Lz);
}

__global__ void k_kick(int64_t n, double* __restrict__ vx, double* __restrict__ vy, double* __restrict__ vz,
                       const double* __restrict__ f, double hk) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    vx[i] = __fma_rn(hk, f[i], vx[i]);
    vy[i] = __fma_rn(hk, f[n + i], vy[i]);
    vz[i] = __fma_rn(hk, f[2 * n + i], vz[i]);
}
}  // namespace

int md_launch_vv(md_neighbors* nl, int phase, int64_t n, double* x, double* y, double* z, double* vx, double* vy, double* vz,
                 const double* f, double mass, double dt, const double box[3], cudaStream_t s, double lam, double mu) {
    if (n == 0) return MD_OK;
    const double hk = 0.5 * dt * MD_KAPPA / mass;
    const unsigned gb = (unsigned)((n + 255) / 256);
    ProfScope prof(nl, MD_KIND_INTEGRATE, 1, s);
    if (phase == 0) k_kick_drift<<<gb, 256, 0, s>>>(n, x, y, z, vx, vy, vz, f, hk, dt, box[0], box[1], box[2], lam, mu);
    else k_kick<<<gb, 256, 0, s>>>(n, vx, vy, vz, f, hk);
    MD_CUDA_TRY(cudaGetLastError());
    return MD_OK;
}

int md_launch_vv_dev(md_neighbors* nl, int64_t n, double* x, double* y, double* z, double* vx, double* vy, double* vz,
                     const double* f, double mass, double dt, const double* d_scal, cudaStream_t s) {
    if (n == 0) return MD_OK;
    const double hk = 0.5 * dt * MD_KAPPA / mass;
    ProfScope prof(nl, MD_KIND_INTEGRATE, 1, s);
    k_kick_drift_dev<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, x, y, z, vx, vy, vz, f, hk, dt, d_scal);
    MD_CUDA_TRY(cudaGetLastError());
    return MD_OK;
}
