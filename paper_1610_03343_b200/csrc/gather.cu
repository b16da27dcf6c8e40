// gather.cu -- step C: one thread per atom, no atomics (Algorithm 2 lines 12-17, PAPER.md:278-291;
// Eqs. 28-30).
//
// The pair kernel left in f / virial the "own" halves  sum_j P_ij  and  -1/2 sum_j r_ij (x) P_ij,
// and pushed P_ji into row i of Q.  Thread i reads its row (coalesced 32-byte records) and finishes
//   F_i  = sum_j P_ij - sum_j P_ji
//   W_i  = -1/2 sum_j r_ij (x) P_ij + 1/2 sum_j r_ij (x) P_ji
//   J_i  = sum_j r_ij (P_ji . v_i)
#include "common.cuh"
#include "real_math.cuh"

namespace {

// GEOM = false: forces only.  GEOM = true: virial and / or heat current too, which need r_ij of every in-range
// neighbour (list entry -> coordinates, two dependent loads).  The first four record slots -- and, where the slot is
// the list position (crystal kernels), their list entries -- are requested before MASK has arrived, the four
// neighbours' coordinates together after it; only rows with more than four in-range neighbours enter the loop.
// Sums run over the in-range slots in ascending order (as in k_gather_vv: bit-identical forces).
template <class T, class Rec, bool GEOM>
__global__ void __launch_bounds__(128)
k_gather(int64_t n, int K, const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
         const double* __restrict__ vx, const double* __restrict__ vy, const double* __restrict__ vz,
         double Lx, double Ly, double Lz, const int32_t* __restrict__ NL, const Rec* Q,
         const unsigned long long* MASK, int dense, double* f, double* virial,    // Q, MASK, f, virial: plain loads --
         double* __restrict__ heat) {                                              // the pair kernel before wrote them
    const int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t i = i0 < n ? i0 : n - 1;
    // Launched as a programmatic dependent of the pair kernel (common.cuh, md_launch_pdl): what that kernel does
    // not write -- the list entries of the first four slots, the atom's position and velocity -- is requested
    // while it drains.
    int hj[4];
#pragma unroll
    for (int sl = 0; sl < 4; ++sl) hj[sl] = GEOM ? NL[(int64_t)(sl < K ? sl : 0) * n + i] : 0;   // slot = list position
    double xi = 0, yi = 0, zi = 0;
    T vxi = T(0), vyi = T(0), vzi = T(0);
    if (GEOM) { xi = x[i]; yi = y[i]; zi = z[i]; }
    if (GEOM && heat) { vxi = (T)vx[i]; vyi = (T)vy[i]; vzi = (T)vz[i]; }
    md_grid_wait();
    md_grid_release();
    if (i0 >= n) return;
    T hx[4], hy[4], hz[4];
#pragma unroll
    for (int sl = 0; sl < 4; ++sl) rm::load_rec_once(&Q[(int64_t)(sl < K ? sl : 0) * n + i], &hx[sl], &hy[sl], &hz[sl]);
    unsigned long long mask = MASK[i];
    // own halves the pair kernel left (read-modify-write at the end): requested now, not after the arithmetic
    double of[3] = {0, 0, 0}, ow[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    if (f) { of[0] = rm::load_once(&f[i]); of[1] = rm::load_once(&f[n + i]); of[2] = rm::load_once(&f[2 * n + i]); }
    if (GEOM && virial) {
#pragma unroll
        for (int q = 0; q < 9; ++q) ow[q] = rm::load_once(&virial[(int64_t)q * n + i]);
    }
    T Fx = T(0), Fy = T(0), Fz = T(0);
    T W[9] = {T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0)};
    T Jx = T(0), Jy = T(0), Jz = T(0);
    auto geom_terms = [&](T px, T py, T pz, double qx, double qy, double qz) {
        const T rx = (T)md_min_image(qx - xi, Lx, 0.5 * Lx);
        const T ry = (T)md_min_image(qy - yi, Ly, 0.5 * Ly);
        const T rz = (T)md_min_image(qz - zi, Lz, 0.5 * Lz);
        if (virial) {
            W[0] += rx * px; W[1] += rx * py; W[2] += rx * pz;
            W[3] += ry * px; W[4] += ry * py; W[5] += ry * pz;
            W[6] += rz * px; W[7] += rz * py; W[8] += rz * pz;
        }
        if (heat) {
            const T dot = px * vxi + py * vyi + pz * vzi;
            Jx += rx * dot; Jy += ry * dot; Jz += rz * dot;
        }
    };
    // the first four slots
    const int cnt = __popcll(mask);
    bool use[4];
    double qx[4], qy[4], qz[4];
    {
        unsigned long long run = mask;
#pragma unroll
        for (int sl = 0; sl < 4; ++sl) {
            use[sl] = dense ? sl < cnt : (mask >> sl & 1ull) != 0;
            if (GEOM) {
                int j = hj[sl];
                if (dense) {                                 // slot sl holds the sl-th in-range list entry
                    const int m = run ? __ffsll((long long)run) - 1 : 0;
                    run &= run - 1;
                    j = NL[(int64_t)m * n + i];
                }
                j = use[sl] ? j : (int)i;
                qx[sl] = x[j]; qy[sl] = y[j]; qz[sl] = z[j];
            }
        }
    }
#pragma unroll
    for (int sl = 0; sl < 4; ++sl)
        if (use[sl]) {
            Fx += hx[sl]; Fy += hy[sl]; Fz += hz[sl];
            if (GEOM) geom_terms(hx[sl], hy[sl], hz[sl], qx[sl], qy[sl], qz[sl]);
        }
    // rows with more in-range neighbours
    if (dense) {
        unsigned long long run = mask;
        for (int sl = 0; sl < 4 && run; ++sl) run &= run - 1;
        for (int sl = 4; sl < cnt; ++sl) {
            const int m = __ffsll((long long)run) - 1;
            run &= run - 1;
            T px, py, pz;
            rm::load_rec_once(&Q[(int64_t)sl * n + i], &px, &py, &pz);
            Fx += px; Fy += py; Fz += pz;
            if (GEOM) {
                const int j = NL[(int64_t)m * n + i];
                geom_terms(px, py, pz, x[j], y[j], z[j]);
            }
        }
    } else {
        mask &= ~15ull;
        while (mask) {
            const int m = __ffsll((long long)mask) - 1;
            mask &= mask - 1;
            T px, py, pz;
            rm::load_rec_once(&Q[(int64_t)m * n + i], &px, &py, &pz);
            Fx += px; Fy += py; Fz += pz;
            if (GEOM) {
                const int j = NL[(int64_t)m * n + i];
                geom_terms(px, py, pz, x[j], y[j], z[j]);
            }
        }
    }
    if (f) {
        f[i] = of[0] - (double)Fx; f[n + i] = of[1] - (double)Fy; f[2 * n + i] = of[2] - (double)Fz;
    }
    if (GEOM && virial) {
#pragma unroll
        for (int q = 0; q < 9; ++q) virial[(int64_t)q * n + i] = ow[q] + (double)(T(0.5) * W[q]);
    }
    if (GEOM && heat) { heat[i] = (double)Jx; heat[n + i] = (double)Jy; heat[2 * n + i] = (double)Jz; }
}

// The same force sum with the velocity-Verlet half steps that follow it fused in (md_nve_run only, where
// neither virial nor heat current is asked for): F_i is complete in registers, so the second half-kick of
// this step and, unless it is the last step, the next step's kick + drift + wrap are applied before
// anything is stored.  The arithmetic is operation for operation that of k_gather followed by k_kick and
// k_kick_drift (integrate.cu), so the trajectory is bit-identical to the unfused composition.
#ifndef MD_GVV_BT
#define MD_GVV_BT 128
#endif
template <class T, class Rec, int MODE>
#ifndef MD_GVV_CPS
#define MD_GVV_CPS 4          // no tighter register cap: 8 CTAs per SM (64 registers) cost a spill and 1 %
#endif
__global__ void __launch_bounds__(MD_GVV_BT, MD_GVV_CPS)
k_gather_vv(int64_t n, int K, const Rec* Q, const unsigned long long* MASK, int dense,   // Q, MASK, f: no __restrict__/.nc --
            double* f, double* __restrict__ x, double* __restrict__ y, double* __restrict__ z,   // the pair kernel
            double* __restrict__ vx, double* __restrict__ vy, double* __restrict__ vz,           // before wrote them
            double hk, double dt, double Lx, double Ly, double Lz) {
    const int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t i = i0 < n ? i0 : n - 1;
    // launched as a programmatic dependent of the pair kernel (common.cuh, md_launch_pdl): the velocity and
    // position of the atom, which the pair kernel does not write, are requested while that kernel drains
    double ux = vx[i], uy = vy[i], uz = vz[i];
    double px = 0, py = 0, pz = 0;
    if (MODE == 2) { px = x[i]; py = y[i]; pz = z[i]; }
    md_grid_wait();
    md_grid_release();
    if (i0 >= n) return;
    // The first four record slots are requested before MASK has arrived (their addresses depend on i only): one
    // dependent load level less.  A slot the mask does not select is loaded and dropped (it lies inside Q).
    T Fx = T(0), Fy = T(0), Fz = T(0);
    T hx[4], hy[4], hz[4];
#pragma unroll
    for (int sl = 0; sl < 4; ++sl) rm::load_rec_once(&Q[(int64_t)(sl < K ? sl : 0) * n + i], &hx[sl], &hy[sl], &hz[sl]);
    unsigned long long mask = rm::load_once(&MASK[i]);
    const double ox = rm::load_once(&f[i]), oy = rm::load_once(&f[n + i]), oz = rm::load_once(&f[2 * n + i]);   // own halves sum_j P_ij
    if (dense) {                                             // popc(mask) consecutive slots
        const int cnt = __popcll(mask);
#pragma unroll
        for (int sl = 0; sl < 4; ++sl)
            if (sl < cnt) { Fx += hx[sl]; Fy += hy[sl]; Fz += hz[sl]; }
        for (int s0 = 4; s0 < cnt; s0 += 4) {                // the rest four at a time: loads first, sums in slot order
#pragma unroll
            for (int u = 0; u < 4; ++u)
                rm::load_rec_once(&Q[(int64_t)(s0 + u < cnt ? s0 + u : s0) * n + i], &hx[u], &hy[u], &hz[u]);
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (s0 + u < cnt) { Fx += hx[u]; Fy += hy[u]; Fz += hz[u]; }
        }
    } else {                                                 // slot = list position
#pragma unroll
        for (int sl = 0; sl < 4; ++sl)
            if (mask >> sl & 1ull) { Fx += hx[sl]; Fy += hy[sl]; Fz += hz[sl]; }
        mask &= ~15ull;
        while (mask) {
            const int m = __ffsll((long long)mask) - 1;
            mask &= mask - 1;
            T qx, qy, qz;
            rm::load_rec_once(&Q[(int64_t)m * n + i], &qx, &qy, &qz);
            Fx += qx; Fy += qy; Fz += qz;
        }
    }
    const double fx = ox - (double)Fx, fy = oy - (double)Fy, fz = oz - (double)Fz;
    ux = __fma_rn(hk, fx, ux); uy = __fma_rn(hk, fy, uy); uz = __fma_rn(hk, fz, uz);     // kick of this step
    if (MODE == 1) { f[i] = fx; f[n + i] = fy; f[2 * n + i] = fz; }
    if (MODE == 2) {
        ux = __fma_rn(hk, fx, ux); uy = __fma_rn(hk, fy, uy); uz = __fma_rn(hk, fz, uz); // kick of the next
        x[i] = md_wrap(__fma_rn(dt, ux, px), Lx);
        y[i] = md_wrap(__fma_rn(dt, uy, py), Ly);
        z[i] = md_wrap(__fma_rn(dt, uz, pz), Lz);
    }
    vx[i] = ux; vy[i] = uy; vz[i] = uz;
}

}  // namespace

int md_launch_gather(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                     const double* vx, const double* vy, const double* vz, const double box[3],
                     int precision, double* f, double* virial, double* heat, const VVFuse* vv, cudaStream_t s) {
    if (nl->virial_own_only) virial = nullptr;               // see common.cuh: only the total virial is wanted
    if (n == 0 || (!f && !virial && !heat)) return MD_OK;
    ProfScope prof(nl, MD_KIND_GATHER, 1, s);
    if (vv) {
        if (!f || virial || heat) return MD_ERR_ARG;
#define MD_GATHER_VV(TT, RR, MODE)                                                                        \
    MD_CUDA_TRY(md_launch_pdl(k_gather_vv<TT, RR, MODE>, dim3((unsigned)((n + MD_GVV_BT - 1) / MD_GVV_BT)), dim3(MD_GVV_BT), 0, s, nl->gather_pdl != 0, n, nl->K, (const RR*)nl->Q,            \
                              nl->MASK, nl->q_dense, f, vv->x, vv->y, vv->z, vv->vx, vv->vy, vv->vz, vv->hk, vv->dt,    \
                              box[0], box[1], box[2]))
        if (precision == MD_FP32) { if (vv->mode == 2) MD_GATHER_VV(float, float4, 2); else MD_GATHER_VV(float, float4, 1); }
        else { if (vv->mode == 2) MD_GATHER_VV(double, PairRec64, 2); else MD_GATHER_VV(double, PairRec64, 1); }
#undef MD_GATHER_VV
        MD_CUDA_TRY(cudaGetLastError());
        return MD_OK;
    }
    const unsigned gg = (unsigned)((n + 127) / 128);
    const bool geom = virial != nullptr || heat != nullptr;
#define MD_GATHER(TT, RR, GEOM)                                                                                   \
    MD_CUDA_TRY(md_launch_pdl(k_gather<TT, RR, GEOM>, dim3(gg), dim3(128), 0, s, nl->gather_pdl != 0, n, nl->K, x, y, z, vx, vy, vz,       \
                              box[0], box[1], box[2], (const int32_t*)nl->NL, (const RR*)nl->Q,                   \
                              (const unsigned long long*)nl->MASK, nl->q_dense, f, virial, heat))
    if (precision == MD_FP32) { if (geom) MD_GATHER(float, float4, true); else MD_GATHER(float, float4, false); }
    else { if (geom) MD_GATHER(double, PairRec64, true); else MD_GATHER(double, PairRec64, false); }
#undef MD_GATHER
    MD_CUDA_TRY(cudaGetLastError());
    return MD_OK;
}
