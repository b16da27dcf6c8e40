// api.cu -- the C ABI declared in include/md.h: argument checks, handle life cycle, and the host-side
// composition of the kernels.  No arithmetic of the method lives here.
#include <algorithm>
#include <cmath>
#include <mutex>
#include <new>
#include <set>
#include <utility>

#include "common.cuh"

namespace {

bool valid_box(const double box[3]) { return box && box[0] > 0 && box[1] > 0 && box[2] > 0; }

void free_all(md_neighbors* nl) {
    cudaFree(nl->NN); cudaFree(nl->NL); cudaFree(nl->REV); cudaFree(nl->HEAD); cudaFree(nl->Q); cudaFree(nl->MASK); cudaFree(nl->bin_list); cudaFree(nl->bin_count);
    cudaFree(nl->cell_count); cudaFree(nl->cell_of); cudaFree(nl->rank_in_cell); cudaFree(nl->sorted); cudaFree(nl->sortedf);
    cudaFree(nl->scan_blocks); cudaFree(nl->d_status); cudaFree(nl->e2e); cudaFree(nl->npt_w); cudaFree(nl->npt_part);
    if (nl->h_npt) cudaFreeHost(nl->h_npt);
    if (nl->npt_event) cudaEventDestroy(nl->npt_event);
    if (nl->h_maxrow) cudaFreeHost(nl->h_maxrow);
    if (nl->ev_list) cudaEventDestroy(nl->ev_list);
    if (nl->ev_fork) cudaEventDestroy(nl->ev_fork);
    if (nl->ev_join) cudaEventDestroy(nl->ev_join);
    if (nl->s_copy) cudaStreamDestroy(nl->s_copy);
    if (nl->ev_pool) for (cudaEvent_t e : *nl->ev_pool) cudaEventDestroy(e);
    delete nl->ev_pool; delete nl->ev_kind;
}

int force_dispatch(md_neighbors* nl, int potential, const void* params, int precision, int64_t n,
                   const double* x, const double* y, const double* z, const double* vx, const double* vy,
                   const double* vz, const double box[3], double* pe, double* f, double* virial,
                   double* heat, const VVFuse* vv, cudaStream_t s) {
    if (potential == MD_TERSOFF)
        return md_launch_tersoff(nl, n, x, y, z, vx, vy, vz, box, (const md_tersoff_params*)params, precision,
                                 pe, f, virial, heat, vv, s);
    return md_launch_sw(nl, n, x, y, z, vx, vy, vz, box, (const md_sw_params*)params, precision, pe, f,
                        virial, heat, vv, s);
}

int check_force_args(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                     const double* vx, const double* vy, const double* vz, const double box[3],
                     const void* p, int precision, const double* heat) {
    if (!nl || n < 0 || !valid_box(box) || !p) return MD_ERR_ARG;
    if (precision != MD_FP64 && precision != MD_FP32) return MD_ERR_ARG;
    if (n > 0 && (!x || !y || !z)) return MD_ERR_ARG;
    if (heat && n > 0 && (!vx || !vy || !vz)) return MD_ERR_ARG;
    if (nl->n != n) return MD_ERR_NO_LIST;
    return MD_OK;
}

}  // namespace

// Kernels that need more than 48 KB of dynamic shared memory must opt in per device (the attribute belongs
// to the function on the current device, not to the process).
int md_allow_dynamic_smem(const void* kernel, int bytes) {
    static std::mutex mu;
    static std::set<std::pair<int, const void*>> done;
    int dev = 0;
    MD_CUDA_TRY(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lock(mu);
    if (done.count({dev, kernel})) return MD_OK;
    MD_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    done.insert({dev, kernel});
    return MD_OK;
}

// ---- per-kind launch counting and event timing --------------------------------------------------
ProfScope::ProfScope(md_neighbors* nl_, int kind, int nk, cudaStream_t s_) : nl(nl_), s(s_), e1(nullptr), on(false) {
    if (!nl) return;
    nl->launches[kind] += nk;
    if (!nl->prof_on || !nl->ev_pool) return;
    while (nl->ev_pool->size() < nl->ev_used + 2) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) return;
        nl->ev_pool->push_back(e);
    }
    cudaEvent_t e0 = (*nl->ev_pool)[nl->ev_used];
    e1 = (*nl->ev_pool)[nl->ev_used + 1];
    nl->ev_used += 2;
    nl->ev_kind->push_back(kind);
    cudaEventRecord(e0, s);
    on = true;
}
ProfScope::~ProfScope() { if (on) cudaEventRecord(e1, s); }

int md_list_row_stats(md_neighbors* nl, int* max_row, int* long_rows, int wait) {
    if (nl->maxrow_pending) {
        // the statistics only steer the choice between two kernels that are both correct for any list, so a
        // force call takes whatever has arrived (no host stall, no idle GPU after a rebuild); only the very
        // first call, or an explicit md_neighbors_row_stats, waits for the copy
        cudaError_t q = (wait || !nl->row_stats_valid) ? cudaEventSynchronize(nl->ev_list) : cudaEventQuery(nl->ev_list);
        if (q == cudaSuccess) {
            nl->row_stats[0] = nl->h_maxrow[0]; nl->row_stats[1] = nl->h_maxrow[1];
            nl->row_stats_valid = 1;
            nl->maxrow_pending = 0;
        } else if (q != cudaErrorNotReady) {
            return MD_ERR_CUDA;
        }
    }
    *max_row = nl->row_stats[0];
    *long_rows = nl->row_stats[1];
    return MD_OK;
}

extern "C" {

int md_profile_enable(md_neighbors* nl, int enable) {
    if (!nl) return MD_ERR_ARG;
    if (enable && !nl->ev_pool) {
        nl->ev_pool = new (std::nothrow) std::vector<cudaEvent_t>();
        nl->ev_kind = new (std::nothrow) std::vector<int>();
        if (!nl->ev_pool || !nl->ev_kind) return MD_ERR_ALLOC;
    }
    nl->prof_on = enable ? 1 : 0;
    return MD_OK;
}

int md_profile_read(md_neighbors* nl, double* ms, int64_t* launches) {
    if (!nl) return MD_ERR_ARG;
    MD_CUDA_TRY(cudaDeviceSynchronize());
    for (int k = 0; k < MD_N_KINDS; ++k) nl->ms_acc[k] = 0.0;
    if (nl->ev_pool && nl->ev_kind) {
        for (size_t q = 0; q < nl->ev_kind->size(); ++q) {
            float t = 0.f;
            if (cudaEventElapsedTime(&t, (*nl->ev_pool)[2 * q], (*nl->ev_pool)[2 * q + 1]) == cudaSuccess)
                nl->ms_acc[(*nl->ev_kind)[q]] += (double)t;
        }
        nl->ev_kind->clear();
        nl->ev_used = 0;
    }
    for (int k = 0; k < MD_N_KINDS; ++k) {
        if (ms) ms[k] = nl->ms_acc[k];
        if (launches) launches[k] = nl->launches[k];
        nl->launches[k] = 0;
    }
    return MD_OK;
}

const char* md_version(void) { return "paper_1610_03343_b200 0.1 (sm_100a)"; }

int md_neighbors_create(md_neighbors** out, int64_t n_atoms, int max_neighbors) {
    if (!out || n_atoms < 0 || max_neighbors < 1 || max_neighbors > MD_MAX_NEIGHBORS) return MD_ERR_ARG;
    if (n_atoms * (int64_t)max_neighbors > (int64_t)2000000000) return MD_ERR_ARG;   // int32 pair indices
    md_neighbors* nl = new (std::nothrow) md_neighbors();
    if (!nl) return MD_ERR_ALLOC;
    *nl = md_neighbors{};
    nl->n_cap = n_atoms; nl->K = max_neighbors;
    const size_t n = (size_t)(n_atoms > 0 ? n_atoms : 1), K = (size_t)max_neighbors;
    bool ok = true;
    ok = ok && cudaMalloc(&nl->NN, n * sizeof(int32_t)) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->NL, n * K * sizeof(int32_t)) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->REV, n * K) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->HEAD, n * sizeof(MdRowHead)) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->Q, n * K * sizeof(PairRec64)) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->MASK, n * sizeof(unsigned long long)) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->bin_list, 3 * n * sizeof(int32_t)) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->bin_count, 8 * sizeof(int32_t)) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->cell_of, n * sizeof(int32_t)) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->rank_in_cell, n * sizeof(int32_t)) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->sorted, n * sizeof(double4)) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->sortedf, n * sizeof(float4)) == cudaSuccess;
    ok = ok && cudaMalloc(&nl->d_status, 3 * sizeof(int)) == cudaSuccess;
    ok = ok && cudaMallocHost(&nl->h_maxrow, 2 * sizeof(int)) == cudaSuccess;
    ok = ok && cudaEventCreateWithFlags(&nl->ev_list, cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { cudaGetLastError(); free_all(nl); delete nl; return MD_ERR_ALLOC; }
    cudaMemset(nl->d_status, 0, 3 * sizeof(int));
    cudaMemset(nl->bin_count, 0, 8 * sizeof(int32_t));
    *out = nl;
    return MD_OK;
}

int md_neighbors_destroy(md_neighbors* nl) {
    if (!nl) return MD_ERR_ARG;
    cudaDeviceSynchronize();
    free_all(nl);
    delete nl;
    return MD_OK;
}

int md_neighbors_status(md_neighbors* nl, int* max_count_seen, void* stream) {
    if (!nl) return MD_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    int h[2] = {0, 0};
    MD_CUDA_TRY(cudaMemcpyAsync(h, nl->d_status, sizeof(h), cudaMemcpyDeviceToHost, s));
    MD_CUDA_TRY(cudaStreamSynchronize(s));
    MD_CUDA_TRY(cudaMemsetAsync(nl->d_status, 0, sizeof(int), s));
    if (max_count_seen) *max_count_seen = h[1];
    if (h[0] & (MD_DEV_ROW_OVERFLOW | MD_DEV_INRANGE_OVERFLOW)) return MD_ERR_NEIGHBOR_OVERFLOW;
    if (h[0] & MD_DEV_NO_REVERSE) return MD_ERR_LIST_ASYMMETRIC;
    return MD_OK;
}

int md_neighbors_row_stats(md_neighbors* nl, int* max_row, int* rows_longer_than_4) {
    if (!nl) return MD_ERR_ARG;
    if (nl->n == 0) return MD_ERR_NO_LIST;
    int a = 0, b = 0;
    const int rc = md_list_row_stats(nl, &a, &b, 1);
    if (rc != MD_OK) return rc;
    if (max_row) *max_row = a;
    if (rows_longer_than_4) *rows_longer_than_4 = b;
    return MD_OK;
}

int md_neighbors_export(md_neighbors* nl, int32_t* NN, int32_t* NL, void* stream) {
    if (!nl || !NN || !NL) return MD_ERR_ARG;
    if (nl->n == 0) return MD_OK;
    cudaStream_t s = (cudaStream_t)stream;
    MD_CUDA_TRY(cudaMemcpyAsync(NN, nl->NN, sizeof(int32_t) * nl->n, cudaMemcpyDeviceToDevice, s));
    MD_CUDA_TRY(cudaMemcpyAsync(NL, nl->NL, sizeof(int32_t) * nl->n * nl->K, cudaMemcpyDeviceToDevice, s));
    return MD_OK;
}

int md_neighbors_import(md_neighbors* nl, int64_t n, const int32_t* NN, const int32_t* NL, void* stream) {
    if (!nl || n < 0 || n > nl->n_cap || (n > 0 && (!NN || !NL))) return MD_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    nl->n = n;
    if (n == 0) return MD_OK;
    MD_CUDA_TRY(cudaMemsetAsync(nl->d_status + 1, 0, 2 * sizeof(int), s));
    MD_CUDA_TRY(cudaMemcpyAsync(nl->NN, NN, sizeof(int32_t) * n, cudaMemcpyDeviceToDevice, s));
    MD_CUDA_TRY(cudaMemcpyAsync(nl->NL, NL, sizeof(int32_t) * n * nl->K, cudaMemcpyDeviceToDevice, s));
    return md_launch_reverse(nl, s, 1);
}

int md_build_neighbors(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                       const double box[3], double r_list, void* stream) {
    if (!nl || n < 0 || n > nl->n_cap || !valid_box(box) || !(r_list > 0)) return MD_ERR_ARG;
    if (n > 0 && (!x || !y || !z)) return MD_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    MD_CUDA_TRY(cudaMemsetAsync(nl->d_status + 1, 0, 2 * sizeof(int), s));
    return md_launch_build(nl, n, x, y, z, box, r_list, s);
}

int md_tersoff_force(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                     const double* vx, const double* vy, const double* vz, const double box[3],
                     const md_tersoff_params* p, int precision,
                     double* pe, double* f, double* virial, double* heat, void* stream) {
    int rc = check_force_args(nl, n, x, y, z, vx, vy, vz, box, p, precision, heat);
    if (rc != MD_OK) return rc;
    if (!(p->S > p->R) || !(p->R > 0) || !(p->n > 0) || !(p->d != 0)) return MD_ERR_ARG;
    return md_launch_tersoff(nl, n, x, y, z, vx, vy, vz, box, p, precision, pe, f, virial, heat, nullptr,
                             (cudaStream_t)stream);
}

int md_tersoff_force_literal(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                             const double* vx, const double* vy, const double* vz, const double box[3],
                             const md_tersoff_params* p, int precision,
                             double* pe, double* f, double* virial, double* heat, void* stream) {
    int rc = check_force_args(nl, n, x, y, z, vx, vy, vz, box, p, precision, heat);
    if (rc != MD_OK) return rc;
    if (!(p->S > p->R) || !(p->R > 0) || !(p->n > 0) || !(p->d != 0)) return MD_ERR_ARG;
    return md_launch_tersoff_literal(nl, n, x, y, z, vx, vy, vz, box, p, precision, pe, f, virial, heat,
                                     (cudaStream_t)stream);
}

int md_tersoff_multi_force(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                           const double* vx, const double* vy, const double* vz, const double box[3],
                           const int32_t* types, const md_tersoff_multi_params* p, int precision,
                           double* pe, double* f, double* virial, double* heat, void* stream) {
    int rc = check_force_args(nl, n, x, y, z, vx, vy, vz, box, p, precision, heat);
    if (rc != MD_OK) return rc;
    if (p->ntypes < 1 || p->ntypes > MD_MAX_TYPES || n >= ((int64_t)1 << 28)) return MD_ERR_ARG;
    if (p->ntypes > 1 && n > 0 && !types) return MD_ERR_ARG;
    for (int t = 0; t < p->ntypes; ++t) {
        const md_tersoff_params& e = p->elem[t];
        if (!(e.S > e.R) || !(e.R > 0) || !(e.n > 0) || !(e.d != 0)) return MD_ERR_ARG;
    }
    return md_launch_tersoff_multi(nl, n, x, y, z, vx, vy, vz, box, types, p, precision, pe, f, virial, heat,
                                   (cudaStream_t)stream);
}

int md_sw_force(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                const double* vx, const double* vy, const double* vz, const double box[3],
                const md_sw_params* p, int precision,
                double* pe, double* f, double* virial, double* heat, void* stream) {
    int rc = check_force_args(nl, n, x, y, z, vx, vy, vz, box, p, precision, heat);
    if (rc != MD_OK) return rc;
    if (!(p->sigma > 0) || !(p->a > 0)) return MD_ERR_ARG;
    return md_launch_sw(nl, n, x, y, z, vx, vy, vz, box, p, precision, pe, f, virial, heat, nullptr,
                        (cudaStream_t)stream);
}

int md_velocity_verlet_step(int phase, int64_t n, double* x, double* y, double* z,
                            double* vx, double* vy, double* vz, const double* f,
                            double mass_amu, double dt_fs, const double box[3], void* stream) {
    if ((phase != 0 && phase != 1) || n < 0 || !(mass_amu > 0)) return MD_ERR_ARG;
    if (n > 0 && (!vx || !vy || !vz || !f)) return MD_ERR_ARG;
    if (phase == 0 && (!valid_box(box) || (n > 0 && (!x || !y || !z)))) return MD_ERR_ARG;
    return md_launch_vv(nullptr, phase, n, x, y, z, vx, vy, vz, f, mass_amu, dt_fs, box, (cudaStream_t)stream);
}

// v_ready (may be null): an event the stream waits for before the first kernel that reads the velocities
static int nve_run_impl(md_neighbors* nl, int potential, const void* params, int precision, int64_t n,
               double* x, double* y, double* z, double* vx, double* vy, double* vz,
               double* f, int f_valid, double* pe, const double box[3], double mass_amu, double dt_fs,
               int first_step, int nsteps, int rebuild_every, double r_list, void* stream, cudaEvent_t v_ready) {
    if (!nl || !params || n < 0 || n > nl->n_cap || !valid_box(box) || nsteps < 0 || rebuild_every < 1 ||
        first_step < 0)
        return MD_ERR_ARG;
    if (potential != MD_TERSOFF && potential != MD_SW) return MD_ERR_ARG;
    if (precision != MD_FP64 && precision != MD_FP32) return MD_ERR_ARG;
    if (!(mass_amu > 0) || !(r_list > 0)) return MD_ERR_ARG;
    if (n > 0 && (!x || !y || !z || !vx || !vy || !vz || !f)) return MD_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    int rc;
    // argument errors have no side effects: everything that can be refused is refused before the first launch
    for (int a = 0; a < 3; ++a)
        if ((int)(box[a] / r_list) < 3) return MD_ERR_BOX_TOO_SMALL;
    const bool first_step_rebuilds = first_step % rebuild_every == 0;
    if (f_valid && nsteps > 0 && !first_step_rebuilds && nl->n != n) return MD_ERR_NO_LIST;
    if (!f_valid) {
        if ((rc = md_build_neighbors(nl, n, x, y, z, box, r_list, stream)) != MD_OK) return rc;
        if ((rc = force_dispatch(nl, potential, params, precision, n, x, y, z, nullptr, nullptr, nullptr, box,
                                 pe, f, nullptr, nullptr, nullptr, s)) != MD_OK) return rc;
    }
    if (v_ready) MD_CUDA_TRY(cudaStreamWaitEvent(s, v_ready, 0));
    if (nsteps == 0) return MD_OK;
    // Step s = kick+drift, [rebuild], force, kick.  The kick that ends step s and the kick+drift that
    // starts step s+1 are fused into the gather kernel of step s (gather.cu, k_gather_vv): per step the
    // loop launches the pair kernel and one fused kernel, plus the list build on rebuild steps.
    VVFuse vv;
    vv.hk = 0.5 * dt_fs * MD_KAPPA / mass_amu; vv.dt = dt_fs;
    vv.x = x; vv.y = y; vv.z = z; vv.vx = vx; vv.vy = vy; vv.vz = vz;
    if ((rc = md_launch_vv(nl, 0, n, x, y, z, vx, vy, vz, f, mass_amu, dt_fs, box, s)) != MD_OK) return rc;
    for (int step = first_step; step < first_step + nsteps; ++step) {
        if (step % rebuild_every == 0)
            if ((rc = md_build_neighbors(nl, n, x, y, z, box, r_list, stream)) != MD_OK) return rc;
        if (nl->n != n) return MD_ERR_NO_LIST;
        const bool last = step == first_step + nsteps - 1;
        vv.mode = last ? 1 : 2;
        vv.pdl_pair = step % rebuild_every != 0;             // the list is the one the kernel before already used
        if ((rc = force_dispatch(nl, potential, params, precision, n, x, y, z, nullptr, nullptr, nullptr, box,
                                 last ? pe : nullptr, f, nullptr, nullptr, &vv, s)) != MD_OK) return rc;
    }
    return MD_OK;
}

int md_nve_run(md_neighbors* nl, int potential, const void* params, int precision, int64_t n,
               double* x, double* y, double* z, double* vx, double* vy, double* vz,
               double* f, int f_valid, double* pe, const double box[3], double mass_amu, double dt_fs,
               int first_step, int nsteps, int rebuild_every, double r_list, void* stream) {
    return nve_run_impl(nl, potential, params, precision, n, x, y, z, vx, vy, vz, f, f_valid, pe, box, mass_amu, dt_fs,
                        first_step, nsteps, rebuild_every, r_list, stream, nullptr);
}

int md_npt_run(md_neighbors* nl, int potential, const void* params, int precision, int64_t n,
               double* x, double* y, double* z, double* vx, double* vy, double* vz,
               double* f, int f_valid, double box[3], double mass_amu, double dt_fs,
               int first_step, int nsteps, int rebuild_every, double r_list,
               const md_berendsen_params* b, double* T_trace, double* P_trace, void* stream) {
    if (!nl || !params || !b || n < 1 || n > nl->n_cap || !valid_box(box) || nsteps < 0 || rebuild_every < 1 ||
        first_step < 0)
        return MD_ERR_ARG;
    if (potential != MD_TERSOFF && potential != MD_SW) return MD_ERR_ARG;
    if (precision != MD_FP64 && precision != MD_FP32) return MD_ERR_ARG;
    if (!(mass_amu > 0) || !(r_list > 0) || !(b->tau_T > 0) || !(b->tau_P > 0)) return MD_ERR_ARG;
    if (!x || !y || !z || !vx || !vy || !vz || !f) return MD_ERR_ARG;
    for (int a = 0; a < 3; ++a)
        if ((int)(box[a] / r_list) < 3) return MD_ERR_BOX_TOO_SMALL;
    if (f_valid && nsteps > 0 && first_step % rebuild_every != 0 && nl->n != n) return MD_ERR_NO_LIST;
    cudaStream_t s = (cudaStream_t)stream;
    if (nl->npt_cap < n || !nl->npt_w) {
        MD_CUDA_TRY(cudaStreamSynchronize(s));
        cudaFree(nl->npt_w); nl->npt_w = nullptr; nl->npt_cap = 0;
        if (cudaMalloc(&nl->npt_w, sizeof(double) * 9 * (size_t)n) != cudaSuccess) { cudaGetLastError(); return MD_ERR_ALLOC; }
        nl->npt_cap = n;
    }
    if (!nl->npt_part) {
        if (cudaMalloc(&nl->npt_part, sizeof(double) * md_npt_scratch_doubles()) != cudaSuccess ||
            cudaMallocHost(&nl->h_npt, 8 * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return MD_ERR_ALLOC; }
    }
    int rc;
    double* W = nl->npt_w;
    // The barostat needs the TOTAL virial only.  Summed over the atoms, Eq. (29) regroups into
    //   sum_i W_i = -1/2 sum_ij r_ij (x) (P_ij - P_ji) = - sum_ij r_ij (x) P_ij = 2 sum_i W_i^own,
    // W_i^own = -1/2 sum_j r_ij (x) P_ij being what the pair kernel leaves in `virial` (r_ji = -r_ij, i <-> j in the
    // second term).  So the gather runs forces-only here (160 instead of 512 bytes per atom, no list or neighbour
    // coordinates) and per-atom W_i is never formed; md_tersoff_force / md_sw_force still deliver it.
    struct OwnOnly { md_neighbors* h; OwnOnly(md_neighbors* q) : h(q) { h->virial_own_only = 1; } ~OwnOnly() { h->virial_own_only = 0; } } own_only(nl);
    if (!f_valid) {
        if ((rc = md_build_neighbors(nl, n, x, y, z, box, r_list, stream)) != MD_OK) return rc;
        if ((rc = force_dispatch(nl, potential, params, precision, n, x, y, z, nullptr, nullptr, nullptr, box,
                                 nullptr, f, W, nullptr, nullptr, s)) != MD_OK) return rc;
    }
    // Per step: kick+drift (with the scaling the step before decided applied first, in the same pass), [rebuild],
    // force with the own-half W, then ONE pass that does the second half-kick and the two sums; a one-thread
    // kernel forms T, P, lambda, mu and the scaled box on the device, and the next step's kick+drift -- which reads
    // them from there -- is enqueued before the host waits for the copy of that record (its box for the next build and
    // pair kernel, the two trace values): the round trip to the host overlaps with that pass.
    const double hk = 0.5 * dt_fs * MD_KAPPA / mass_amu;
    double lam_p = 1.0, mu_p = 1.0;
    bool drift_enqueued = false;
    const int last = first_step + nsteps - 1;
    for (int step = first_step; step <= last; ++step) {
        if (!drift_enqueued &&
            (rc = md_launch_vv(nl, 0, n, x, y, z, vx, vy, vz, f, mass_amu, dt_fs, box, s, lam_p, mu_p)) != MD_OK) return rc;
        drift_enqueued = false;
        if (step % rebuild_every == 0)
            if ((rc = md_build_neighbors(nl, n, x, y, z, box, r_list, stream)) != MD_OK) return rc;
        if (nl->n != n) return MD_ERR_NO_LIST;
        if ((rc = force_dispatch(nl, potential, params, precision, n, x, y, z, nullptr, nullptr, nullptr, box,
                                 nullptr, f, W, nullptr, nullptr, s)) != MD_OK) return rc;
        if ((rc = md_launch_npt_sums(nl, n, vx, vy, vz, W, f, hk, mass_amu, dt_fs, box, b, s)) != MD_OK) return rc;
        if (step < last) {
            if ((rc = md_launch_vv_dev(nl, n, x, y, z, vx, vy, vz, f, mass_amu, dt_fs, md_npt_scal(nl), s)) != MD_OK) return rc;
            drift_enqueued = true;
        }
        double rec[7];
        if ((rc = md_npt_sums_wait(nl, rec)) != MD_OK) return rc;
        const double ke2 = rec[0] * mass_amu / MD_KAPPA;                  // 2 KE
        const double V = box[0] * box[1] * box[2];
        const double T = ke2 / (3.0 * (double)n * MD_KB), P = (ke2 + 2.0 * rec[1]) / (3.0 * V);   // tr sum W = 2 tr sum W^own
        if (T_trace) T_trace[step - first_step] = T;
        if (P_trace) P_trace[step - first_step] = P;
        lam_p = rec[2]; mu_p = rec[3];
        for (int a = 0; a < 3; ++a) box[a] = rec[4 + a];
    }
    if (nsteps > 0 && (rc = md_launch_npt_scale(nl, n, x, y, z, vx, vy, vz, lam_p, mu_p, s)) != MD_OK) return rc;
    return MD_OK;
}

int md_nve_heat_run(md_neighbors* nl, int potential, const void* params, int precision, int64_t n,
                    double* x, double* y, double* z, double* vx, double* vy, double* vz,
                    double* f, int f_valid, const double box[3], double mass_amu, double dt_fs,
                    int first_step, int nsteps, int rebuild_every, double r_list, int sample_every,
                    double* J_pot, double* J_kin, void* stream) {
    if (!nl || !params || n < 1 || n > nl->n_cap || !valid_box(box) || nsteps < 0 || rebuild_every < 1 ||
        first_step < 0 || sample_every < 1)
        return MD_ERR_ARG;
    if (potential != MD_TERSOFF && potential != MD_SW) return MD_ERR_ARG;
    if (precision != MD_FP64 && precision != MD_FP32) return MD_ERR_ARG;
    if (!(mass_amu > 0) || !(r_list > 0)) return MD_ERR_ARG;
    if (!x || !y || !z || !vx || !vy || !vz || !f) return MD_ERR_ARG;
    for (int a = 0; a < 3; ++a)
        if ((int)(box[a] / r_list) < 3) return MD_ERR_BOX_TOO_SMALL;
    if (f_valid && nsteps > 0 && first_step % rebuild_every != 0 && nl->n != n) return MD_ERR_NO_LIST;
    cudaStream_t s = (cudaStream_t)stream;
    // scratch: per-atom heat current [3][n] and energy [n] live in the NPT virial buffer ([9][n])
    if (nl->npt_cap < n || !nl->npt_w) {
        MD_CUDA_TRY(cudaStreamSynchronize(s));
        cudaFree(nl->npt_w); nl->npt_w = nullptr; nl->npt_cap = 0;
        if (cudaMalloc(&nl->npt_w, sizeof(double) * 9 * (size_t)n) != cudaSuccess) { cudaGetLastError(); return MD_ERR_ALLOC; }
        nl->npt_cap = n;
    }
    if (!nl->npt_part) {
        if (cudaMalloc(&nl->npt_part, sizeof(double) * md_npt_scratch_doubles()) != cudaSuccess ||
            cudaMallocHost(&nl->h_npt, 8 * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return MD_ERR_ALLOC; }
    }
    double* J = nl->npt_w;
    double* pe = nl->npt_w + 3 * n;
    // The steps between two samples run as one fused md_nve_run segment (pair kernel + fused gather per step,
    // chained as programmatic dependents); its last step leaves the forces, U_i and -- still valid -- the pair
    // records of the sampled state, so a sample costs one more gather (Eq. 30 with that state's velocities) and
    // the reduction.  The trajectory is bit-identical to the unfused composition (tests/test_gpu_parity.py).
    int rc, ns = 0, done = 0, fv = f_valid;
    while (done < nsteps) {
        const int seg = std::min(sample_every - done % sample_every, nsteps - done);
        if ((rc = nve_run_impl(nl, potential, params, precision, n, x, y, z, vx, vy, vz, f, fv, pe, box, mass_amu, dt_fs,
                               first_step + done, seg, rebuild_every, r_list, stream, nullptr)) != MD_OK) return rc;
        done += seg; fv = 1;
        if (done % sample_every != 0) break;                  // a trailing partial segment: no sample
        nl->gather_pdl = 0;                                   // the kernel before (the last kick) wrote the velocities it reads
        if ((rc = md_launch_gather(nl, n, x, y, z, vx, vy, vz, box, precision, nullptr, nullptr, J, nullptr, s)) != MD_OK)
            return rc;
        double out[6];
        if ((rc = md_launch_heat_sums(nl, n, vx, vy, vz, pe, J, mass_amu, out, s)) != MD_OK) return rc;
        for (int a = 0; a < 3; ++a) {
            if (J_pot) J_pot[3 * ns + a] = out[a];
            if (J_kin) J_kin[3 * ns + a] = out[3 + a];
        }
        ++ns;
    }
    return MD_OK;
}

int md_nve_run_host(md_neighbors* nl, int potential, const void* params, int precision, int64_t n,
                    double* x, double* y, double* z, double* vx, double* vy, double* vz,
                    double* f, double* pe, const double box[3], double mass_amu, double dt_fs,
                    int nsteps, int rebuild_every, double r_list, void* stream) {
    if (!nl || n < 0 || n > nl->n_cap) return MD_ERR_ARG;
    if (n > 0 && (!x || !y || !z || !vx || !vy || !vz)) return MD_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    if (nl->e2e_cap < n || !nl->e2e) {
        MD_CUDA_TRY(cudaStreamSynchronize(s));
        if (nl->e2e) cudaFree(nl->e2e);
        nl->e2e = nullptr; nl->e2e_cap = 0;
        if (cudaMalloc(&nl->e2e, sizeof(double) * 10 * (size_t)(n > 0 ? n : 1)) != cudaSuccess) {
            cudaGetLastError();
            return MD_ERR_ALLOC;
        }
        nl->e2e_cap = n;
    }
    double* d = nl->e2e;
    double* host_in[6] = {x, y, z, vx, vy, vz};
    const size_t bytes = sizeof(double) * (size_t)n;
    if (!nl->s_copy) {
        if (cudaStreamCreateWithFlags(&nl->s_copy, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&nl->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&nl->ev_join, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return MD_ERR_ALLOC; }
    }
    // positions on the caller's stream; velocities on the copy stream (after whatever `s` still does with the
    // buffers), joined just before the first kick: list build and first force evaluation overlap with them
    MD_CUDA_TRY(cudaEventRecord(nl->ev_fork, s));
    MD_CUDA_TRY(cudaStreamWaitEvent(nl->s_copy, nl->ev_fork, 0));
    for (int a = 0; a < 3; ++a)
        MD_CUDA_TRY(cudaMemcpyAsync(d + a * n, host_in[a], bytes, cudaMemcpyHostToDevice, s));
    for (int a = 3; a < 6; ++a)
        MD_CUDA_TRY(cudaMemcpyAsync(d + a * n, host_in[a], bytes, cudaMemcpyHostToDevice, nl->s_copy));
    MD_CUDA_TRY(cudaEventRecord(nl->ev_join, nl->s_copy));
    int rc = nve_run_impl(nl, potential, params, precision, n, d, d + n, d + 2 * n, d + 3 * n, d + 4 * n, d + 5 * n,
                          d + 6 * n, 0, d + 9 * n, box, mass_amu, dt_fs, 0, nsteps, rebuild_every, r_list, stream,
                          nl->ev_join);
    if (rc != MD_OK) return rc;
    for (int a = 0; a < 6; ++a)
        MD_CUDA_TRY(cudaMemcpyAsync(host_in[a], d + a * n, bytes, cudaMemcpyDeviceToHost, s));
    if (f) MD_CUDA_TRY(cudaMemcpyAsync(f, d + 6 * n, 3 * bytes, cudaMemcpyDeviceToHost, s));
    if (pe) MD_CUDA_TRY(cudaMemcpyAsync(pe, d + 9 * n, bytes, cudaMemcpyDeviceToHost, s));
    // this call synchronises anyway, so it reports what the device latched (row or in-range overflow)
    return md_neighbors_status(nl, nullptr, stream);
}

int md_pair_counts(md_neighbors* nl, int64_t out[3], void* stream) {
    if (!nl || !out) return MD_ERR_ARG;
    if (nl->n == 0) { out[0] = out[1] = out[2] = 0; return MD_OK; }
    return md_launch_pair_counts(nl, out, (cudaStream_t)stream);
}

int md_probe_fp64_peak(int iters, double* tflops, void* stream) {
    if (iters < 1 || !tflops) return MD_ERR_ARG;
    return md_launch_probe_fp64(iters, tflops, (cudaStream_t)stream);
}

}  // extern "C"
