// common.cuh -- handle layout and small device helpers shared by the CUDA translation units.
// Product code: shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "md.h"

#define MD_CUDA_TRY(expr)                         \
    do {                                          \
        cudaError_t e__ = (expr);                 \
        if (e__ != cudaSuccess) return MD_ERR_CUDA; \
    } while (0)

// device-latched status bits (md_neighbors::d_status[0])
enum : int {
    MD_DEV_ROW_OVERFLOW = 1,     // neighbour row longer than max_neighbors
    MD_DEV_NO_REVERSE = 2,       // i not found in row j
    MD_DEV_INRANGE_OVERFLOW = 4  // more in-range neighbours than the pair kernel's cap
};

// 32-byte per-pair record {Px, Py, Pz, pad} = one DRAM sector (FP64 mode);
// FP32 mode stores float4 in the first 16 bytes of a 16-byte-strided array.
struct __align__(32) PairRec64 { double x, y, z, w; };

// Head of a list row for the crystal pair kernel: first four entries, their reverse slots, the row length (32 bytes).
struct __align__(32) MdRowHead { int j[4]; unsigned rev; int nn; int pad[2]; };

struct md_neighbors {
    int64_t n_cap;          // capacity in atoms
    int64_t n;              // atoms of the current list (0 = none)
    int K;                  // max_neighbors
    // list
    int32_t* NN;            // [n]
    int32_t* NL;            // [K][n] neighbour-major
    uint8_t* REV;           // [K][n] position of i in row NL[m][i]
    MdRowHead* HEAD;        // [n] the first four entries of each row with their reverse slots (k_reverse writes it)
    // per-pair records, pushed layout: Q[m*n + i] = P_{j i}, j = NL[m][i]
    void* Q;                // K*n*32 bytes
    unsigned long long* MASK;  // [n] bit m set <=> slot m is inside the force range
    int32_t* bin_list;      // [3][n] atom indices by in-range-count bin (pair_sort.cuh, Bins), written by k_screen
    int32_t* bin_count;     // [2][4] two sets used alternately (bin_phase), each zeroed by the launch before its use
    int bin_phase;
    int gather_pdl;         // the last pair launch wants the fused gather as its programmatic dependent (measured per
                            // path: +3 % after k_tersoff_lean, 0 after k_sw_sorted, -6 % after k_tersoff_hot, whose 148
                            // long-running tail CTAs then share their SMs with early-resident gather CTAs)
    int virial_own_only;    // md_npt_run: the force call leaves only the pair kernel's own half -1/2 sum_j r_ij (x) P_ij in
                            // `virial` (the gather runs forces-only); the TOTAL virial is twice the sum of the own halves
    int q_dense;            // layout of the records the last pair kernel wrote: 1 = slot counts in-range entries
                            // (sorted kernels, MASK known beforehand), 0 = slot is the list position
    // cell structures
    int64_t cell_cap;
    int32_t* cell_count;    // [ncell+1] -> exclusive scan in place = cell_start
    int32_t* cell_of;       // [n]
    int32_t* rank_in_cell;  // [n]
    double4* sorted;        // [n] {x,y,z, index bits} in cell order
    float4* sortedf;        // [n] the same in float (FP32 screen of the candidate search)
    int32_t* scan_blocks;   // block sums scratch
    // status
    int* d_status;          // [3]: status bits, max row length seen, number of rows longer than 4
    // row statistics of the list, mirrored to the host for kernel selection: written by an async copy at
    // the end of every build / import.  A force call never waits for them (md_list_row_stats(wait = 0)): it
    // uses the statistics of the last build whose copy has arrived, and waits only if there are none yet.
    int* h_maxrow;          // pinned [2]: longest row, number of rows longer than 4 (landing zone of the copy)
    int row_stats[2];       // the last values known to have arrived
    int row_stats_valid;
    cudaEvent_t ev_list;
    int maxrow_pending;
    // profiling (md_profile_*)
    int prof_on;
    int64_t launches[MD_N_KINDS];
    std::vector<cudaEvent_t>* ev_pool;                 // all events ever created (reused)
    std::vector<int>* ev_kind;                         // kind of each recorded pair
    size_t ev_used;                                    // events handed out since the last read
    double ms_acc[MD_N_KINDS];
    // Berendsen NPT (md_npt_run): per-atom virial [9][n], reduction scratch, pinned landing zone
    double* npt_w; int64_t npt_cap; double* npt_part; double* h_npt; cudaEvent_t npt_event;
    // md_nve_run_host: the velocities travel on a second stream while the list build and the first force
    // evaluation (which need positions only) already run
    cudaStream_t s_copy; cudaEvent_t ev_fork, ev_join;
    // e2e device state (md_nve_run_host)
    double* e2e;            // [13][n] x,y,z,vx,vy,vz,f[3],pe + spare
    int64_t e2e_cap;
};

__device__ __forceinline__ double md_min_image(double d, double L, double halfL) {
    // reading A7: coordinates in [0,L) => |d| < L, one conditional shift
    if (d > halfL) d -= L;
    else if (d < -halfL) d += L;
    return d;
}

// velocity-Verlet pieces shared by integrate.cu and the fused gather kernel
constexpr double MD_KAPPA = 9.648533215665e-3;   // (A/fs^2) per (eV/A/amu)
constexpr double MD_KB = 8.617333262e-5;         // Boltzmann constant, eV/K
__device__ __forceinline__ double md_wrap(double c, double L) {
    c -= L * floor(c / L);
    return (c >= L || c < 0.0) ? 0.0 : c;        // reading A8
}
// What md_nve_run fuses into the gather kernel after the force is complete (nullptr = nothing):
//   mode 1: v += hk F                                  (second half-kick of the step; F is stored)
//   mode 2: v += hk F; v += hk F; x += dt v; wrap      (that kick and the next step's kick+drift; F is
//           not stored: nothing reads it before the next force evaluation overwrites it)
struct VVFuse {
    int mode;
    double hk, dt;
    double *x, *y, *z, *vx, *vy, *vz;
    int pdl_pair;   // 1: the kernel launched just before this step's pair phase was this loop's own k_gather_vv /
                    // k_kick_drift and the list has not changed since (md_launch_pdl below)
};

// Programmatic dependent launch (sm_90+; md_nve_run only).  A kernel launched with `pdl` may start while the
// kernel before it on the stream is draining its last CTAs: everything it does before md_grid_wait() overlaps
// with that tail (and with the launch latency), so it may only READ there what the kernel before it does not
// write.  md_grid_wait() returns when that kernel has completed and its writes are visible;
// md_grid_release() lets the NEXT kernel on the stream be scheduled once every CTA of this one has called it.
// Every kernel calls release only AFTER its own wait, so "the kernel before has completed" is transitive: when a
// dependent starts, every earlier kernel of the stream is complete.  Launched without the attribute both calls
// are no-ops.
__device__ __forceinline__ void md_grid_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void md_grid_release() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <class... KArgs, class... Args>
inline cudaError_t md_launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s,
                                 bool pdl, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// RAII scope: counts `nk` kernel launches of `kind` and, if profiling is on, brackets them with events.
struct ProfScope {
    md_neighbors* nl; cudaStream_t s; cudaEvent_t e1; bool on;
    ProfScope(md_neighbors* nl_, int kind, int nk, cudaStream_t s_);
    ~ProfScope();
};

// Shared-memory pool of the sorted loop kernels (pair_sort.cuh), in in-range slots per atom of a 128-atom
// tile.  A warp of the sorted tile takes 32 x (largest M among its atoms) slots, so the caps documented in
// md.h are: sum over the tile's four warps of that largest M <= 4 x the figure below.
constexpr int MD_SW_POOL_PER_ATOM = 12;
constexpr int MD_TERSOFF_POOL_PER_ATOM = 8;

// cudaFuncAttributeMaxDynamicSharedMemorySize, set once per (device, kernel); thread-safe (api.cu)
int md_allow_dynamic_smem(const void* kernel, int bytes);

// kernels' launchers (defined in the .cu files)
int md_launch_build(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                    const double box[3], double r_list, cudaStream_t s);
int md_launch_reverse(md_neighbors* nl, cudaStream_t s, int check);   // check = 1: imported list (verify symmetry)
int md_list_row_stats(md_neighbors* nl, int* max_row, int* long_rows, int wait);   // host copies; wait = 1: of the current list
int md_launch_tersoff(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                      const double* vx, const double* vy, const double* vz, const double box[3],
                      const md_tersoff_params* p, int precision, double* pe, double* f, double* virial,
                      double* heat, const VVFuse* vv, cudaStream_t s);
int md_launch_tersoff_literal(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                              const double* vx, const double* vy, const double* vz, const double box[3],
                              const md_tersoff_params* p, int precision, double* pe, double* f, double* virial,
                              double* heat, cudaStream_t s);
int md_launch_tersoff_multi(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                            const double* vx, const double* vy, const double* vz, const double box[3],
                            const int32_t* types, const md_tersoff_multi_params* p, int precision, double* pe,
                            double* f, double* virial, double* heat, cudaStream_t s);
int md_launch_sw(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                 const double* vx, const double* vy, const double* vz, const double box[3],
                 const md_sw_params* p, int precision, double* pe, double* f, double* virial,
                 double* heat, const VVFuse* vv, cudaStream_t s);
int md_launch_gather(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                     const double* vx, const double* vy, const double* vz, const double box[3],
                     int precision, double* f, double* virial, double* heat, const VVFuse* vv, cudaStream_t s);
int md_launch_vv(md_neighbors* nl, int phase, int64_t n, double* x, double* y, double* z, double* vx, double* vy, double* vz,
                 const double* f, double mass, double dt, const double box[3], cudaStream_t s,
                 double lam = 1.0, double mu = 1.0);   // phase 0 only: v *= lam, x *= mu first (Berendsen scaling of md_npt_run)
const double* md_math_tables();   // device tables of fastmath.cuh for the current device (nullptr on failure)
int md_launch_probe_fp64(int iters, double* tflops, cudaStream_t s);
int md_launch_vv_dev(md_neighbors* nl, int64_t n, double* x, double* y, double* z, double* vx, double* vy, double* vz,
                     const double* f, double mass, double dt, const double* d_scal, cudaStream_t s);
// sums, thermostat / barostat factors and the scaled box on the device (d_scal = md_npt_scal(nl)), copy to the host
// enqueued; md_npt_sums_wait blocks until that copy has arrived: out = {sum v^2, tr sum W^own, lam, mu, Lx, Ly, Lz}
int md_launch_npt_sums(md_neighbors* nl, int64_t n, double* vx, double* vy, double* vz,
                       const double* W, const double* f, double hk, double mass, double dt, const double box[3],
                       const md_berendsen_params* b, cudaStream_t s);
int md_npt_sums_wait(md_neighbors* nl, double out[7]);
const double* md_npt_scal(md_neighbors* nl);
int md_launch_npt_scale(md_neighbors* nl, int64_t n, double* x, double* y, double* z, double* vx, double* vy,
                        double* vz, double lam, double mu, cudaStream_t s);
int md_launch_heat_sums(md_neighbors* nl, int64_t n, const double* vx, const double* vy, const double* vz,
                        const double* pe, const double* J, double mass, double out[6], cudaStream_t s);
int md_npt_scratch_doubles();
int md_launch_pair_counts(md_neighbors* nl, int64_t out[3], cudaStream_t s);
