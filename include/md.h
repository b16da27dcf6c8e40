/* md.h -- C ABI of the B200-native many-body force library (arXiv 1610.03343 hot path).
 *
 * Write-conflict-free force evaluation for many-body potentials:
 *   1. periodic cell-list neighbour build
 *   2. per-pair kernel: bond order zeta_ij, b_ij and the partial derivative
 *      P_ij = dU_i/dr_ij of every listed pair        (Eq. 14, Alg. 3 at 295-322)
 *   3. one-thread-per-atom gather, no atomics:
 *        F_i = sum_j (P_ij - P_ji)                   (Eq. 28)
 *        W_i = -1/2 sum_j r_ij (x) (P_ij - P_ji)     (Eq. 29)
 *        J_i = sum_j r_ij (P_ji . v_i)               (Eq. 30)
 *   4. velocity-Verlet NVE
 *
 * Conventions
 *   - Units: Angstrom, fs, amu, eV; velocities in A/fs; forces in eV/A.
 *   - r_ij = r_j - r_i, minimum image in an orthorhombic fully periodic box
 *     (PAPER.md:272).  Coordinates must lie in [0, box[a]); md_velocity_verlet_step keeps them there.
 *   - Unless marked HOST, every pointer is a DEVICE pointer owned by the caller.  Vectors are
 *     structure-of-arrays: f[3][n], virial[9][n] (row-major ab, a from r, b from F: W_ab = -1/2 sum r^a F^b),
 *     heat[3][n].  Nothing in caller arrays is permuted.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls enqueue work and
 *     return without synchronising unless stated.  The force calls never wait for the device: the choice
 *     between the Tersoff kernels uses the row statistics of the last list build whose (asynchronous)
 *     copy to the host has arrived; only the very first force call on a handle waits for its build.
 *   - Return value: MD_OK or a negative md_status.  Argument errors are detected synchronously and
 *     have no side effects.  Conditions found on the device (a neighbour row longer than
 *     max_neighbors, a missing reverse entry, too many in-range neighbours) latch a status word in
 *     the handle; md_neighbors_status() synchronises the stream and returns it.
 *   - Capacity limits beyond max_neighbors (all latch MD_ERR_NEIGHBOR_OVERFLOW, results are then invalid):
 *     at most 32 neighbours of one atom inside the force range (also the limit of the warp-per-atom general
 *     path that the register Tersoff kernels use for rows longer than 4); the sorted kernels keep the in-range
 *     neighbours of a 128-atom tile in a shared-memory pool of 128 x 8 (Tersoff) or 128 x 12
 *     (Stillinger-Weber) slots, of which each of the tile's four warps (atoms sorted by in-range count) takes
 *     32 x its largest count: the four largest-per-warp counts must sum to <= 32 (Tersoff) / 48 (SW).
 *     With several elements (md_tersoff_multi_force) a tile is 256 atoms sorted into eight blocks of 32, taken
 *     four at a time: the same bound holds for the largest counts of {two largest, two smallest blocks} and of
 *     the four blocks in the middle.
 *   - There is no CPU fallback: every entry point needs a CUDA device.
 */
#ifndef MD_H_
#define MD_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    MD_OK = 0,
    MD_ERR_ARG = -1,
    MD_ERR_ALLOC = -2,
    MD_ERR_BOX_TOO_SMALL = -3,       /* fewer than 3 cells of edge >= r_list on some axis */
    MD_ERR_NEIGHBOR_OVERFLOW = -4,   /* a row needs more than max_neighbors entries */
    MD_ERR_CUDA = -5,
    MD_ERR_NO_LIST = -6,             /* force call before a list was built or imported */
    MD_ERR_LIST_ASYMMETRIC = -7,     /* j in row i but i not in row j (imported list) */
    MD_ERR_STATIC_CAPACITY = -8      /* md_tersoff_force_static: n * max_neighbors > MD_STATIC_MAX_PAIRS */
} md_status;

enum { MD_FP64 = 0, MD_FP32 = 1 };          /* arithmetic of the force kernels (reading A10) */
enum { MD_TERSOFF = 0, MD_SW = 1 };
enum { MD_MAX_NEIGHBORS = 64 };

/* Tersoff parameters, single element (Eqs. 1-6); HOST struct, copied by the call.
 * f_R = A exp(-lambda r), f_A = B exp(-mu r), f_C: 1 below R, cosine taper to 0 at S. */
typedef struct { double A, B, lambda, mu, beta, n, c, d, h, R, S; } md_tersoff_params;

/* Stillinger-Weber parameters (Ref. [18]); cutoff r_c = a*sigma; cos0 = -1/3 for Si. */
typedef struct { double epsilon, sigma, a, lambda, gamma, A, B, p, q, cos0; } md_sw_params;

/* Opaque handle: library-owned device scratch (cell arrays, NN, NL, reverse index, per-pair records). */
typedef struct md_neighbors md_neighbors;

/* Create / destroy the handle for up to n_atoms atoms and rows of up to max_neighbors
 * (1..MD_MAX_NEIGHBORS) entries.  Allocates device memory (synchronous). */
int md_neighbors_create(md_neighbors** out, int64_t n_atoms, int max_neighbors);
int md_neighbors_destroy(md_neighbors* nl);

/* Synchronises `stream`, returns the latched device status (MD_OK if none) and clears it.
 * max_count_seen (HOST, may be NULL) receives the longest row of the last build. */
int md_neighbors_status(md_neighbors* nl, int* max_count_seen, void* stream);

/* Row statistics of the current list (HOST ints, either may be NULL): the longest row and the number
 * of rows longer than 4 entries.  Waits for the last build / import on its stream to finish.  The
 * Tersoff call uses them to choose its kernel: the register kernel (k_tersoff_lean, with or without the virial
 * own half) while at most one row in 256 is longer than 4, else k_screen + the binned kernels (k_tersoff_sorted on
 * the atoms with more than 4 in-range neighbours beside k_tersoff_binned on the others; FP32: k_tersoff_hot). */
int md_neighbors_row_stats(md_neighbors* nl, int* max_row, int* rows_longer_than_4);

/* Copy the current list out / in (DEVICE int32 buffers): NN[n]; NL[max_neighbors][n] neighbour-major,
 * NL[m*n + i] = index of the m-th neighbour of atom i, rows sorted by index.
 * Import also rebuilds the reverse index; it lets a test drive the force kernels with an
 * externally built list.  Imported rows must be sorted by index and the list symmetric (j in row i <=> i in
 * row j); otherwise MD_ERR_LIST_ASYMMETRIC is latched. */
int md_neighbors_export(md_neighbors* nl, int32_t* NN, int32_t* NL, void* stream);
int md_neighbors_import(md_neighbors* nl, int64_t n, const int32_t* NN, const int32_t* NL, void* stream);

/* Step 1.  Verlet list by the cell-list method: all j != i with minimum-image
 * d2 = fma(dz,dz,fma(dy,dy,dx*dx)) < r_list*r_list (strict; reading A7).
 * box: HOST double[3].  Needs floor(box[a]/r_list) >= 3 on every axis. */
int md_build_neighbors(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                       const double box[3], double r_list, void* stream);

/* Steps 2+3 for the Tersoff potential.  vx,vy,vz are read only when heat != NULL.
 * Outputs (any may be NULL): pe[n] = U_i, f[3][n], virial[9][n], heat[3][n].
 * precision: MD_FP64 or MD_FP32 (float arithmetic on r_ij formed in double; outputs stay double). */
int md_tersoff_force(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                     const double* vx, const double* vy, const double* vz, const double box[3],
                     const md_tersoff_params* p, int precision,
                     double* pe, double* f, double* virial, double* heat, void* stream);

/* The paper's literal two-kernel scheme as an A/B against the stored-P design: Algorithm 3
 * stores b_ij and db_ij/dzeta_ij per listed pair (16 bytes), Algorithm 2
 * recomputes dU_j/dr_ji inside thread i and writes every per-atom output once; no pair records, no gather
 * kernel.  Same arguments, outputs and tolerances as md_tersoff_force. */
int md_tersoff_force_literal(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                             const double* vx, const double* vy, const double* vz, const double box[3],
                             const md_tersoff_params* p, int precision,
                             double* pe, double* f, double* virial, double* heat, void* stream);

/* Multi-element Tersoff ("systems with more than one type of atom"; reading A17 =
 * Tersoff's multicomponent form): elem[t] are the per-element parameters, the pair (a,b) uses
 * lambda, mu = arithmetic means, A, B, R, S = geometric means, and chi[a][b] (chi[a][a] = 1) multiplies the
 * attractive term; g and b use c, d, h, beta, n of the CENTRAL atom.  types: DEVICE int32[n], values in
 * 0..ntypes-1.  The list must have been built with r_list >= max S + skin.  n < 2^28.  Same outputs, layouts
 * and error behaviour as md_tersoff_force; with ntypes = 1 it computes exactly that potential. */
enum { MD_MAX_TYPES = 4 };
typedef struct {
    int ntypes;
    md_tersoff_params elem[MD_MAX_TYPES];
    double chi[MD_MAX_TYPES][MD_MAX_TYPES];
} md_tersoff_multi_params;
int md_tersoff_multi_force(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                           const double* vx, const double* vy, const double* vz, const double box[3],
                           const int32_t* types, const md_tersoff_multi_params* p, int precision,
                           double* pe, double* f, double* virial, double* heat, void* stream);

/* Same for Stillinger-Weber; three-body energy is attributed to the central atom (reading A6). */
int md_sw_force(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                const double* vx, const double* vy, const double* vz, const double box[3],
                const md_sw_params* p, int precision,
                double* pe, double* f, double* virial, double* heat, void* stream);

/* Step 4.  One half of a velocity-Verlet step, in place.
 *   phase 0: v += (dt/2)(kappa/m) f ; x += dt v ; wrap into [0, box)
 *   phase 1: v += (dt/2)(kappa/m) f
 * kappa = 9.648533215665e-3 (A/fs^2)/(eV/A/amu). */
int md_velocity_verlet_step(int phase, int64_t n, double* x, double* y, double* z,
                            double* vx, double* vy, double* vz, const double* f,
                            double mass_amu, double dt_fs, const double box[3], void* stream);

/* Convenience: nsteps NVE steps composed of the four calls above, list rebuilt after the drift of
 * every step s (counted from first_step) with s % rebuild_every == 0.  `params` is a HOST md_tersoff_params* or md_sw_params*
 * according to `potential`.  f[3][n] must hold the forces of the incoming state if f_valid != 0,
 * otherwise they are computed first (with a list built at the incoming positions).
 * pe[n] (may be NULL) receives U_i of the final state. */
int md_nve_run(md_neighbors* nl, int potential, const void* params, int precision, int64_t n,
               double* x, double* y, double* z, double* vx, double* vy, double* vz,
               double* f, int f_valid, double* pe, const double box[3], double mass_amu, double dt_fs,
               int first_step, int nsteps, int rebuild_every, double r_list, void* stream);

/* NPT by weak coupling: Berendsen thermostat and barostat, the paper's benchmark ensemble (
 * SURVEY 8(f-3); reading A18).  Each step is a velocity-Verlet step (as md_nve_run) followed by
 *   T = 2 KE / (3 n kB),  P = (2 KE + tr sum_i W_i) / (3 V)      with sum_i W_i of Eq. (29), formed as
 *   -sum_ij r_ij (x) dU_i/dr_ij (the same sum regrouped pair by pair; per-atom W_i is not stored by this call)
 *   v *= sqrt(1 + (dt/tau_T)(T0/T - 1));   x, box *= (1 - beta (dt/tau_P)(P0 - P))^(1/3)
 * T0 in K, tau in fs, P0 in eV/A^3 (1 eV/A^3 = 160.21766 GPa), beta (compressibility) in A^3/eV.
 * box: HOST double[3], read and UPDATED.  T_trace, P_trace: HOST [nsteps] (may be NULL), the values measured
 * before each step's scaling.  The call reads two scalars back per step, so it synchronises `stream`. */
typedef struct { double T0, tau_T, P0, tau_P, beta; } md_berendsen_params;
int md_npt_run(md_neighbors* nl, int potential, const void* params, int precision, int64_t n,
               double* x, double* y, double* z, double* vx, double* vy, double* vz,
               double* f, int f_valid, double box[3], double mass_amu, double dt_fs,
               int first_step, int nsteps, int rebuild_every, double r_list,
               const md_berendsen_params* b, double* T_trace, double* P_trace, void* stream);

/* Green-Kubo workload (the application of the paper's Ref. [27]): NVE steps as
 * md_nve_run (the steps between two samples run as one fused segment), and after every `sample_every`-th step the
 * total heat current of that state:
 *   J_pot = sum_i J_i (Eq. 30)      J_kin = sum_i (m v_i^2 / 2 + U_i) v_i   (convective part)
 * in eV A/fs.  J_pot, J_kin: HOST [nsteps / sample_every][3] (either may be NULL).  Reads six scalars back per
 * sample, so it synchronises `stream`.  The autocorrelation and its integral are the caller's
 * (paper_1610_03343_b200.green_kubo). */
int md_nve_heat_run(md_neighbors* nl, int potential, const void* params, int precision, int64_t n,
                    double* x, double* y, double* z, double* vx, double* vy, double* vz,
                    double* f, int f_valid, const double box[3], double mass_amu, double dt_fs,
                    int first_step, int nsteps, int rebuild_every, double r_list, int sample_every,
                    double* J_pot, double* J_kin, void* stream);

/* End-to-end variant with HOST buffers (pinned or pageable): copies x,y,z,vx,vy,vz to the device,
 * runs md_nve_run from scratch (f_valid = 0), copies x,y,z,vx,vy,vz, f[3][n] and pe[n] back and
 * synchronises.  Device buffers are owned by the handle.  The velocities are uploaded on a second, handle-owned
 * stream and joined before the first kick, so the list build and the first force evaluation (positions only)
 * overlap with that half of the transfer.  Returns the latched device status (as md_neighbors_status would)
 * since it has synchronised anyway. */
int md_nve_run_host(md_neighbors* nl, int potential, const void* params, int precision, int64_t n,
                    double* x, double* y, double* z, double* vx, double* vy, double* vz,
                    double* f, double* pe, const double box[3], double mass_amu, double dt_fs,
                    int nsteps, int rebuild_every, double r_list, void* stream);

/* Diagnostic: runs an independent-chain DFMA kernel for `iters` fused multiply-adds per thread on a
 * full grid and returns the achieved FP64 rate in *tflops (HOST); used as the measured ALU peak of
 * the roofline.  Synchronous. */
int md_probe_fp64_peak(int iters, double* tflops, void* stream);

/* Diagnostic: out[k] = fn(in[k]) with the FP64 device functions the pair kernels use (fastmath.cuh):
 * fn 0 exp, 1 log (in > 0, normal), 2 reciprocal, 3 reciprocal square root, 4 sin and 5 cos on [0, pi].
 * DEVICE buffers of n doubles.  Lets a test bound their error against a long-double reference. */
int md_math_probe(int fn, int64_t n, const double* in, double* out, void* stream);

/* Per-kernel-kind device timing (CUDA events on the launching stream) and launch counts.
 * md_profile_enable(nl, 1) starts recording an event pair around every kernel group launched
 * through `nl`; md_profile_read synchronises the device, adds up the elapsed times and resets.
 * kinds: 0 neighbour build, 1 pair kernel, 2 gather kernel, 3 integrator.  ms[4], launches[4] HOST.
 * Launch counts (kernels enqueued) are kept whether or not timing is enabled. */
enum { MD_KIND_BUILD = 0, MD_KIND_PAIR = 1, MD_KIND_GATHER = 2, MD_KIND_INTEGRATE = 3, MD_N_KINDS = 4 };
int md_profile_enable(md_neighbors* nl, int enable);
int md_profile_read(md_neighbors* nl, double* ms, int64_t* launches);

/* Diagnostic: exact integer counts over the current list and the in-range masks the LAST force call left
 * (HOST int64 out[3]): out[0] = listed directed pairs (sum of row lengths), out[1] = directed pairs inside the
 * force range, out[2] = ordered in-range triplets sum_i M_i (M_i - 1).  bench.py multiplies them by the
 * per-unit operation counts of DESIGN.md section 3 to get the algorithmic work of a launch.  Synchronous. */
int md_pair_counts(md_neighbors* nl, int64_t out[3], void* stream);

/* Tersoff energies and forces for callers that may not allocate (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): the stored-P scheme of steps 2+3 (P_ij = dU_i/dr_ij per listed pair, Eq. 14 at
 * PAPER.md:173-176; F_i = sum_j (P_ij - P_ji), Eq. 28 at PAPER.md:330) with its per-pair records in a fixed
 * file-scope device array of the library instead of a handle: 32 bytes x MD_STATIC_MAX_PAIRS + 256 bytes = 16 MiB,
 * held by every GPU that loads the library until the process exits.  The call needs no md_neighbors handle and calls
 * no cudaMalloc, cudaFree or allocating library routine; FP64 arithmetic, the same formulas and device functions as
 * md_tersoff_force.
 *   n, max_neighbors: n * max_neighbors <= MD_STATIC_MAX_PAIRS, else MD_ERR_STATIC_CAPACITY (nothing is enqueued);
 *       1 <= max_neighbors <= MD_MAX_NEIGHBORS.
 *   NN[n], NL[max_neighbors][n] (DEVICE int32): the list in the layout of md_neighbors_export; it must be symmetric
 *       (j in row i <=> i in row j).  Rows need not be sorted.
 *   x, y, z (DEVICE), box (HOST double[3]): coordinates in [0, box[a]), minimum image, box[a] >= 2 S.
 *   pe[n], f[3][n] (DEVICE, either may be NULL): U_i and F_i.
 *   status (DEVICE int32*, may be NULL): receives 0, or bit 0 (1) = some NN[i] > max_neighbors (row clamped),
 *       bit 1 (2) = some listed j has no entry i in its own row (F of that atom is NaN) or is
 *       outside [0, n) (the row ends there); written on `stream`.
 * Every call on a device shares the one array, and the array keeps the last call's contents: each call clears its
 * status word and writes every record before reading it, so calls on ONE stream (or ordered by events) are
 * independent of each other, but two calls that overlap on the GPU (two streams, two host threads) race and give
 * wrong results.  The first call on a device looks the array's address up (cudaGetSymbolAddress, loads the
 * module): make it outside stream capture.  Asynchronous like the other force calls. */
enum { MD_STATIC_MAX_PAIRS = 524288 };
int md_tersoff_force_static(int64_t n, int max_neighbors, const int32_t* NN, const int32_t* NL,
                            const double* x, const double* y, const double* z, const double box[3],
                            const md_tersoff_params* p, double* pe, double* f, int32_t* status, void* stream);

/* Library version string (HOST, static storage). */
const char* md_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MD_H_ */
