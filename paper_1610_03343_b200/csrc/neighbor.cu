// neighbor.cu -- periodic cell-list Verlet neighbour build (A7).
//
//   k_bin      cell id per atom + histogram (integer atomics; the force path has none)
//   k_scan_*   exclusive prefix sum of the histogram with warp-shuffle scans (counting sort)
//   k_scatter  atoms -> cell order as 32-byte {x,y,z,index} records, plus a 16-byte float copy
//   k_search   one thread per atom (cell order): 27-cell search.  Candidates are screened in FP32 on
//              the float copy (the FP64 pipe would otherwise bound the build: ~58 candidates x ~15
//              FP64 instructions per atom, more than the Tersoff force itself); the few that pass are
//              decided by the canonical FP64 predicate, strict d2 < r_list^2.  The z-neighbour cells
//              of a column are contiguous in cell order, so an interior atom scans 9 ranges, not 27.
//              Rows are kept sorted by index in a shared-memory scratch [K][128] (no local memory) and
//              stored neighbour-major, NL[m*n+i]
//   k_reverse  REV[m*n+i] = position of i in row NL[m*n+i] (binary search on the sorted row)
#include "common.cuh"

namespace {

struct Grid {
    int nc[3];
    double inv_cell[3];   // nc / L
    double L[3], halfL[3];
    double rc2;
};

__device__ __forceinline__ int cell_coord(double c, double inv, int nc) {
    int k = (int)(c * inv);
    k = k < 0 ? 0 : k;
    return k >= nc ? nc - 1 : k;
}

__global__ void k_bin(int64_t n, const double* __restrict__ x, const double* __restrict__ y,
                      const double* __restrict__ z, Grid g, int32_t* __restrict__ cell_of,
                      int32_t* __restrict__ rank, int32_t* __restrict__ cell_count) {
    md_grid_wait();                                          // chained build kernels: see md_launch_build
    md_grid_release();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int cx = cell_coord(x[i], g.inv_cell[0], g.nc[0]);
    const int cy = cell_coord(y[i], g.inv_cell[1], g.nc[1]);
    const int cz = cell_coord(z[i], g.inv_cell[2], g.nc[2]);
    const int c = (cx * g.nc[1] + cy) * g.nc[2] + cz;
    cell_of[i] = c;
    rank[i] = atomicAdd(&cell_count[c], 1);
}

// ---- exclusive scan: tile-local scan, scan of tile totals, add back -------------------------
constexpr int SCAN_BT = 512;
constexpr int SCAN_IT = 4;

__device__ __forceinline__ int warp_inclusive_scan(int v) {
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v += t;
    }
    return v;
}

// block-wide exclusive scan of one value per thread; returns the exclusive prefix, *total = block sum
__device__ __forceinline__ int block_exclusive_scan(int v, int* total, int* warp_sums /*[32]*/) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int inc = warp_inclusive_scan(v);
    if (lane == 31) warp_sums[wid] = inc;
    __syncthreads();
    if (wid == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        int s = lane < nw ? warp_sums[lane] : 0;
        s = warp_inclusive_scan(s);
        warp_sums[lane] = s;
    }
    __syncthreads();
    const int base = wid ? warp_sums[wid - 1] : 0;
    *total = warp_sums[31];
    __syncthreads();
    return base + inc - v;
}

__global__ void k_scan_local(int32_t* __restrict__ data, int64_t n, int32_t* __restrict__ tile_sums) {
    md_grid_wait();                                          // chained build kernels: see md_launch_build
    md_grid_release();
    __shared__ int warp_sums[32];
    const int64_t base = ((int64_t)blockIdx.x * SCAN_BT + threadIdx.x) * SCAN_IT;
    int v[SCAN_IT];
    int s = 0;
#pragma unroll
    for (int k = 0; k < SCAN_IT; ++k) {
        v[k] = base + k < n ? data[base + k] : 0;
        s += v[k];
    }
    int total;
    int pre = block_exclusive_scan(s, &total, warp_sums);
#pragma unroll
    for (int k = 0; k < SCAN_IT; ++k) {
        if (base + k < n) data[base + k] = pre;
        pre += v[k];
    }
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

__global__ void k_scan_tiles(int32_t* __restrict__ tile_sums, int ntiles) {
    md_grid_wait();                                          // chained build kernels: see md_launch_build
    md_grid_release();
    __shared__ int warp_sums[32];
    int carry = 0;
    for (int b = 0; b < ntiles; b += blockDim.x) {
        const int idx = b + threadIdx.x;
        const int v = idx < ntiles ? tile_sums[idx] : 0;
        int total;
        const int pre = block_exclusive_scan(v, &total, warp_sums);
        if (idx < ntiles) tile_sums[idx] = carry + pre;
        carry += total;
    }
}

__global__ void k_scan_add(int32_t* __restrict__ data, int64_t n, const int32_t* tile_sums,   // plain loads: note below
                           int32_t grand_total) {
    md_grid_wait();                                          // chained build kernels: see md_launch_build
    md_grid_release();
    const int64_t base = ((int64_t)blockIdx.x * SCAN_BT + threadIdx.x) * SCAN_IT;
    const int add = tile_sums[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_IT; ++k)
        if (base + k < n) data[base + k] += add;
    if (blockIdx.x == 0 && threadIdx.x == 0) data[n] = grand_total;
}

__global__ void k_scatter(int64_t n, const double* __restrict__ x, const double* __restrict__ y,
                          const double* __restrict__ z, const int32_t* __restrict__ cell_of,
                          const int32_t* __restrict__ rank, const int32_t* cell_start,
                          double4* __restrict__ sorted, float4* __restrict__ sortedf) {
    md_grid_wait();                                          // chained build kernels: see md_launch_build
    md_grid_release();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int pos = cell_start[cell_of[i]] + rank[i];
    const double xi = x[i], yi = y[i], zi = z[i];
    sorted[pos] = make_double4(xi, yi, zi, __longlong_as_double((long long)i));
    sortedf[pos] = make_float4((float)xi, (float)yi, (float)zi, __int_as_float((int)i));
}

constexpr int SEARCH_BT = 128;
#ifndef SEARCH_UNROLL
#define SEARCH_UNROLL 2
#endif

#ifndef SEARCH_MIN_CTAS
#define SEARCH_MIN_CTAS 8
#endif
__global__ void __launch_bounds__(SEARCH_BT, SEARCH_MIN_CTAS)
k_search(int64_t n, Grid g, const double4* sorted, const float4* sortedf,
         const int32_t* __restrict__ cell_start, int K, float rc2_lo, float rc2_hi, int32_t* __restrict__ NN,
         int32_t* __restrict__ NL, int* __restrict__ status) {
    md_grid_wait();
    md_grid_release();
    extern __shared__ int s_nb[];                            // [K + 1][SEARCH_BT]: this thread's row (+ a scratch slot)
    const int tid = threadIdx.x;
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + tid;
    if (t >= n) return;
    const double4 a = sorted[t];
    const int i = (int)__double_as_longlong(a.w);
    const float xf = (float)a.x, yf = (float)a.y, zf = (float)a.z;
    const int cx = cell_coord(a.x, g.inv_cell[0], g.nc[0]);  // as in k_bin, bit for bit
    const int cy = cell_coord(a.y, g.inv_cell[1], g.nc[1]);
    const int cz = cell_coord(a.z, g.inv_cell[2], g.nc[2]);
    const float Lxf = (float)g.L[0], Lyf = (float)g.L[1], Lzf = (float)g.L[2];
    int cnt = 0;

    // One candidate, branch-free.  The FP32 distance decides whenever it is outside the band [rc2_lo, rc2_hi)
    // that its error bound leaves open (see md_launch_build).  A candidate below rc2_hi is a provisional hit; one
    // inside the band (about one candidate in 10^4) only marks the row as `unc`ertain, and such a row is checked
    // entry by entry with the canonical FP64 predicate of reading A7 after the scan, so the outcome is always that
    // predicate's.  The candidate's cell-order position is written to the row's next slot unconditionally and
    // the slot advances only on a hit (no branch, no reconvergence point in the loop: the branchy version spent
    // ~35 instructions per candidate, this one ~16).
    unsigned unc = 0u;
    const int Kslot = K;                                     // row slot K is a scratch slot: entries 0..K-1 stay valid on overflow
    auto test = [&](int q, const float4 bf, float xs, float ys, float zs) {
        const float fx = bf.x - xs, fy = bf.y - ys, fz = bf.z - zs;
        const float d2f = fmaf(fz, fz, fmaf(fy, fy, fx * fx));
        const bool hit = d2f < rc2_hi && __float_as_int(bf.w) != i;
        unc |= (hit && d2f >= rc2_lo) ? 1u : 0u;
        s_nb[min(cnt, Kslot) * SEARCH_BT + tid] = q;
        cnt += hit ? 1 : 0;
    };
    // a contiguous range of the cell-ordered array, SEARCH_UNROLL candidates in flight at a time
    auto scan = [&](int beg, int end, float xs, float ys, float zs) {
        const float4 far = make_float4(1e18f, 1e18f, 1e18f, __int_as_float(i));
        for (int q = beg; q < end; q += SEARCH_UNROLL) {
            float4 c[SEARCH_UNROLL];
#pragma unroll
            for (int u = 0; u < SEARCH_UNROLL; ++u) c[u] = (u == 0 || q + u < end) ? sortedf[q + u] : far;
#pragma unroll
            for (int u = 0; u < SEARCH_UNROLL; ++u) test(q + u, c[u], xs, ys, zs);
        }
    };

    int axs[3], ays[3];
    float xss[3], yss[3];
#pragma unroll
    for (int o = 0; o < 3; ++o) {                            // the reference is shifted, not the candidate
        int ax = cx + o - 1; float xs = xf;
        if (ax < 0) { ax += g.nc[0]; xs += Lxf; } else if (ax >= g.nc[0]) { ax -= g.nc[0]; xs -= Lxf; }
        int ay = cy + o - 1; float ys = yf;
        if (ay < 0) { ay += g.nc[1]; ys += Lyf; } else if (ay >= g.nc[1]) { ay -= g.nc[1]; ys -= Lyf; }
        axs[o] = ax; xss[o] = xs; ays[o] = ay; yss[o] = ys;
    }
    // The z-neighbour cells of a column are contiguous in cell order, so the 27 cells are 9 ranges (the window
    // cz-1..cz+1 clipped to the column) plus, for an atom in the first or last cell of its column, the 9 single
    // cells on the far side of the periodic boundary.  All lanes walk the same loop structure: a lane without
    // a wrapped part sees nine empty ranges there (a warp of 32 cell-ordered atoms spans ~15 of a column's cells,
    // so every other warp holds such an atom; as a separate 27-range code path it cost those warps a second pass).
    const int nz = g.nc[2];
    const int zlo = cz > 0 ? cz - 1 : 0, zhi = cz < nz - 1 ? cz + 1 : nz - 1;
    int beg[9], end[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) {                            // all 18 bounds are fetched before the first scan
        const int base = (axs[c / 3] * g.nc[1] + ays[c % 3]) * nz;
        beg[c] = cell_start[base + zlo];
        end[c] = cell_start[base + zhi + 1];
    }
#pragma unroll
    for (int c = 0; c < 9; ++c) scan(beg[c], end[c], xss[c / 3], yss[c % 3], zf);
    if (cz == 0 || cz == nz - 1) {
        const int wz = cz == 0 ? nz - 1 : 0;
        const float zs = cz == 0 ? zf + Lzf : zf - Lzf;
#pragma unroll
        for (int c = 0; c < 9; ++c) {
            const int base = (axs[c / 3] * g.nc[1] + ays[c % 3]) * nz + wz;
            beg[c] = cell_start[base];
            end[c] = cell_start[base + 1];
        }
#pragma unroll
        for (int c = 0; c < 9; ++c) scan(beg[c], end[c], xss[c / 3], yss[c % 3], zs);
    }
    if (cnt > K) { atomicOr(&status[0], MD_DEV_ROW_OVERFLOW); cnt = K; }   // counted before the check below: conservative
    {   // cell-order position -> atom index; rows marked uncertain keep only what the FP64 predicate confirms
        int out = 0;
        for (int m = 0; m < cnt; ++m) {
            const int q = s_nb[m * SEARCH_BT + tid];
            const double4 b = sorted[q];
            bool ok = true;
            if (unc) {
                const double dx = md_min_image(__dsub_rn(b.x, a.x), g.L[0], g.halfL[0]);
                const double dy = md_min_image(__dsub_rn(b.y, a.y), g.L[1], g.halfL[1]);
                const double dz = md_min_image(__dsub_rn(b.z, a.z), g.L[2], g.halfL[2]);
                ok = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx))) < g.rc2;
            }
            if (ok) s_nb[out++ * SEARCH_BT + tid] = (int)__double_as_longlong(b.w);
        }
        cnt = out;
    }
    {   // longest row: one atomic per warp
        const unsigned act = __activemask();
        const int wmax = __reduce_max_sync(act, cnt);
        if ((tid & 31) == __ffs(act) - 1 && wmax > __ldcg(&status[1])) atomicMax(&status[1], wmax);   // 16 000 warps, one word: only a larger value goes out
    }
    NN[i] = cnt;
    for (int m = 1; m < cnt; ++m) {                          // insertion sort of the (short) row by index
        const int j = s_nb[m * SEARCH_BT + tid];
        int p = m;
        while (p > 0 && s_nb[(p - 1) * SEARCH_BT + tid] > j) {
            s_nb[p * SEARCH_BT + tid] = s_nb[(p - 1) * SEARCH_BT + tid];
            --p;
        }
        s_nb[p * SEARCH_BT + tid] = j;
    }
    for (int m = 0; m < cnt; ++m) NL[(int64_t)m * n + i] = s_nb[m * SEARCH_BT + tid];
}

// REV[m*n+i] = position of i in row j = NL[m*n+i].  Rows are sorted by index, so that position is the
// number of entries of row j smaller than i: a branch-free binary search of fixed depth (the longest row of
// this list, read from the status word the search kernel just wrote), four searches of a thread interleaved so
// that their dependent loads overlap.  (Round 1 walked row j entry by entry with an early exit: a chain of
// up to NN[j] dependent loads per entry, 124 us per build for the 16-18-entry Stillinger-Weber rows.)
// CHECK = true (imported lists): every entry is range-checked and the hit verified, a miss latches
// MD_DEV_NO_REVERSE.  Lists built by k_search are symmetric by construction (the predicate is) and skip that.
template <bool CHECK>
__global__ void __launch_bounds__(128)
k_reverse(int64_t n, int K, const int32_t* NN, const int32_t* NL,
          uint8_t* __restrict__ REV, int* __restrict__ status, MdRowHead* __restrict__ HEAD) {
    md_grid_wait();
    md_grid_release();
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int nn = min(NN[i], K);
    {   // longest row (also for imported lists): one atomic per warp
        const unsigned act = __activemask();
        const int wmax = __reduce_max_sync(act, nn);
        const int nlong = __popc(__ballot_sync(act, nn > 4));
        if ((threadIdx.x & 31) == __ffs(act) - 1) {
            if (wmax > __ldcg(&status[1])) atomicMax(&status[1], wmax);
            if (nlong) atomicAdd(&status[2], nlong);
        }
    }
    for (int m0 = 0; m0 < nn; m0 += 4) {
        int j[4], lo[4], hi[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int m = m0 + u < nn ? m0 + u : m0;
            j[u] = NL[(int64_t)m * n + i];
            if (CHECK && (unsigned)j[u] >= (unsigned long long)n) { atomicOr(&status[0], MD_DEV_NO_REVERSE); j[u] = (int)i; }
        }
        // The first four entries of every partner row are read unconditionally (16 independent loads: for
        // crystal rows that is the whole answer after two dependent levels); the position is the number of
        // entries smaller than i, and only if all four are smaller does a binary search of [4, NN[j]) follow.
        int nj[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) nj[u] = min(NN[j[u]], K);
        int head[4][4];
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int q = 0; q < 4; ++q) head[u][q] = NL[(int64_t)(q < K ? q : 0) * n + j[u]];
        bool live = false;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            int c = 0;
#pragma unroll
            for (int q = 0; q < 4; ++q) c += (q < nj[u] && head[u][q] < (int)i) ? 1 : 0;
            lo[u] = c;
            hi[u] = c == 4 ? nj[u] : c;                          // c < 4: found (lo == hi); else search [4, nj)
            live = live || lo[u] < hi[u];
        }
        if (__any_sync(__activemask(), live)) {
#pragma unroll 1
            for (int it = 0; it < 7; ++it) {                     // rows have at most 64 entries
                int v[4], mid[4];
                bool more = false;
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    mid[u] = (lo[u] + hi[u]) >> 1;
                    more = more || lo[u] < hi[u];
                    v[u] = lo[u] < hi[u] ? NL[(int64_t)mid[u] * n + j[u]] : 0;
                }
                if (!__any_sync(__activemask(), more)) break;
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (lo[u] < hi[u]) { if (v[u] < (int)i) lo[u] = mid[u] + 1; else hi[u] = mid[u]; }
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (m0 + u >= nn) continue;
            if (CHECK) {
                const bool found = lo[u] < min(NN[j[u]], K) && NL[(int64_t)lo[u] * n + j[u]] == (int)i;
                if (!found) { atomicOr(&status[0], MD_DEV_NO_REVERSE); lo[u] = 0; }
            }
            REV[(int64_t)(m0 + u) * n + i] = (uint8_t)lo[u];
        }
        if (m0 == 0) {
            // the row's head as ONE 32-byte record for the crystal pair kernel (k_tersoff_lean): its first four
            // entries, their reverse slots (one byte each) and the row length
            MdRowHead hd;
            hd.j[0] = j[0]; hd.j[1] = j[1]; hd.j[2] = j[2]; hd.j[3] = j[3];
            hd.rev = (unsigned)lo[0] | (unsigned)lo[1] << 8 | (unsigned)lo[2] << 16 | (unsigned)lo[3] << 24;
            hd.nn = nn; hd.pad[0] = hd.pad[1] = 0;
            HEAD[i] = hd;
        }
    }
    if (nn == 0) { MdRowHead hd = {{0, 0, 0, 0}, 0u, 0, {0, 0}}; HEAD[i] = hd; }
}

}  // namespace

int md_launch_reverse(md_neighbors* nl, cudaStream_t s, int check) {
    const int64_t n = nl->n;
    if (n == 0) return MD_OK;
    ProfScope prof(nl, MD_KIND_BUILD, 1, s);
    // after k_search (a build) as a programmatic dependent; after the copies of an import as a normal launch
    if (check) k_reverse<true><<<(unsigned)((n + 127) / 128), 128, 0, s>>>(n, nl->K, nl->NN, nl->NL, nl->REV, nl->d_status, nl->HEAD);
    else MD_CUDA_TRY(md_launch_pdl(k_reverse<false>, dim3((unsigned)((n + 127) / 128)), dim3(128), 0, s, true, n, nl->K, nl->NN,
                                   nl->NL, nl->REV, nl->d_status, nl->HEAD));
    MD_CUDA_TRY(cudaGetLastError());
    MD_CUDA_TRY(cudaMemcpyAsync(nl->h_maxrow, nl->d_status + 1, 2 * sizeof(int), cudaMemcpyDeviceToHost, s));
    MD_CUDA_TRY(cudaEventRecord(nl->ev_list, s));
    nl->maxrow_pending = 1;
    return MD_OK;
}

int md_launch_build(md_neighbors* nl, int64_t n, const double* x, const double* y, const double* z,
                    const double box[3], double r_list, cudaStream_t s) {
    Grid g;
    int64_t ncell = 1;
    for (int a = 0; a < 3; ++a) {
        g.nc[a] = (int)(box[a] / r_list);
        if (g.nc[a] < 3) return MD_ERR_BOX_TOO_SMALL;
        g.inv_cell[a] = (double)g.nc[a] / box[a];
        g.L[a] = box[a];
        g.halfL[a] = 0.5 * box[a];
        ncell *= g.nc[a];
    }
    g.rc2 = r_list * r_list;
    if (ncell + 1 > nl->cell_cap) {                       // grow cell arrays (rare: first build)
        if (ncell + 1 > (int64_t)2000000000) return MD_ERR_ARG;
        MD_CUDA_TRY(cudaStreamSynchronize(s));
        if (nl->cell_count) cudaFree(nl->cell_count);
        if (nl->scan_blocks) cudaFree(nl->scan_blocks);
        nl->cell_count = nullptr; nl->scan_blocks = nullptr; nl->cell_cap = 0;
        const int64_t tiles = (ncell + SCAN_BT * SCAN_IT - 1) / (SCAN_BT * SCAN_IT);
        if (cudaMalloc(&nl->cell_count, sizeof(int32_t) * (ncell + 1)) != cudaSuccess) return MD_ERR_ALLOC;
        if (cudaMalloc(&nl->scan_blocks, sizeof(int32_t) * (tiles + 1)) != cudaSuccess) return MD_ERR_ALLOC;
        nl->cell_cap = ncell + 1;
    }
    nl->n = n;
    if (n == 0) return MD_OK;
    const int ntiles = (int)((ncell + SCAN_BT * SCAN_IT - 1) / (SCAN_BT * SCAN_IT));
    const unsigned gb = (unsigned)((n + 255) / 256);
    {
    ProfScope prof(nl, MD_KIND_BUILD, 6, s);
    MD_CUDA_TRY(cudaMemsetAsync(nl->cell_count, 0, sizeof(int32_t) * (ncell + 1), s));
    // (What a kernel reads from the kernel directly before it is passed without __restrict__, so that it is read
    // by plain coherent loads after the wait, never through the non-coherent path: tile_sums in k_scan_add,
    // cell_start in k_scatter, sorted / sortedf in k_search, NN / NL in k_reverse.)
    // The seven kernels of a build each need everything the one before wrote, so each starts with
    // griddepcontrol.wait and is launched as a programmatic dependent: only the launch latency and ramp of the
    // next kernel overlap with the drain of the previous one (k_bin follows a memset and is launched normally).
    k_bin<<<gb, 256, 0, s>>>(n, x, y, z, g, nl->cell_of, nl->rank_in_cell, nl->cell_count);
    MD_CUDA_TRY(md_launch_pdl(k_scan_local, dim3(ntiles), dim3(SCAN_BT), 0, s, true, nl->cell_count, ncell, nl->scan_blocks));
    MD_CUDA_TRY(md_launch_pdl(k_scan_tiles, dim3(1), dim3(1024), 0, s, true, nl->scan_blocks, ntiles));
    MD_CUDA_TRY(md_launch_pdl(k_scan_add, dim3(ntiles), dim3(SCAN_BT), 0, s, true, nl->cell_count, ncell, nl->scan_blocks, (int32_t)n));
    MD_CUDA_TRY(md_launch_pdl(k_scatter, dim3(gb), dim3(256), 0, s, true, n, x, y, z, nl->cell_of, nl->rank_in_cell,
                              nl->cell_count, nl->sorted, nl->sortedf));
    // FP32 screen.  A coordinate in [0, L) rounds to float within u = 2^-24 Lmax; the shifted reference
    // x +- L carries at most 4u, so each float component differs from the canonical FP64 one by less than
    // 5u (+ 1e-13 of FP64 rounding), and for a candidate near the cut-off |d2_f32 - d2| is below
    // 2 sqrt(3) (r_list + 5u) 5u + 3 (5u)^2 + 2^-22 d2 < 18 (r_list + e) e with e = 6u.  The band
    // [rc2 - m, rc2 + m) with m = 32 (r_list + e) e + 1e-6 rc2 is nearly twice that bound: outside it
    // the float comparison and the FP64 predicate agree; inside it the FP64 predicate is evaluated.
    const double Lmax = fmax(box[0], fmax(box[1], box[2]));
    const double e = 6.0 * Lmax * 5.9604645e-8;
    const double band = 32.0 * (r_list + e) * e + 1e-6 * g.rc2;
    const float rc2_lo = (float)(g.rc2 - band) , rc2_hi = (float)(g.rc2 + band);
    MD_CUDA_TRY(md_launch_pdl(k_search, dim3((unsigned)((n + SEARCH_BT - 1) / SEARCH_BT)), dim3(SEARCH_BT),
                              sizeof(int) * SEARCH_BT * (nl->K + 1), s, true, n, g, nl->sorted, nl->sortedf, nl->cell_count, nl->K,
                              rc2_lo, rc2_hi, nl->NN, nl->NL, nl->d_status));
    }
    MD_CUDA_TRY(cudaGetLastError());
    return md_launch_reverse(nl, s, 0);
}
