// pair_sort.cuh -- front end shared by the loop-structured pair kernels (Tersoff with rows of any length,
// Stillinger-Weber): per-atom screen of the listed neighbours against the force range, and a CTA-local
// reassignment of atoms to threads ordered by their number M of in-range neighbours.
//
// Why.  The pair arithmetic of one atom costs ~M pair terms + M(M-1) triplet terms.  With one thread per atom
// in list order a warp runs to the largest M of its 32 lanes: for the Stillinger-Weber list (16-18 listed,
// 4-12 in range, mean 5.9) that is 2.5x the triplet work actually needed.  After the screen every CTA sorts its
// BT atoms by M (a counting sort on ballots, deterministic: ties keep list order) and thread `tid` takes the
// atom of rank `tid`, so the lanes of a warp have (nearly) the same M, the loops over in-range neighbours have
// warp-uniform trip counts, and no lane idles.  The per-slot data of a thread live in shared-memory columns
// addressed [slot][lane] inside a region owned by its warp and sized by the warp's largest M, so the CTA's
// pool is used by what the atoms need (sum over warps of 32 * M_max), not by the worst case of one atom.
//
// The screen is the only place where "in range" is decided (one helper, explicit roundings, see in_range_d2):
// the decision for (i,j) and (j,i) must agree bit for bit, because atom i pushes P_ij into the slot of row j
// that j's MASK bit says j will read (push layout).
#pragma once
#include "common.cuh"

namespace ps {

// d2 of a listed pair, the same roundings wherever MASK is decided (k_tersoff_lean, the warp-per-atom general path, the
// screen below): dx*dx rounded, then two fused multiply-adds.  x_j - x_i and the minimum-image shift are exact
// negations of each other for (i,j) and (j,i), so both ends compute the same bits.
__device__ __forceinline__ double in_range_d2(double dx, double dy, double dz) {
    return __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
}
__device__ __forceinline__ float in_range_d2(float dx, float dy, float dz) {
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

// Minimum image of a listed pair, coordinates in [0, L).  A pair that needs the +-L shift on some axis has an
// unwrapped |d_a| > L_a/2, hence an unwrapped d2 > (L_min/2)^2; a pair that does not is (for any list worth
// the name) far below that.  So the hot path forms d2 from the unwrapped differences and looks at ONE integer
// compare on its high word (`far`, no FP64-pipe instruction); only when some lane of the warp sees a far pair
// -- warps at the faces of the box, 1 in 10 at 512 000 atoms -- are the three components tested and shifted
// and d2 formed again.  d - 0.0 == d, so the result is the same bits whichever path a warp takes, and the
// shift is an exact negation between (i,j) and (j,i).
struct MinImage {
    double Lx, Ly, Lz;
    int hx, hy, hz;          // high words of L/2
    int far_hi;              // high word of (min L / 2)^2, rounded down: d2 above it may need a shift
    static __device__ __forceinline__ double shift(double d, double L, int hi_half) {
        const int hi = __double2hiint(d);
        const int sL = __double2hiint(L) | (hi & 0x80000000);            // copysign(L, d), high word
        const double s = (hi & 0x7fffffff) > hi_half ? __hiloint2double(sL, __double2loint(L)) : 0.0;
        return d - s;
    }
    __device__ __forceinline__ void wrap(double& dx, double& dy, double& dz) const {
        dx = shift(dx, Lx, hx); dy = shift(dy, Ly, hy); dz = shift(dz, Lz, hz);
    }
    // d2 (arithmetic type T) above which a pair may need the shift; T = float rounds d first, hence the margin
    template <class T> __device__ __forceinline__ bool far(T d2) const {
        return __double2hiint((double)d2) >= far_hi;
    }
};

__device__ __forceinline__ MinImage make_min_image(double lx, double ly, double lz) {
    MinImage m;
    m.Lx = lx; m.Ly = ly; m.Lz = lz;
    m.hx = __double2hiint(0.5 * lx); m.hy = __double2hiint(0.5 * ly); m.hz = __double2hiint(0.5 * lz);
    const double lm = fmin(lx, fmin(ly, lz));
    m.far_hi = __double2hiint(0.2499 * lm * lm) - 1;        // a little below (L_min/2)^2: conservative
    return m;
}

constexpr int MBINS = 33;        // in-range counts 0..32 (a list row has at most 64 entries; > 32 in range: overflow)

template <int BT>
struct SortScratch {
    unsigned long long mask[BT];     // in-range bits over the list row of atom t (tile order)
    unsigned short perm[BT];         // perm[rank] = t
    int atom[BT];                    // atom index of tile entry t (-1: none)
    int cnt[BT / 32][MBINS + 3];     // per warp: atoms with M == b; then exclusive offsets (padded: 36 ints)
    int wmax[BT / 32];               // per warp (after the sort): largest M
};

// Screen: in-range bit mask of atom i over its list row (thread-per-atom, coalesced row reads, U
// neighbours in flight: their list entries first, then their 3 U coordinates).  T is the arithmetic type of the
// force kernel: in FP32 mode r_ij is formed in double, rounded to float, and the float d2 decides (reading
// A10) -- for both ends.  Indices are 32-bit: n * max_neighbors <= 2e9 is checked at md_neighbors_create.
// Force range per pair of elements (multi-element Tersoff): r2[ti * nt + tj] = S_ij^2.  nt = 1: one range.
template <class T> struct RangeTab { int nt; T r2[16]; };

template <class T, int U>
__device__ __forceinline__ unsigned long long
screen_row(unsigned i, unsigned n, int nn, const double* x, const double* y, const double* z,   // plain loads: see k_screen
           const MinImage& mi, const int32_t* __restrict__ NL,
           const RangeTab<T>& rt, const int32_t* __restrict__ types) {
    const int trow = types ? types[i] * rt.nt : 0;
    const double xi = x[i], yi = y[i], zi = z[i];
    unsigned long long mask = 0ull;
    for (int m0 = 0; m0 < nn; m0 += U) {
        int j[U];
        double dx[U], dy[U], dz[U];
        T d2[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const unsigned m = m0 + u < nn ? m0 + u : m0;       // a valid row entry for the idle tail
            j[u] = NL[m * n + i];
        }
#pragma unroll
        for (int u = 0; u < U; ++u) { dx[u] = x[j[u]] - xi; dy[u] = y[j[u]] - yi; dz[u] = z[j[u]] - zi; }
        bool far = false;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            d2[u] = in_range_d2((T)dx[u], (T)dy[u], (T)dz[u]);
            far = far || mi.far(d2[u]);
        }
        if (__any_sync(__activemask(), far)) {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                mi.wrap(dx[u], dy[u], dz[u]);
                d2[u] = in_range_d2((T)dx[u], (T)dy[u], (T)dz[u]);
            }
        }
        unsigned bits = 0u;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const T range2 = types ? rt.r2[trow + types[j[u]]] : rt.r2[0];
            bits |= d2[u] < range2 ? 1u << u : 0u;
        }
        const int left = nn - m0;                                // entries of this chunk that exist
        if (left < U) bits &= (1u << left) - 1u;
        mask |= (unsigned long long)bits << m0;
    }
    return mask;
}

// The screen as a kernel of its own: MASK[i] for every atom.  It is bound by the latency of the two dependent
// loads (list entry -> coordinates), so it runs with small CTAs and few registers at full occupancy instead
// of inside the pair kernel (whose shared-memory pool holds it to 12-16 warps per SM), and it makes every
// MASK known before any pair record is written, which is what the dense record layout needs (dense_slot).
// Bins of atoms by their number M of in-range neighbours: bin 0: M <= b0, bin 1: b0 < M <= b1, bin 2: M > b1.
// The screen appends every atom to the index list of its bin (one atomic per warp and bin; the order inside a
// list is whatever the warps' atomics make it, which is harmless: what is computed for an atom does not depend
// on which thread computes it).  Each bin then gets a kernel specialised for its M.
struct Bins {
    int b0, b1;
    int32_t* list;      // [3][n]
    int32_t* count;     // [4] of this launch: zero on entry
    int32_t* count_next;// [4] of the next launch (the other half of a ping-pong pair): zeroed by this one, whose
                        // wait has seen the last reader of that half finish -- no memset between the kernels
};

template <class T>
__global__ void __launch_bounds__(256, 4)
k_screen(unsigned n, const double* x, const double* y, const double* z,
         double Lx, double Ly, double Lz, const int32_t* __restrict__ NN, const int32_t* __restrict__ NL,
         const __grid_constant__ RangeTab<T> rt,              // indexed in place (a by-value copy lands on the stack)
         const int32_t* __restrict__ types, unsigned long long* __restrict__ MASK, Bins bins) {
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    int bin = -1;
    // Inside md_nve_run: a programmatic dependent of the fused gather that wrote x, y, z (common.cuh,
    // md_launch_pdl); the row length is requested while that kernel drains, the coordinates are read after the
    // wait through plain (non-.nc) loads.
    int nn = i < n ? NN[i] : 0;
    md_grid_wait();
    md_grid_release();
    if (bins.count_next && i < 4) bins.count_next[i] = 0;
    if (i < n) {
        const MinImage mi = make_min_image(Lx, Ly, Lz);
        if (nn > 64) nn = 64;
        const unsigned long long mask = screen_row<T, 4>(i, n, nn, x, y, z, mi, NL, rt, types);
        MASK[i] = mask;
        const int M = __popcll(mask);
        bin = M <= bins.b0 ? 0 : (M <= bins.b1 ? 1 : 2);
    }
    if (!bins.list) return;
    // One atomic per CTA and bin (not per warp: 16 000 warps adding to the same three counters serialise in L2):
    // per-warp counts -> shared memory, warp 0 reserves the CTA's range of each bin, every warp takes its part.
    // The order inside a bin's list is whatever the CTAs' atomics make it, which is harmless: what is computed for an
    // atom does not depend on which thread computes it.
    __shared__ int s_cnt[3][8], s_base[3][8];                // 256 threads = 8 warps
    const unsigned lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    unsigned v[3];
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        v[b] = __ballot_sync(0xffffffffu, bin == b);
        if (lane == 0) s_cnt[b][wid] = __popc(v[b]);
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        const int b = threadIdx.x;
        int tot = 0, off[8];
#pragma unroll
        for (int w = 0; w < 8; ++w) { off[w] = tot; tot += s_cnt[b][w]; }
        const int base = tot ? atomicAdd(&bins.count[b], tot) : 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) s_base[b][w] = base + off[w];
    }
    __syncthreads();
    if (bin >= 0) bins.list[(size_t)bin * n + s_base[bin][wid] + __popc(v[bin] & ((1u << lane) - 1u))] = (int)i;
}

// Dense record layout: the record of pair (i -> j) goes to the slot of row j that counts the in-range entries
// of row j before i's position rev, so the gather of j reads popc(MASK_j) consecutive slots (coalesced over
// atoms) instead of the in-range ones scattered over a 16-18-entry row.
__device__ __forceinline__ unsigned dense_slot(unsigned long long mask_j, int rev) {
    return (unsigned)__popcll(mask_j & ((1ull << rev) - 1ull));
}

// A load the compiler may not sink to its first use (prefetch of the next chunk's data into registers).
__device__ __forceinline__ double ld_early(const double* p) {
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ int ld_early(const int32_t* p) {
    int v;
    asm volatile("ld.global.nc.s32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ int ld_early(const uint8_t* p) {
    int v;
    asm volatile("ld.global.nc.u8 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ unsigned long long ld_early(const unsigned long long* p) {   // MASK: written by the kernel
    unsigned long long v;                                                               // before (k_screen): no .nc
    asm volatile("ld.global.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}

// Sort the CTA's atoms by M = popc(mask) (ascending, ties in tile order).  On return thread `tid` owns tile
// atom *t (its mask in *mask), its warp's column region starts at pool slot *base and holds *M_w slots per
// lane (M_w = largest M in the warp, clamped so that the region fits `pool_slots`; a clamp latches
// MD_DEV_INRANGE_OVERFLOW and the caller drops the pairs beyond *M_w).  Atoms with t >= na (tile tail) carry
// mask 0 and sort to the front with M = 0.  Uses four __syncthreads().
template <int BT, class SS>
__device__ __forceinline__ void
sort_by_count(SS& s, unsigned long long my_mask, int pool_slots, int* __restrict__ status,
              int* t_out, unsigned long long* mask_out, int* base_out, int* Mw_out) {
    constexpr int NW = BT / 32;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    int M = __popcll(my_mask);
    if (M > MBINS - 1) { atomicOr(&status[0], MD_DEV_INRANGE_OVERFLOW); M = MBINS - 1; }
    s.mask[tid] = my_mask;
    // per-warp histogram on ballots: lane b keeps the count of bin b (bins 32.. fold into lane 0's second word)
    // (only the bins between the warp's smallest and largest M can be occupied)
    int mine = 0, mine32 = 0;
    unsigned same = 0u;
    const int blo = __reduce_min_sync(0xffffffffu, M), bhi = __reduce_max_sync(0xffffffffu, M);
#pragma unroll 1
    for (int b = blo; b <= bhi; ++b) {
        const unsigned v = __ballot_sync(0xffffffffu, M == b);
        if (b < 32) { if (lane == b) mine = __popc(v); } else { if (lane == 0) mine32 = __popc(v); }
        if (M == b) same = v;
    }
    s.cnt[wid][lane] = mine;
    if (lane == 0) s.cnt[wid][32] = mine32;
    __syncthreads();
    // warp 0: exclusive offsets, bin-major then warp-major (the order of the sorted sequence)
    if (wid == 0) {
        int run = 0;
#pragma unroll 1
        for (int b0 = 0; b0 < MBINS; b0 += 32) {
            const int b = b0 + lane;
            int c[NW], tot = 0;
#pragma unroll
            for (int w = 0; w < NW; ++w) { c[w] = b < MBINS ? s.cnt[w][b] : 0; tot += c[w]; }
            int inc = tot;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, inc, d);
                if (lane >= d) inc += v;
            }
            int off = run + inc - tot;
            if (b < MBINS) {
#pragma unroll
                for (int w = 0; w < NW; ++w) { s.cnt[w][b] = off; off += c[w]; }
            }
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
    }
    __syncthreads();
    const int rank = s.cnt[wid][M] + __popc(same & ((1u << lane) - 1u));
    s.perm[rank] = (unsigned short)tid;
    __syncthreads();
    const int t = s.perm[tid];
    const unsigned long long mk = s.mask[t];
    const int Mt = min(__popcll(mk), MBINS - 1);
    const int wmax = __reduce_max_sync(0xffffffffu, Mt);
    if (lane == 0) s.wmax[wid] = wmax;
    __syncthreads();
    int base = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) base += w < wid ? 32 * s.wmax[w] : 0;
    int Mw = wmax;
    if (base + 32 * Mw > pool_slots) {                       // pool exhausted: keep what fits, flag it
        if (lane == 0) atomicOr(&status[0], MD_DEV_INRANGE_OVERFLOW);
        Mw = base < pool_slots ? (pool_slots - base) / 32 : 0;
    }
    *t_out = t; *mask_out = mk; *base_out = base; *Mw_out = Mw;
}

// The same sort for a tile of 2 * BT atoms and BT threads (scratch: SortScratch<2 * BT>; thread `tid` brings the masks
// of tile entries tid and BT + tid).  The sorted sequence is cut into 2 * BT / 32 blocks of 32 ranks; warp w takes
// block w in round 0 and block 2 NW - 1 - w in round 1.  With one block per warp the warp that holds the largest
// counts decides when the CTA is done (cost grows as M^2 in the Tersoff loop code: the other warps idled a third of
// the time at the next tile's barrier); a small block plus a large one per warp evens that out, and between the two
// rounds no CTA barrier is needed: the column region of a warp (sized by the larger of its two blocks) is its own.
// Returns per round r: tile entry t[r], its mask and the warp's column region (base[r], M_w[r]); *sync_between says
// whether the CTA must meet at a barrier between the rounds (see below).
template <int BT, class SS>
__device__ __forceinline__ void
sort_by_count_x2(SS& s, const unsigned long long (&my_mask)[2], int pool_slots, int* __restrict__ status,
                 int (&t_out)[2], unsigned long long (&mask_out)[2], int (&base_out)[2], int (&Mw_out)[2],
                 bool* sync_between) {
    constexpr int NW = BT / 32;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    int M[2];
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        M[r] = __popcll(my_mask[r]);
        if (M[r] > MBINS - 1) { atomicOr(&status[0], MD_DEV_INRANGE_OVERFLOW); M[r] = MBINS - 1; }
        s.mask[r * BT + tid] = my_mask[r];
    }
    // per-warp histogram over its 64 entries; `before[r]` = entries of the warp that precede this one inside its bin
    int mine = 0, mine32 = 0, before[2] = {0, 0};
    const int blo = __reduce_min_sync(0xffffffffu, min(M[0], M[1])), bhi = __reduce_max_sync(0xffffffffu, max(M[0], M[1]));
    const unsigned below = (1u << lane) - 1u;
#pragma unroll 1
    for (int b = blo; b <= bhi; ++b) {
        const unsigned v0 = __ballot_sync(0xffffffffu, M[0] == b), v1 = __ballot_sync(0xffffffffu, M[1] == b);
        const int c = __popc(v0) + __popc(v1);
        if (b < 32) { if (lane == b) mine = c; } else { if (lane == 0) mine32 = c; }
        if (M[0] == b) before[0] = __popc(v0 & below);
        if (M[1] == b) before[1] = __popc(v0) + __popc(v1 & below);
    }
    s.cnt[wid][lane] = mine;
    if (lane == 0) s.cnt[wid][32] = mine32;
    __syncthreads();
    if (wid == 0) {                                          // exclusive offsets, bin-major then warp-major
        int run = 0;
#pragma unroll 1
        for (int b0 = 0; b0 < MBINS; b0 += 32) {
            const int b = b0 + lane;
            int c[NW], tot = 0;
#pragma unroll
            for (int w = 0; w < NW; ++w) { c[w] = b < MBINS ? s.cnt[w][b] : 0; tot += c[w]; }
            int inc = tot;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, inc, d);
                if (lane >= d) inc += v;
            }
            int off = run + inc - tot;
            if (b < MBINS) {
#pragma unroll
                for (int w = 0; w < NW; ++w) { s.cnt[w][b] = off; off += c[w]; }
            }
            run += __shfl_sync(0xffffffffu, inc, 31);
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 2; ++r) s.perm[s.cnt[wid][M[r]] + before[r]] = (unsigned short)(r * BT + tid);
    __syncthreads();
    // largest count of every block (warp w looks at blocks w and 2 NW - 1 - w)
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        const int block = r == 0 ? wid : 2 * NW - 1 - wid;
        const int m = min(__popcll(s.mask[s.perm[block * 32 + lane]]), MBINS - 1);
        const int wm = __reduce_max_sync(0xffffffffu, m);
        if (lane == 0) s.wmax[block] = wm;
    }
    __syncthreads();
    // The blocks are in ascending order of M, so the four large ones run side by side in the balanced assignment
    // and the pool has to hold them together.  If it cannot (hot or strongly disordered inputs), the tile runs as
    // {two largest, two smallest blocks}, CTA barrier, {the four in the middle}, with the pool divided anew for
    // each round: about the demand of two tiles of BT atoms.  The choice is the same for every thread of the CTA.
    int top = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) top += s.wmax[2 * NW - 1 - w];
    const bool balanced = 32 * top <= pool_slots;
    *sync_between = !balanced;
#pragma unroll
    for (int r = 0; r < 2; ++r) {
        auto block_of = [&](int w) {
            if (balanced) return r == 0 ? w : 2 * NW - 1 - w;
            return r == 0 ? (w < NW / 2 ? 2 * NW - 1 - w : NW - 1 - w) : NW / 2 + w;
        };
        auto need_of = [&](int w) { return balanced ? s.wmax[2 * NW - 1 - w] : s.wmax[block_of(w)]; };
        int base = 0;
#pragma unroll
        for (int w = 0; w < NW; ++w) base += w < wid ? 32 * need_of(w) : 0;
        int Mw = need_of(wid);
        if (base + 32 * Mw > pool_slots) {                   // pool exhausted: keep what fits, flag it
            if (lane == 0) atomicOr(&status[0], MD_DEV_INRANGE_OVERFLOW);
            Mw = base < pool_slots ? (pool_slots - base) / 32 : 0;
        }
        t_out[r] = s.perm[block_of(wid) * 32 + lane];
        mask_out[r] = s.mask[t_out[r]];
        base_out[r] = base; Mw_out[r] = Mw;
    }
}

}  // namespace ps
