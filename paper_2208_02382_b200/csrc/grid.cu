// S4-S7: particle-grid kernels -- CIC deposit and trilinear gather + kick (+ adjacent drifts).
//
// Canonical index/weights (R11), identical expression on every path so that only the summation
// order of the deposit differs from the definition:
//   u = (q - lo) * inv_d   (one rounded subtract, one rounded multiply; explicit _rn intrinsics so
//                           that nvcc can never contract zscale*t - lo into an FMA)
//   i = floor(u), w1 = u - i (exact), w0 = 1 - w1 ; node weight (wx*wy)*wz.
// Inside iff 0 <= i <= n-2 on all axes, tested as (u >= 0 && u < n-1) so NaN is outside (R13).
#include "bt_internal.h"
#include "grid_dev.cuh"
#include "bulk_copy.cuh"

#include <math_constants.h>
#include <stdlib.h>

namespace bt {

// ---- S5 deposit, mode 0: one particle per thread, (ORDER+1)^3 global fp64 reductions (RED.E.ADD.F64) ----------
template <int ORDER>
__global__ void __launch_bounds__(256) deposit_atomic_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                                             const double *__restrict__ t, long long n, GridDev g,
                                                             double qw, double zscale, double *__restrict__ rho) {
    constexpr int NW = ORDER + 1;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride) {
        Cic c;
        if (!shape_locate<ORDER>(g, x[p], y[p], t[p], zscale, c)) continue;
        double w[NW * NW * NW];
        node_weights<ORDER>(c, qw, w);
        double *base = rho + ((long long)c.k * g.ny + c.j) * g.nx + c.i;
#pragma unroll
        for (int dz = 0; dz < NW; ++dz)
#pragma unroll
            for (int dy = 0; dy < NW; ++dy)
#pragma unroll
                for (int dx = 0; dx < NW; ++dx) atomicAdd(base + ((long long)dz * g.ny + dy) * g.nx + dx, w[(dz * NW + dy) * NW + dx]);
    }
}

// ---- per-lane runs of R consecutive particles: 256-bit streaming access --------------------------------
// A lane owns R consecutive particles of the storage order (R = 4 or 8), i.e. 32*R/4 bytes per array = whole
// 32-byte sectors: every LDG.256 / STG.256 of a warp touches 32 distinct, fully used sectors.
__device__ __forceinline__ void ld256(const double *p, double &a, double &b, double &c, double &d) {
    asm volatile("ld.global.cs.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
// VEC: p0 + R <= n and 32-byte aligned arrays guaranteed by the caller; else guarded scalar loads with `fill`.
template <int R, bool VEC>
__device__ __forceinline__ void load_run(const double *__restrict__ q, long long p0, long long n, double fill, double (&v)[R]) {
    if (VEC && p0 + R <= n) {
#pragma unroll
        for (int r = 0; r < R; r += 4) ld256(q + p0 + r, v[r], v[r + 1], v[r + 2], v[r + 3]);
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = (p0 + r < n) ? q[p0 + r] : fill;
    }
}
// ---- run flush: the node sums of one stencil position -> (ORDER+1)^3 RED.E.ADD.F64 ------------------------------
template <int NW>
__device__ __forceinline__ void flush_cell(double *__restrict__ rho, int key, const double (&acc)[NW * NW * NW], int nx, long long nxy) {
    if (key < 0) return;
    double *plane = rho + key;  // key = linear index of the lowest node of the stencil
#pragma unroll
    for (int dz = 0; dz < NW; ++dz, plane += nxy) {
        double *row = plane;
#pragma unroll
        for (int dy = 0; dy < NW; ++dy, row += nx)
#pragma unroll
            for (int dx = 0; dx < NW; ++dx) atomicAdd(row + dx, acc[(dz * NW + dy) * NW + dx]);
    }
}

// ---- S4+S5 deposit, mode 1 (default): block-local cell binning in shared memory + run accumulation ------------
// A block of NT threads owns chunks of NT*R consecutive particles (storage order); NT = 256, R = 8 measured best on B200
// (10-step mean on 4A: 256x8 131 us, 128x8 134, 256x4 134, 512x4 140, 512x8 152, 1024x4 164: block barriers over many
// warps cost more than the extra warps hide).  The particles of a chunk are binned by cell
// INSIDE the block (counting sort over the chunk's bounding box of cells: one shared-memory integer atomic per run of
// same-cell particles of a thread gives count and rank at once, a block scan gives the offsets), so that afterwards every thread walks R
// entries of the cell-ordered list and sums same-cell particles in registers; a run is flushed with 8 RED.E.ADD.F64
// when the cell changes, and the lanes' open runs are merged by a segmented shuffle reduction first.  Global
// reductions per chunk = 8 x (distinct cells + warp seams) instead of 8 x particles, for ANY order in which a chunk
// is spatially compact (bt_beam_sort_by_cell once, then many drift/kick steps: particles wander a few cells, the
// chunk's box stays small).  Consecutive lanes flush x-adjacent cells, so the REDs of one instruction share
// 32-byte sectors (measured: 0.6-0.8 SM-cycles per RED lane against 1.55 for scattered sectors).
// A chunk whose box exceeds kBinCap cells (unsorted input, the thin tails of the bunch) bins what falls into a fixed 16^3
// box around its first inside particle and sends the rest straight to RED.  Weights are the canonical R11 / R16
// expression on every path.
constexpr int kBinCap = 4096;  // cells of the chunk's bounding box that the shared histogram can hold

// Runs hold UNSCALED weight sums (wx*wy)*wz and are scaled by q_weight once, at the flush.
template <int NW>
__device__ __forceinline__ void flush_cell_scaled(double *__restrict__ rho, int key, const double (&acc)[NW * NW * NW], double qw, int nx,
                                                  long long nxy) {
    if (key < 0) return;
    double *plane = rho + key;
#pragma unroll
    for (int dz = 0; dz < NW; ++dz, plane += nxy) {
        double *row = plane;
#pragma unroll
        for (int dy = 0; dy < NW; ++dy, row += nx)
#pragma unroll
            for (int dx = 0; dx < NW; ++dx) atomicAdd(row + dx, __dmul_rn(qw, acc[(dz * NW + dy) * NW + dx]));
    }
}
// merge the lanes' open runs (segmented suffix reduction over CONTIGUOUS equal keys), heads flush
template <int NW>
__device__ __forceinline__ void merge_and_flush_scaled(double *__restrict__ rho, int cur, double (&acc)[NW * NW * NW], double qw, int nx,
                                                       long long nxy) {
    const int lane = threadIdx.x & 31;
    const int prev = __shfl_up_sync(0xffffffffu, cur, 1);
    const bool head = (lane == 0) || (prev != cur);
    const unsigned heads = __ballot_sync(0xffffffffu, head);
    if (heads != 0xffffffffu) {  // warp-uniform: some run spans lanes
        const unsigned above = (lane == 31) ? 0u : (heads >> (lane + 1));
        const int end = above ? lane + __ffs(above) - 1 : 31;  // last lane of this lane's run
        const int span = __reduce_max_sync(0xffffffffu, end - lane);
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            if (d > span) break;  // warp-uniform
            const bool take = lane + d <= end;
#pragma unroll
            for (int k = 0; k < NW * NW * NW; ++k) {
                const double o = __shfl_down_sync(0xffffffffu, acc[k], d);
                if (take) acc[k] += o;
            }
        }
    }
    if (head) flush_cell_scaled<NW>(rho, cur, acc, qw, nx, nxy);
}

// The same merge for lanes that also carry a HEAD run: the first run of a lane's entries, which may be the continuation of
// the run the previous lanes ended with (a lane's first key change used to flush that part on its own: with runs of ~10
// particles and 8 entries per lane nearly every lane has such a seam, and the flushed runs were half as long as the cells'
// populations allow -- profiles/r02_summary.md).  nrun = runs seen by the lane; nrun >= 2: (head_key, head) is the first,
// (cur, acc) the last; nrun == 1: the single run is (cur, acc); nrun == 0: cur = -1.  Tails are merged over contiguous
// equal keys as before; the head lane of each merged block additionally takes the head run of the lane that follows the
// block when its key matches, so every run of the chunk's cell-ordered list reaches rho exactly once.
template <int NW>
__device__ __forceinline__ void merge_heads_and_flush_scaled(double *__restrict__ rho, int cur, double (&acc)[NW * NW * NW], int nrun, int head_key,
                                                             const double (&head)[NW * NW * NW], double qw, int nx, long long nxy) {
    constexpr unsigned kFull = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int prev = __shfl_up_sync(kFull, cur, 1);
    const bool first = (lane == 0) || (prev != cur);
    const unsigned firsts = __ballot_sync(kFull, first);
    const unsigned above = (lane == 31) ? 0u : (firsts >> (lane + 1));
    const int end = above ? lane + __ffs(above) - 1 : 31;  // last lane of the block of equal tail keys this lane is in
    if (firsts != kFull) {                                  // warp-uniform: some block spans lanes
        const int span = __reduce_max_sync(kFull, end - lane);
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            if (d > span) break;  // warp-uniform
            const bool take = lane + d <= end;
#pragma unroll
            for (int k = 0; k < NW * NW * NW; ++k) {
                const double o = __shfl_down_sync(kFull, acc[k], d);
                if (take) acc[k] += o;
            }
        }
    }
    // head runs: donated to the block that ends in the previous lane when the keys match, else flushed by their own lane
    const int hk = nrun >= 2 ? head_key : -2;
    // (only a lane that STARTS a block can donate: the block before it then ends at lane - 1 and looks at this lane; a lane
    // inside a block whose head happens to carry the block's key -- aliased bins: runs X Y X -- flushes the head itself)
    const bool donated = lane > 0 && first && hk == prev;   // prev = tail key of lane - 1 = key of the block ending there
    const int donor = (end + 1) & 31;
    const int donor_hk = __shfl_sync(kFull, hk, donor);
    const bool take_head = first && end < 31 && donor_hk == cur && cur >= 0;
    if (__any_sync(kFull, take_head)) {
#pragma unroll
        for (int k = 0; k < NW * NW * NW; ++k) {
            const double o = __shfl_sync(kFull, head[k], donor);
            if (take_head) acc[k] += o;
        }
    }
    if (first) flush_cell_scaled<NW>(rho, cur, acc, qw, nx, nxy);
    if (nrun >= 2 && !donated) flush_cell_scaled<NW>(rho, head_key, head, qw, nx, nxy);
}

template <int NT, int R>
struct BinSmem {
    static constexpr int CH = NT * R;
    static constexpr int PAD = CH + CH / 8;  // one pad slot per 8 entries: a thread's R-entry walk is conflict-free
    alignas(16) int hist[kBinCap + 16];      // bins [0, ncell) = cells of the box, bin kBinCap = particles that are not binned
    int box[2][8];  // imin, jmin, kmin, imax, jmax, kmax, lowest thread holding an inside particle; double-buffered by chunk parity
    int anchor[4];
    int warp_tot[NT / 32];
    int key[PAD];
    double w1[3][PAD];
};

// register budget per thread: 128 for 8 particles per thread or 27 run accumulators, else 80 (64 in blocks of >= 512 threads)
template <int NT, int R, int ORDER>
constexpr int kBinRegs = (R >= 8 || ORDER > 1) ? 128 : (NT >= 512 ? 64 : 80);
template <int NT, int R, int ORDER>
constexpr int kBinMinBlocks = (65536 / NT) / kBinRegs<NT, R, ORDER> > 0 ? (65536 / NT) / kBinRegs<NT, R, ORDER> : 1;

template <int NT, int R, bool VEC, int ORDER>
__global__ void __launch_bounds__(NT, kBinMinBlocks<NT, R, ORDER>) deposit_binned_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                                                   const double *__restrict__ t, long long n, GridDev g, double qw,
                                                                   double zscale, double *__restrict__ rho) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    BinSmem<NT, R> &sm = *reinterpret_cast<BinSmem<NT, R> *>(smem_raw);
    constexpr int CH = BinSmem<NT, R>::CH;
    constexpr int BPT = kBinCap / NT;  // histogram bins per thread in the scan (a multiple of 4)
    constexpr int NW = ORDER + 1, NN = NW * NW * NW;
    constexpr int kBig = 0x7fffffff;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const long long nxy = (long long)g.nx * g.ny;
    const long long nchunks = (n + CH - 1) / CH;
    if (tid < 8) sm.box[0][tid] = (tid >= 3 && tid < 6) ? -1 : kBig;
    for (int s4 = tid * 4; s4 < kBinCap + 16; s4 += NT * 4) *reinterpret_cast<int4 *>(&sm.hist[s4]) = make_int4(0, 0, 0, 0);
    __syncthreads();
    int parity = 0;
    for (long long ch = blockIdx.x; ch < nchunks; ch += gridDim.x, parity ^= 1) {
        int *box = sm.box[parity];
        const long long p0 = ch * CH + (long long)tid * R;
        double qx[R], qy[R], qt[R];
        load_run<R, VEC>(x, p0, n, CUDART_NAN, qx);  // NaN => outside => contributes nothing
        load_run<R, VEC>(y, p0, n, 0.0, qy);
        load_run<R, VEC>(t, p0, n, 0.0, qt);
        Cic c[R];
        bool in[R];
        int lo_i = kBig, lo_j = kBig, lo_k = kBig, hi_i = -1, hi_j = -1, hi_k = -1;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            in[r] = shape_locate<ORDER>(g, qx[r], qy[r], qt[r], zscale, c[r]);
            if (in[r]) {
                lo_i = min(lo_i, c[r].i), hi_i = max(hi_i, c[r].i);
                lo_j = min(lo_j, c[r].j), hi_j = max(hi_j, c[r].j);
                lo_k = min(lo_k, c[r].k), hi_k = max(hi_k, c[r].k);
            }
        }
        const int first_tid = __reduce_min_sync(0xffffffffu, hi_i >= 0 ? tid : kBig);
        lo_i = __reduce_min_sync(0xffffffffu, lo_i), hi_i = __reduce_max_sync(0xffffffffu, hi_i);
        lo_j = __reduce_min_sync(0xffffffffu, lo_j), hi_j = __reduce_max_sync(0xffffffffu, hi_j);
        lo_k = __reduce_min_sync(0xffffffffu, lo_k), hi_k = __reduce_max_sync(0xffffffffu, hi_k);
        if (lane == 0 && hi_i >= 0) {
            atomicMin(&box[0], lo_i), atomicMin(&box[1], lo_j), atomicMin(&box[2], lo_k);
            atomicMax(&box[3], hi_i), atomicMax(&box[4], hi_j), atomicMax(&box[5], hi_k);
            atomicMin(&box[6], first_tid);
        }
        __syncthreads();  // (1) box complete
        if (tid < 8) sm.box[parity ^ 1][tid] = (tid >= 3 && tid < 6) ? -1 : kBig;  // next chunk's box (its readers passed barrier 2 of the previous chunk)
        if (box[3] < 0) {  // no particle of this chunk is inside the grid (block-uniform)
            __syncthreads();  // orders the re-initialisation above before the next chunk's box atomics
            continue;
        }
        int i0 = box[0], j0 = box[1], k0 = box[2];
        int bx = box[3] - i0 + 1, by = box[4] - j0 + 1, bz = box[5] - k0 + 1;
        // A chunk that is not spatially compact (unsorted input, the thin tails): bin what falls into a fixed 16^3 box
        // around the first inside particle -- this catches a cold core even in unsorted order -- the rest goes direct.
        const bool big = (long long)bx * by * bz > kBinCap;
        if (big) {  // block-uniform; compact chunks skip this barrier (the histogram was cleared during the previous walk)
            if (tid == box[6]) {
#pragma unroll
                for (int r = R - 1; r >= 0; --r)
                    if (in[r]) sm.anchor[0] = c[r].i, sm.anchor[1] = c[r].j, sm.anchor[2] = c[r].k;
            }
            __syncthreads();  // (2) anchor published
            i0 = sm.anchor[0] - 8, j0 = sm.anchor[1] - 8, k0 = sm.anchor[2] - 8;
            bx = by = bz = 16;
        }
        int lc[R], rank[R];
        if (big) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const unsigned li = (unsigned)(c[r].i - i0), lj = (unsigned)(c[r].j - j0), lk = (unsigned)(c[r].k - k0);
                const bool binned = in[r] && li < 16u && lj < 16u && lk < 16u;
                if (in[r] && !binned) {
                    double w[NN];
                    node_weights<ORDER>(c[r], qw, w);
                    flush_cell<NW>(rho, (c[r].k * g.ny + c[r].j) * g.nx + c[r].i, w, g.nx, nxy);
                }
                in[r] = binned;
                lc[r] = binned ? (int)((lk * 16u + lj) * 16u + li) : kBinCap;
            }
        } else {
#pragma unroll
            for (int r = 0; r < R; ++r) lc[r] = in[r] ? ((c[r].k - k0) * by + (c[r].j - j0)) * bx + (c[r].i - i0) : kBinCap;
        }
        // count and rank within the cell in one pass.  A thread's R particles are consecutive in storage, so in a cell-sorted
        // chunk they mostly share a bin: one atomic per RUN of equal bins (same-address shared atomics serialise, measured
        // ~1 SM-cycle each).
        {
            int len[R];
            len[R - 1] = 1;
#pragma unroll
            for (int r = R - 2; r >= 0; --r) len[r] = (lc[r] == lc[r + 1]) ? len[r + 1] + 1 : 1;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const bool head = (r == 0) || (lc[r] != lc[r - 1]);
                if (head) rank[r] = atomicAdd(&sm.hist[lc[r]], len[r]);
                else rank[r] = rank[r - 1] + 1;
            }
        }
        __syncthreads();  // (3) histogram complete
        // exclusive scan of hist[0..ncell) in place: BPT consecutive bins per thread (LDS.128), warp scan, block carry;
        // the spill bin hist[kBinCap] is not part of it
        int total = 0;
        {
            // a thread owns the bins {4 NT q + 4 tid + 0..3}: 128-bit accesses contiguous across the warp (conflict-free);
            // the scan order (thread-major) is a fixed permutation of the bins, which is all a counting sort needs
            const int ncell = big ? kBinCap : bx * by * bz;  // bins >= ncell are empty: skip their quarter of the table (block-uniform)
            int4 v[BPT / 4];
            int s = 0;
#pragma unroll
            for (int q = 0; q < BPT / 4; ++q) {
                v[q] = make_int4(0, 0, 0, 0);
                if (4 * NT * q < ncell) v[q] = *reinterpret_cast<const int4 *>(&sm.hist[4 * NT * q + 4 * tid]);
                s += v[q].x + v[q].y + v[q].z + v[q].w;
            }
            int incl = s;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += o;
            }
            if (lane == 31) sm.warp_tot[wid] = incl;
            __syncthreads();  // (4)
            int off = incl - s;
#pragma unroll
            for (int w = 0; w < NT / 32; ++w) {
                const int wt = sm.warp_tot[w];
                off += (w < wid) ? wt : 0;
                total += wt;
            }
#pragma unroll
            for (int q = 0; q < BPT / 4; ++q) {
                int4 o;
                o.x = off, off += v[q].x;
                o.y = off, off += v[q].y;
                o.z = off, off += v[q].z;
                o.w = off, off += v[q].w;
                if (4 * NT * q < ncell) *reinterpret_cast<int4 *>(&sm.hist[4 * NT * q + 4 * tid]) = o;
            }
        }
        __syncthreads();  // (5) offsets ready; total = number of binned particles
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (in[r]) {
                const int e = sm.hist[lc[r]] + rank[r];
                const int slot = e + (e >> 3);
                sm.key[slot] = (c[r].k * g.ny + c[r].j) * g.nx + c[r].i;
                sm.w1[0][slot] = c[r].wx1;
                sm.w1[1][slot] = c[r].wy1;
                sm.w1[2][slot] = c[r].wz1;
            }
        __syncthreads();  // (6) cell-ordered entry list complete
        // the histogram is dead from here on: clear it for the next chunk (whose first access follows its barrier (1))
        for (int s4 = tid * 4; s4 < kBinCap + 16; s4 += NT * 4) *reinterpret_cast<int4 *>(&sm.hist[s4]) = make_int4(0, 0, 0, 0);
        {
            int cur = -1;
            double acc[NN];
#pragma unroll
            for (int d = 0; d < NN; ++d) acc[d] = 0.0;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int e = tid * R + r;
                if (e >= total) break;
                const int slot = e + (e >> 3);
                Cic cc;
                cc.i = cc.j = cc.k = 0;
                cc.wx1 = sm.w1[0][slot], cc.wy1 = sm.w1[1][slot], cc.wz1 = sm.w1[2][slot];
                double w[NN];
                node_weights_unscaled<ORDER>(cc, w);
                const int key = sm.key[slot];
                if (key != cur) {  // a new run: the finished one leaves (scaled by q_weight), the accumulators restart from zero
                    flush_cell_scaled<NW>(rho, cur, acc, qw, g.nx, nxy);
                    cur = key;
#pragma unroll
                    for (int d = 0; d < NN; ++d) acc[d] = 0.0;
                }
#pragma unroll
                for (int d = 0; d < NN; ++d) acc[d] += w[d];
            }
            merge_and_flush_scaled<NW>(rho, cur, acc, qw, g.nx, nxy);
        }
        // no barrier here: the next chunk touches hist / entries only after its barrier (1), which every thread of this
        // chunk's walk must reach first
    }
}

// ---- S4+S5 deposit, mode 1 (default): WARP-private cell binning + run accumulation ---------------------------------------
// Same idea as deposit_binned_kernel (bin the chunk's particles by cell in shared memory, then sum same-cell particles in
// registers and flush a run with (ORDER+1)^3 reductions), re-cut so that nothing in it needs a block barrier:
//   * a WARP owns a chunk of 32*R consecutive particles (R = 8: 256 particles) and its own slice of shared memory; warps
//     only ever __syncwarp, so the warps of an SM drift apart and cover each other's latencies (the block-wide version
//     ran 5-6 __syncthreads per 2048 particles at 16 resident warps: 41 % issue utilisation, profiles/r01b_summary.md);
//   * no bounding box: the bin is the low three bits of each cell index, (k&7, j&7, i&7) -> 512 bins.  It is injective
//     whenever the chunk spans <= 8 cells per axis, which is what a cell-sorted chunk does for many steps (the dense
//     part of the bunch); where it is not (thin tails, unsorted input) aliased cells merely interleave inside a bin and
//     shorten the runs -- the walk compares full node keys, so the result never depends on the hash;
//   * the located particles (node key, the three weight fractions) are parked in shared memory in LOAD order right
//     away and only a 2-byte slot index is sorted, so registers hold R bins + R ranks across the scan instead of R
//     located particles (round 1: 128 registers, 16 warps per SM; here <= 96 and 20);
//   * runs accumulate the UNSCALED weights (wx*wy)*wz and are scaled by q_weight once per flush
//     (q*(w1+w2+...) instead of q*w1+q*w2+...: one rounding of difference, far inside R15's 1e-12).
constexpr int kWarpBins = 512;

template <int R>
struct WarpBinSmem {
    static constexpr int CW = 32 * R;        // particles per warp chunk
    static constexpr int CWP = 32 * (R + 1); // padded slots: lane l, particle r -> l*(R+1) + r (64-bit accesses: 2 wavefronts)
    alignas(16) int hist[kWarpBins];
    alignas(16) unsigned short idx[CW];      // cell-ordered list of slots
    int key[CWP];
    double w1[3][CWP];
};

template <int R, int ORDER>
constexpr int kWarpDepBlocks = ORDER == 1 ? (R >= 8 ? 5 : 6) : 4;  // 128-thread blocks per SM (shared memory and registers)

template <int R, bool VEC, int ORDER>
__global__ void __launch_bounds__(128, kWarpDepBlocks<R, ORDER>) deposit_warp_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                                                                   const double *__restrict__ t, long long n, GridDev g,
                                                                                   double qw, double zscale, double *__restrict__ rho) {
    extern __shared__ __align__(16) unsigned char wsmem_raw[];
    constexpr int CW = WarpBinSmem<R>::CW;
    constexpr int BPL = kWarpBins / 32;  // bins per lane in the scan
    constexpr int NW = ORDER + 1, NN = NW * NW * NW;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    WarpBinSmem<R> &sm = reinterpret_cast<WarpBinSmem<R> *>(wsmem_raw)[wid];
    const long long nxy = (long long)g.nx * g.ny;
    const long long nchunks = (n + CW - 1) / CW;
    const long long warps_total = (long long)gridDim.x * (blockDim.x >> 5);
    // a lane owns the bins {128 q + 4 lane + 0..3}: its 128-bit accesses are contiguous across the warp (conflict-free)
#pragma unroll
    for (int q = 0; q < BPL / 4; ++q) *reinterpret_cast<int4 *>(&sm.hist[128 * q + 4 * lane]) = make_int4(0, 0, 0, 0);
    __syncwarp();
    for (long long ch = (long long)blockIdx.x * (blockDim.x >> 5) + wid; ch < nchunks; ch += warps_total) {
        // ---- phase 1: load, locate, park in shared memory, count per bin (one atomic per run of equal bins) ----
        int bin[R], rank[R];
        {
            // sub-batches of 8 particles per lane keep the loaded coordinates at 24 doubles whatever R is
            constexpr int SB = R < 8 ? R : 8;
#pragma unroll
            for (int h = 0; h < R / SB; ++h) {
                const long long p0 = ch * CW + (long long)lane * R + h * SB;
                double qx[SB], qy[SB], qt[SB];
                load_run<SB, VEC>(x, p0, n, CUDART_NAN, qx);  // NaN => outside => contributes nothing
                load_run<SB, VEC>(y, p0, n, 0.0, qy);
                load_run<SB, VEC>(t, p0, n, 0.0, qt);
#pragma unroll
                for (int r = 0; r < SB; ++r) {
                    Cic c;
                    const bool in = shape_locate<ORDER>(g, qx[r], qy[r], qt[r], zscale, c);
                    const int slot = lane * (R + 1) + h * SB + r;
                    sm.key[slot] = (c.k * g.ny + c.j) * g.nx + c.i;
                    sm.w1[0][slot] = c.wx1;
                    sm.w1[1][slot] = c.wy1;
                    sm.w1[2][slot] = c.wz1;
                    bin[h * SB + r] = in ? (((c.k & 7) << 6) | ((c.j & 7) << 3) | (c.i & 7)) : -1;
                }
            }
            int len[R];
            len[R - 1] = 1;
#pragma unroll
            for (int r = R - 2; r >= 0; --r) len[r] = (bin[r] == bin[r + 1]) ? len[r + 1] + 1 : 1;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const bool head = (r == 0) || (bin[r] != bin[r - 1]);
                if (head) rank[r] = bin[r] >= 0 ? atomicAdd(&sm.hist[bin[r]], len[r]) : 0;
                else rank[r] = rank[r - 1] + 1;
            }
        }
        __syncwarp();
        // ---- phase 2: exclusive scan of the 512 counters (16 per lane, lane-major order), in place ----
        int total;
        {
            int4 v[BPL / 4];
            int s = 0;
#pragma unroll
            for (int q = 0; q < BPL / 4; ++q) {
                v[q] = *reinterpret_cast<const int4 *>(&sm.hist[128 * q + 4 * lane]);
                s += v[q].x + v[q].y + v[q].z + v[q].w;
            }
            int incl = s;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += o;
            }
            total = __shfl_sync(0xffffffffu, incl, 31);
            int off = incl - s;
#pragma unroll
            for (int q = 0; q < BPL / 4; ++q) {
                int4 o;
                o.x = off, off += v[q].x;
                o.y = off, off += v[q].y;
                o.z = off, off += v[q].z;
                o.w = off, off += v[q].w;
                *reinterpret_cast<int4 *>(&sm.hist[128 * q + 4 * lane]) = o;
            }
        }
        __syncwarp();
        // ---- phase 3: the cell-ordered list of slots ----
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (bin[r] >= 0) sm.idx[sm.hist[bin[r]] + rank[r]] = (unsigned short)(lane * (R + 1) + r);
        __syncwarp();
        // the counters are dead: clear them for the next chunk
#pragma unroll
        for (int q = 0; q < BPL / 4; ++q) *reinterpret_cast<int4 *>(&sm.hist[128 * q + 4 * lane]) = make_int4(0, 0, 0, 0);
        // ---- phase 4: every lane walks R consecutive entries of the list, sums same-cell particles, merges, flushes ----
        {
            unsigned short my[R];
            static_assert(R == 4 || R == 8, "idx is read as one 8- or 16-byte word per lane");
            if (R == 8) {
                const uint4 u = *reinterpret_cast<const uint4 *>(&sm.idx[lane * R]);
                my[0] = u.x & 0xffff, my[1] = u.x >> 16, my[2] = u.y & 0xffff, my[3] = u.y >> 16;
                my[4 % R] = u.z & 0xffff, my[5 % R] = u.z >> 16, my[6 % R] = u.w & 0xffff, my[7 % R] = u.w >> 16;
            } else {
                const uint2 u = *reinterpret_cast<const uint2 *>(&sm.idx[lane * R]);
                my[0] = u.x & 0xffff, my[1] = u.x >> 16, my[2] = u.y & 0xffff, my[3] = u.y >> 16;
            }
            // HEADS: the lane's first run is kept and merged across lanes too (order 1: 8 more accumulators; at order 2 the 27
            // would not fit the register file, there a lane's first key change flushes as in round 1)
            constexpr bool HEADS = ORDER == 1;
            int cur = -1, nrun = 0, head_key = -1;
            double acc[NN], head[HEADS ? NN : 1];
#pragma unroll
            for (int d = 0; d < NN; ++d) acc[d] = 0.0;
#pragma unroll
            for (int d = 0; d < (HEADS ? NN : 1); ++d) head[d] = 0.0;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (lane * R + r >= total) break;
                const int slot = my[r];
                Cic cc;
                cc.i = cc.j = cc.k = 0;
                cc.wx1 = sm.w1[0][slot], cc.wy1 = sm.w1[1][slot], cc.wz1 = sm.w1[2][slot];
                double w[NN];
                node_weights_unscaled<ORDER>(cc, w);
                const int key = sm.key[slot];
                if (key != cur) {  // a new run starts
                    if (HEADS && nrun == 1) {  // the lane's first run ends: kept as the head run (merged across lanes below)
                        head_key = cur;
#pragma unroll
                        for (int d = 0; d < (HEADS ? NN : 1); ++d) head[d] = acc[d];
                    } else {                   // a run that began and ended inside this lane's entries (no-op for cur = -1)
                        flush_cell_scaled<NW>(rho, cur, acc, qw, g.nx, nxy);
                    }
                    ++nrun;
                    cur = key;
#pragma unroll
                    for (int d = 0; d < NN; ++d) acc[d] = 0.0;
                }
#pragma unroll
                for (int d = 0; d < NN; ++d) acc[d] += w[d];
            }
            if constexpr (HEADS) merge_heads_and_flush_scaled<NW>(rho, cur, acc, nrun, head_key, head, qw, g.nx, nxy);
            else merge_and_flush_scaled<NW>(rho, cur, acc, qw, g.nx, nxy);
        }
        __syncwarp();  // the next chunk overwrites the parked particles and the list
    }
}

// cudaFuncSetAttribute + the occupancy query, once per (kernel instantiation, device)
template <auto kernel>
static int blocks_per_sm(int threads, int smem, int device, int *out) {
    static std::atomic<int> cache[kMaxDevices];  // 0 = not queried yet; one array per kernel instantiation
    if (device < 0 || device >= kMaxDevices) return fail(BT_ERR_UNSUPPORTED, "device index too large");
    int v = cache[device].load(std::memory_order_acquire);
    if (v == 0) {
        BT_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        BT_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&v, kernel, threads, smem));
        if (v < 1) v = 1;
        cache[device].store(v, std::memory_order_release);
    }
    *out = v;
    return BT_OK;
}

template <int NT, int R, bool VEC, int ORDER>
static int launch_deposit_binned(Beam *b, Grid *g, const GridDev &gd, double q_weight, double zscale) {
    const int smem = (int)sizeof(BinSmem<NT, R>);
    const long long nchunks = (b->n + BinSmem<NT, R>::CH - 1) / BinSmem<NT, R>::CH;
    int per_sm = 1;
    const int qrc = blocks_per_sm<deposit_binned_kernel<NT, R, VEC, ORDER>>(NT, smem, b->device, &per_sm);
    if (qrc != BT_OK) return qrc;
    long long blocks = (long long)b->num_sms * (per_sm > 0 ? per_sm : 1);
    if (blocks > nchunks) blocks = nchunks;
    deposit_binned_kernel<NT, R, VEC, ORDER><<<(int)blocks, NT, smem, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight,
                                                                                     zscale, g->rho);
    return BT_OK;
}

template <int R, bool VEC, int ORDER>
static int launch_deposit_warp(Beam *b, Grid *g, const GridDev &gd, double q_weight, double zscale) {
    constexpr int kWarps = 4;  // 128-thread blocks
    const int smem = (int)sizeof(WarpBinSmem<R>) * kWarps;
    const long long nchunks = (b->n + WarpBinSmem<R>::CW - 1) / WarpBinSmem<R>::CW;
    int per_sm = 1;
    const int qrc = blocks_per_sm<deposit_warp_kernel<R, VEC, ORDER>>(32 * kWarps, smem, b->device, &per_sm);
    if (qrc != BT_OK) return qrc;
    long long blocks = (long long)b->num_sms * per_sm;
    if (blocks > (nchunks + kWarps - 1) / kWarps) blocks = (nchunks + kWarps - 1) / kWarps;
    deposit_warp_kernel<R, VEC, ORDER><<<(int)blocks, 32 * kWarps, smem, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight, zscale,
                                                                                     g->rho);
    return BT_OK;
}

template <int ORDER>
static int launch_deposit_order(Beam *b, Grid *g, const GridDev &gd, double q_weight, double zscale) {
    // knob deposit_mode: 0 = one particle per thread, (ORDER+1)^3 reductions each (baseline, kept for measurements);
    // 1 (default) = warp-private cell binning, 8 particles per lane (at order 2 as well: longer lane segments mean fewer
    // separately flushed head runs of 27 reductions each -- 4A 322 -> 284 us, 4B 298 -> 196 us against 4 per lane);
    // 2 = warp-private binning with 4 particles per lane; 3 = round 1's block-wide binning (2048-particle chunks,
    // 1024 at order 2)
    const int mode = knob(KNOB_DEPOSIT_MODE, 1);
    if (mode == 0) {
        const int block = 256;
        long long blocks = (b->n + block - 1) / block;
        const long long cap = (long long)b->num_sms * 16;
        if (blocks > cap) blocks = cap;
        deposit_atomic_kernel<ORDER><<<(int)blocks, block, 0, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight, zscale, g->rho);
        return BT_OK;
    }
    if (mode == 3) {
        if constexpr (ORDER == 1)
            return b->aligned32 ? launch_deposit_binned<256, 8, true, ORDER>(b, g, gd, q_weight, zscale)
                                : launch_deposit_binned<256, 8, false, ORDER>(b, g, gd, q_weight, zscale);
        return b->aligned32 ? launch_deposit_binned<256, 4, true, ORDER>(b, g, gd, q_weight, zscale)
                            : launch_deposit_binned<256, 4, false, ORDER>(b, g, gd, q_weight, zscale);
    }
    if (mode != 2)
        return b->aligned32 ? launch_deposit_warp<8, true, ORDER>(b, g, gd, q_weight, zscale)
                            : launch_deposit_warp<8, false, ORDER>(b, g, gd, q_weight, zscale);
    return b->aligned32 ? launch_deposit_warp<4, true, ORDER>(b, g, gd, q_weight, zscale)
                        : launch_deposit_warp<4, false, ORDER>(b, g, gd, q_weight, zscale);
}

int launch_deposit(Beam *b, Grid *g, double q_weight, double zscale) {
    const GridDev gd = make_grid_dev(*g);
    const int rc = g->order == 2 ? launch_deposit_order<2>(b, g, gd, q_weight, zscale) : launch_deposit_order<1>(b, g, gd, q_weight, zscale);
    if (rc != BT_OK) return rc;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_deposit_cic launch: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(1);
    return BT_OK;
}

// ---- field re-layout: (Ex,Ey,Ez) planar -> 32-byte node records (Ex,Ey,Ez,0) ---------------------
// One node = one 32-byte sector = one 256-bit load; the 8 nodes of a cell are 4 x 64 contiguous bytes.
__global__ void __launch_bounds__(256) field_pack_kernel(const double *__restrict__ ex, const double *__restrict__ ey,
                                                         const double *__restrict__ ez, long long nn, double4 *__restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nn) out[i] = make_double4(ex[i], ey[i], ez[i], 0.0);
}

int launch_field_pack(Grid *g, const double *ex, const double *ey, const double *ez, cudaStream_t s) {
    const int block = 256;
    const long long blocks = (g->nn + block - 1) / block;
    field_pack_kernel<<<(int)blocks, block, 0, s>>>(ex, ey, ez, g->nn, reinterpret_cast<double4 *>(g->field));
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_grid_set_field launch: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(1);
    return BT_OK;
}

// ---- S6/S7 gather + kick with the adjacent drifts fused -----------------------------------------
struct GatherArgs {
    double *q[6];
    const double *field;  // 4 doubles per node
    long long n;
    GridDev g;
    double coef[3];
    double zscale;
    double hb, tcb, ha, tca;  // drift before / after: x += h px, y += h py, t += tc pt
};

__device__ __forceinline__ void ld_node(const double *f, double &ex, double &ey, double &ez) {
    asm volatile("{ .reg .f64 pad; ld.global.nc.v4.f64 {%0,%1,%2,pad}, [%3]; }" : "=d"(ex), "=d"(ey), "=d"(ez) : "l"(f));
}

// One particle through [drift] -> gather over the (ORDER+1)^3 stencil -> kick -> [drift]; shared by both gather kernels.
// Gather order dz, dy, dx (R12); weight (wx*wy)*wz with explicit roundings, field accumulated with FMAs.
template <int ORDER>
__device__ __forceinline__ void gather_kick_one(const GatherArgs &a, double &x, double &px, double &y, double &py, double &t, double &pt) {
    constexpr int NW = ORDER + 1;
    // R4 drift before the kick (a zero-length drift is no map at all: positions stay bit-identical, also for non-finite momenta)
    if (a.hb != 0.0 || a.tcb != 0.0) {
        x = fma(a.hb, px, x);
        y = fma(a.hb, py, y);
        t = fma(a.tcb, pt, t);
    }
    Cic c;
    if (shape_locate<ORDER>(a.g, x, y, t, a.zscale, c)) {
        const double *base = a.field + 4 * (((long long)c.k * a.g.ny + c.j) * a.g.nx + c.i);
        double wx[NW], wy[NW], wz[NW];
        axis_weights<ORDER>(c.wx1, wx);
        axis_weights<ORDER>(c.wy1, wy);
        axis_weights<ORDER>(c.wz1, wz);
        double ex = 0.0, ey = 0.0, ez = 0.0;
        // one z-plane of the stencil at a time (loads of a plane are independent of its FMAs); summation order dz, dy, dx
#pragma unroll
        for (int dz = 0; dz < NW; ++dz) {
            double fx[NW * NW], fy[NW * NW], fz[NW * NW];
#pragma unroll
            for (int dy = 0; dy < NW; ++dy)
#pragma unroll
                for (int dx = 0; dx < NW; ++dx)
                    ld_node(base + 4 * (((long long)dz * a.g.ny + dy) * a.g.nx + dx), fx[dy * NW + dx], fy[dy * NW + dx], fz[dy * NW + dx]);
#pragma unroll
            for (int dy = 0; dy < NW; ++dy)
#pragma unroll
                for (int dx = 0; dx < NW; ++dx) {
                    const double w = __dmul_rn(__dmul_rn(wx[dx], wy[dy]), wz[dz]);
                    ex = fma(w, fx[dy * NW + dx], ex);
                    ey = fma(w, fy[dy * NW + dx], ey);
                    ez = fma(w, fz[dy * NW + dx], ez);
                }
        }
        px = fma(a.coef[0], ex, px);
        py = fma(a.coef[1], ey, py);
        pt = fma(a.coef[2], ez, pt);
    }
    // R4 drift after the kick
    if (a.ha != 0.0 || a.tca != 0.0) {
        x = fma(a.ha, px, x);
        y = fma(a.ha, py, y);
        t = fma(a.tca, pt, t);
    }
}

template <int ORDER>
__global__ void __launch_bounds__(256) gather_kick_kernel(const __grid_constant__ GatherArgs a) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < a.n; p += stride) {
        double x = __ldcs(a.q[0] + p), px = __ldcs(a.q[1] + p), y = __ldcs(a.q[2] + p);
        double py = __ldcs(a.q[3] + p), t = __ldcs(a.q[4] + p), pt = __ldcs(a.q[5] + p);
        gather_kick_one<ORDER>(a, x, px, y, py, t, pt);
        __stcs(a.q[0] + p, x);
        __stcs(a.q[1] + p, px);
        __stcs(a.q[2] + p, y);
        __stcs(a.q[3] + p, py);
        __stcs(a.q[4] + p, t);
        __stcs(a.q[5] + p, pt);
    }
}

// ---- S6/S7, streaming pipeline: particle chunks ride the copy engine, the field comes through L1 ------------------
// A persistent block cycles through kGpStages shared-memory stages of CH particles x 6 coordinates:
//   chunk k+2 is being loaded (cp.async.bulk global->shared, completion on an mbarrier),
//   chunk k   is updated IN PLACE in shared memory by the threads (drift, 8-node gather, kick, drift),
//   chunk k-1 is being stored (cp.async.bulk shared->global).
// Particle I/O therefore needs no registers and no warp ever waits on a particle load: ~96 KiB per SM are in flight in
// each direction, independent of occupancy.  Threads address a stage with stride blockDim (conflict-free LDS/STS).  The
// 8 node records (32 B each, one LDG.E.ENL2.256 through the read-only path) of a particle's cell are L1/L2 hits: a chunk
// of cell-ordered particles covers a few hundred cells.  Same per-particle arithmetic as gather_kick_kernel.
// Full chunks only; the ragged tail of the bunch (< CH particles) is done by gather_kick_kernel.
constexpr int kGpStages = 3;

template <int CH>
struct GpSmem {
    alignas(128) double q[kGpStages][6][CH];
    alignas(8) uint64_t full[kGpStages];
};

template <int NT, int R, int ORDER>
__global__ void __launch_bounds__(NT) gather_kick_pipe_kernel(const __grid_constant__ GatherArgs a, long long nchunks, int store_positions) {
    constexpr int CH = NT * R;
    constexpr uint32_t kArrBytes = CH * sizeof(double);
    extern __shared__ __align__(128) unsigned char gp_smem_raw[];
    GpSmem<CH> &sm = *reinterpret_cast<GpSmem<CH> *>(gp_smem_raw);
    const int tid = threadIdx.x;
    const auto issue_load = [&](long long ch, int s) {
        mbar_expect_tx(&sm.full[s], 6 * kArrBytes);
#pragma unroll
        for (int c = 0; c < 6; ++c) bulk_g2s(sm.q[s][c], a.q[c] + ch * CH, kArrBytes, &sm.full[s]);
    };
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kGpStages; ++s) mbar_init(&sm.full[s], 1);
        mbar_init_fence();
        if ((long long)blockIdx.x < nchunks) issue_load(blockIdx.x, 0);
        if ((long long)blockIdx.x + gridDim.x < nchunks) issue_load((long long)blockIdx.x + gridDim.x, 1);
    }
    __syncthreads();
    int s = 0;
    uint32_t parity = 0;
    for (long long ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
        mbar_wait(&sm.full[s], parity);
        double(*q)[CH] = sm.q[s];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int e = r * NT + tid;
            double x = q[0][e], px = q[1][e], y = q[2][e], py = q[3][e], t = q[4][e], pt = q[5][e];
            gather_kick_one<ORDER>(a, x, px, y, py, t, pt);
            q[0][e] = x, q[1][e] = px, q[2][e] = y, q[3][e] = py, q[4][e] = t, q[5][e] = pt;
        }
        fence_proxy_async_smem();  // this thread's shared-memory writes -> visible to the copy engine
        __syncthreads();
        if (tid == 0) {
#pragma unroll
            for (int c = 0; c < 6; ++c)
                if (store_positions || (c & 1)) bulk_s2g(a.q[c] + ch * CH, sm.q[s][c], kArrBytes);
            bulk_commit();
            // the stage two chunks ahead is the one stored in the previous iteration: wait until that store has read it
            const long long nxt = ch + 2LL * gridDim.x;
            if (nxt < nchunks) {
                bulk_wait_read<1>();
                issue_load(nxt, (s + 2) % kGpStages);
            }
        }
        if (++s == kGpStages) s = 0, parity ^= 1;
    }
    if (tid == 0) bulk_wait_all<0>();  // shared memory must outlive the last stores
}

template <int NT, int R, int ORDER>
static int launch_gather_pipe(Beam *b, const GatherArgs &a0) {
    constexpr int CH = NT * R;
    const int smem = (int)sizeof(GpSmem<CH>);
    const long long nchunks = b->n / CH;
    if (nchunks > 0) {
        int per_sm = 1;
        const int qrc = blocks_per_sm<gather_kick_pipe_kernel<NT, R, ORDER>>(NT, smem, b->device, &per_sm);
        if (qrc != BT_OK) return qrc;
        long long blocks = (long long)b->num_sms * (per_sm > 0 ? per_sm : 1);
        if (blocks > nchunks) blocks = nchunks;
        const int store_positions = (a0.hb != 0.0 || a0.ha != 0.0 || a0.tcb != 0.0 || a0.tca != 0.0) ? 1 : 0;
        gather_kick_pipe_kernel<NT, R, ORDER><<<(int)blocks, NT, smem, b->stream>>>(a0, nchunks, store_positions);
    }
    const long long done = nchunks * CH;
    if (done < b->n) {  // ragged tail: one particle per thread
        GatherArgs t = a0;
        for (int c = 0; c < 6; ++c) t.q[c] = a0.q[c] + done;
        t.n = b->n - done;
        gather_kick_kernel<ORDER><<<(int)((t.n + 255) / 256), 256, 0, b->stream>>>(t);
    }
    return BT_OK;
}

// ---- S6/S7, streaming pipeline with the chunk's field tile staged in shared memory ---------------------------------
// B:north_star's gather: "stages the field tile in shared memory".  Same particle pipeline as gather_kick_pipe_kernel
// (bulk copies in, in-place update, bulk copies out); in addition the block finds the bounding box of its chunk's stencils
// (warp REDUX + shared atomics), loads the box's node records ONCE, coalesced row by row, into three planar shared arrays
// (Ex, Ey, Ez: 24 bytes per node, no pad) and every particle then reads its (ORDER+1)^3 nodes with LDS.64.  Why it pays:
// the L1 -> register return path delivers ~64 B/clk/SM and every lane needs its own copy of every node record
// ((ORDER+1)^3 x 32 B per particle: 864 B at order 2, where the L1 path is flat at 0.23 of the HBM bound even when all
// lanes read the same records), while shared memory returns 128 B/clk and lanes that share a node are served by one
// broadcast wavefront.  A chunk whose box exceeds kTileCap nodes (unsorted input, thin tails) reads through L1 as before.
constexpr int kTileCap = 1280;  // nodes: 30 KiB of shared memory; a drifted 256-particle chunk of configs[4] needs ~1200 at order 2

constexpr int kGtBins = 512;  // regrouping bins: the low three bits of each index of the stencil's base node

template <int CH>
struct GtSmem {
    alignas(128) double q[kGpStages][6][CH];
    alignas(16) double tile[3][kTileCap];
    alignas(16) int hist[kGtBins + 8];  // [kGtBins] = particles outside the grid
    unsigned short idx[CH];             // REGROUP: slot of the particle a thread works on (cell order)
    int warp_tot[8];
    int box[2][8];
    alignas(8) uint64_t full[kGpStages];
};

// REGROUP (default at order 2): the threads of a block work on the chunk's particles in CELL order instead of storage
// order -- a counting sort of the 256 slots by the stencil's base cell (shared histogram, block scan, 2-byte slot list),
// results written back IN PLACE, so nothing moves in HBM and no id travels.  Why: the 27 x 3 LDS.64 per particle are what
// loads the L1 data pipe (76 % of peak, 3.4 wavefronts per LDS.64 with the lanes of a warp spread over ~12 cells after a few
// steps of wandering); lanes that sit in the same cell read the same words (one broadcast wavefront), lanes in x-adjacent
// cells read adjacent words (no bank conflict), so a warp of cell-ordered particles needs 1-2 wavefronts per load.
template <int ORDER, bool REGROUP>
__global__ void __launch_bounds__(256, 3) gather_kick_tile_kernel(const __grid_constant__ GatherArgs a, long long nchunks, int store_positions) {
    constexpr int NT = 256, CH = 256, NW = ORDER + 1;
    constexpr uint32_t kArrBytes = CH * sizeof(double);
    constexpr int kBig = 0x7fffffff;
    extern __shared__ __align__(128) unsigned char gt_smem_raw[];
    GtSmem<CH> &sm = *reinterpret_cast<GtSmem<CH> *>(gt_smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const auto issue_load = [&](long long ch, int s) {
        mbar_expect_tx(&sm.full[s], 6 * kArrBytes);
#pragma unroll
        for (int c = 0; c < 6; ++c) bulk_g2s(sm.q[s][c], a.q[c] + ch * CH, kArrBytes, &sm.full[s]);
    };
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kGpStages; ++s) mbar_init(&sm.full[s], 1);
        mbar_init_fence();
        if ((long long)blockIdx.x < nchunks) issue_load(blockIdx.x, 0);
        if ((long long)blockIdx.x + gridDim.x < nchunks) issue_load((long long)blockIdx.x + gridDim.x, 1);
    }
    if (tid < 8) sm.box[0][tid] = (tid >= 3 && tid < 6) ? -1 : kBig;
    if (REGROUP) {
        sm.hist[2 * tid] = 0, sm.hist[2 * tid + 1] = 0;
        if (tid < 8) sm.hist[kGtBins + tid] = 0;
    }
    __syncthreads();
    int s = 0, bpar = 0;
    uint32_t parity = 0;
    for (long long ch = blockIdx.x; ch < nchunks; ch += gridDim.x, bpar ^= 1) {
        mbar_wait(&sm.full[s], parity);
        double(*q)[CH] = sm.q[s];
        int *box = sm.box[bpar];
        double x = q[0][tid], px = q[1][tid], y = q[2][tid], py = q[3][tid], t = q[4][tid], pt = q[5][tid];
        // R4 drift before the kick (skipped when zero-length, as in gather_kick_one)
        if (a.hb != 0.0 || a.tcb != 0.0) {
            x = fma(a.hb, px, x);
            y = fma(a.hb, py, y);
            t = fma(a.tcb, pt, t);
        }
        Cic c;
        bool in = shape_locate<ORDER>(a.g, x, y, t, a.zscale, c);
        {   // bounding box of the chunk's stencil bases
            int lo_i = in ? c.i : kBig, lo_j = in ? c.j : kBig, lo_k = in ? c.k : kBig;
            int hi_i = in ? c.i : -1, hi_j = in ? c.j : -1, hi_k = in ? c.k : -1;
            lo_i = __reduce_min_sync(0xffffffffu, lo_i), hi_i = __reduce_max_sync(0xffffffffu, hi_i);
            lo_j = __reduce_min_sync(0xffffffffu, lo_j), hi_j = __reduce_max_sync(0xffffffffu, hi_j);
            lo_k = __reduce_min_sync(0xffffffffu, lo_k), hi_k = __reduce_max_sync(0xffffffffu, hi_k);
            if (lane == 0 && hi_i >= 0) {
                atomicMin(&box[0], lo_i), atomicMin(&box[1], lo_j), atomicMin(&box[2], lo_k);
                atomicMax(&box[3], hi_i), atomicMax(&box[4], hi_j), atomicMax(&box[5], hi_k);
            }
        }
        int bin = 0, rank = 0;
        if (REGROUP) {
            bin = in ? (((c.k & 7) << 6) | ((c.j & 7) << 3) | (c.i & 7)) : kGtBins;
            rank = atomicAdd(&sm.hist[bin], 1);
        }
        __syncthreads();  // (1) box (and histogram) complete
        if (tid < 8) sm.box[bpar ^ 1][tid] = (tid >= 3 && tid < 6) ? -1 : kBig;  // next chunk's box
        const int i0 = box[0], j0 = box[1], k0 = box[2];
        const int tx = box[3] - i0 + NW, ty = box[4] - j0 + NW, tz = box[5] - k0 + NW;  // nodes per axis of the tile
        const bool staged = box[3] >= 0 && (long long)tx * ty * tz <= kTileCap;  // block-uniform
        if (staged) {
            // rows of tx consecutive node records (x fastest): 16 lanes per row, 16 rows per sweep
            const int rows = ty * tz;
            for (int row = tid >> 4; row < rows; row += NT / 16) {
                const int iz = row / ty, iy = row - iz * ty;
                const double *src = a.field + 4 * ((((long long)(k0 + iz)) * a.g.ny + (j0 + iy)) * a.g.nx + i0);
                for (int xx = tid & 15; xx < tx; xx += 16) {
                    double fx, fy, fz;
                    ld_node(src + 4 * xx, fx, fy, fz);
                    const int idx = row * tx + xx;
                    sm.tile[0][idx] = fx, sm.tile[1][idx] = fy, sm.tile[2][idx] = fz;
                }
            }
        }
        int slot = tid;  // the particle this thread works on
        if (REGROUP) {
            // exclusive scan of the 512 counters (two per thread), the slot list, then every thread picks up the particle
            // at ITS position of the cell order and locates it again (cheaper than parking the located particles)
            const int v0 = sm.hist[2 * tid], v1 = sm.hist[2 * tid + 1];
            const int sum = v0 + v1;
            int incl = sum;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += o;
            }
            if (lane == 31) sm.warp_tot[wid] = incl;
            __syncthreads();  // (2) warp totals (and every thread has read its two counters)
            int off = incl - sum, inside = 0;
#pragma unroll
            for (int w = 0; w < NT / 32; ++w) {
                const int wt = sm.warp_tot[w];
                off += (w < wid) ? wt : 0;
                inside += wt;
            }
            sm.hist[2 * tid] = off, sm.hist[2 * tid + 1] = off + v0;
            __syncthreads();  // (3) offsets ready
            const int pos = (bin < kGtBins ? sm.hist[bin] : inside) + rank;
            sm.idx[pos] = (unsigned short)tid;
            __syncthreads();  // (4) slot list complete (and the tile is staged)
            sm.hist[2 * tid] = 0, sm.hist[2 * tid + 1] = 0;  // for the next chunk (its first atomic follows barrier (5))
            if (tid == 0) sm.hist[kGtBins] = 0;
            slot = sm.idx[tid];
            x = q[0][slot], px = q[1][slot], y = q[2][slot], py = q[3][slot], t = q[4][slot], pt = q[5][slot];
            if (a.hb != 0.0 || a.tcb != 0.0) {
                x = fma(a.hb, px, x);
                y = fma(a.hb, py, y);
                t = fma(a.tcb, pt, t);
            }
            in = shape_locate<ORDER>(a.g, x, y, t, a.zscale, c);
        } else {
            __syncthreads();  // (2) tile staged
        }
        if (in) {
            double wx[NW], wy[NW], wz[NW];
            axis_weights<ORDER>(c.wx1, wx);
            axis_weights<ORDER>(c.wy1, wy);
            axis_weights<ORDER>(c.wz1, wz);
            double ex = 0.0, ey = 0.0, ez = 0.0;
            if (staged) {
                const int base = ((c.k - k0) * ty + (c.j - j0)) * tx + (c.i - i0);
#pragma unroll
                for (int dz = 0; dz < NW; ++dz)
#pragma unroll
                    for (int dy = 0; dy < NW; ++dy)
#pragma unroll
                        for (int dx = 0; dx < NW; ++dx) {
                            const double w = __dmul_rn(__dmul_rn(wx[dx], wy[dy]), wz[dz]);
                            const int idx = base + (dz * ty + dy) * tx + dx;
                            ex = fma(w, sm.tile[0][idx], ex);
                            ey = fma(w, sm.tile[1][idx], ey);
                            ez = fma(w, sm.tile[2][idx], ez);
                        }
            } else {
                const double *gbase = a.field + 4 * (((long long)c.k * a.g.ny + c.j) * a.g.nx + c.i);
#pragma unroll
                for (int dz = 0; dz < NW; ++dz)
#pragma unroll
                    for (int dy = 0; dy < NW; ++dy)
#pragma unroll
                        for (int dx = 0; dx < NW; ++dx) {
                            const double w = __dmul_rn(__dmul_rn(wx[dx], wy[dy]), wz[dz]);
                            double fx, fy, fz;
                            ld_node(gbase + 4 * (((long long)dz * a.g.ny + dy) * a.g.nx + dx), fx, fy, fz);
                            ex = fma(w, fx, ex);
                            ey = fma(w, fy, ey);
                            ez = fma(w, fz, ez);
                        }
            }
            px = fma(a.coef[0], ex, px);
            py = fma(a.coef[1], ey, py);
            pt = fma(a.coef[2], ez, pt);
        }
        // R4 drift after the kick
        if (a.ha != 0.0 || a.tca != 0.0) {
            x = fma(a.ha, px, x);
            y = fma(a.ha, py, y);
            t = fma(a.tca, pt, t);
        }
        q[0][slot] = x, q[1][slot] = px, q[2][slot] = y, q[3][slot] = py, q[4][slot] = t, q[5][slot] = pt;
        fence_proxy_async_smem();  // this thread's shared-memory writes -> visible to the copy engine
        __syncthreads();           // (last) stage complete; everyone is done with the tile
        if (tid == 0) {
#pragma unroll
            for (int cc = 0; cc < 6; ++cc)
                if (store_positions || (cc & 1)) bulk_s2g(a.q[cc] + ch * CH, sm.q[s][cc], kArrBytes);
            bulk_commit();
            const long long nxt = ch + 2LL * gridDim.x;
            if (nxt < nchunks) {
                bulk_wait_read<1>();
                issue_load(nxt, (s + 2) % kGpStages);
            }
        }
        if (++s == kGpStages) s = 0, parity ^= 1;
    }
    if (tid == 0) bulk_wait_all<0>();  // shared memory must outlive the last stores
}

template <int ORDER, bool REGROUP>
static int launch_gather_tile(Beam *b, const GatherArgs &a0) {
    constexpr int CH = 256;
    const int smem = (int)sizeof(GtSmem<CH>);
    const long long nchunks = b->n / CH;
    if (nchunks > 0) {
        int per_sm = 1;
        const int qrc = blocks_per_sm<gather_kick_tile_kernel<ORDER, REGROUP>>(256, smem, b->device, &per_sm);
        if (qrc != BT_OK) return qrc;
        long long blocks = (long long)b->num_sms * (per_sm > 0 ? per_sm : 1);
        if (blocks > nchunks) blocks = nchunks;
        const int store_positions = (a0.hb != 0.0 || a0.ha != 0.0 || a0.tcb != 0.0 || a0.tca != 0.0) ? 1 : 0;
        gather_kick_tile_kernel<ORDER, REGROUP><<<(int)blocks, 256, smem, b->stream>>>(a0, nchunks, store_positions);
    }
    const long long done = nchunks * CH;
    if (done < b->n) {  // ragged tail: one particle per thread
        GatherArgs t = a0;
        for (int c = 0; c < 6; ++c) t.q[c] = a0.q[c] + done;
        t.n = b->n - done;
        gather_kick_kernel<ORDER><<<(int)((t.n + 255) / 256), 256, 0, b->stream>>>(t);
    }
    return BT_OK;
}

template <int ORDER>
static int launch_gather_order(Beam *b, const GatherArgs &a) {
    // knob gather_mode: 0 = one particle per thread, everything through registers (also the path for arrays that are not
    // 16-byte aligned); 1 (default) = streaming pipeline, 256-particle chunks, field through L1 (order 1) or staged in shared
    // memory (order 2); 2 / 3 = L1 pipeline with 512 / 128-particle chunks; 4 = shared-memory tile at any order (threads work in cell order at
    // order 2); 5 = the tile with the other regrouping choice
    const int mode = knob(KNOB_GATHER_MODE, 1);
    // field tile staged in shared memory: the default at order 2 (measured 4A 10-step mean 547 -> 477 us, 4B 529 -> 430 us),
    // selectable at order 1 (knob gather_mode = 4), where the L1 path is faster (181 against 216 us)
    // only on cell-sorted beams: in the caller's order no chunk's box fits the tile and the pass through L1 is faster from
    // the plain pipeline (order 2, unsorted kick: 0.79 against 1.51 ms)
    if ((mode == 4 || (mode == 1 && ORDER == 2 && b->permuted)) && b->aligned16) return launch_gather_tile<ORDER, ORDER == 2>(b, a);
    if (mode == 5 && b->aligned16) return launch_gather_tile<ORDER, ORDER != 2>(b, a);  // the other regrouping choice, for A/B runs
    if (mode >= 1 && b->aligned16)
        return mode == 2 ? launch_gather_pipe<512, 1, ORDER>(b, a) : mode == 3 ? launch_gather_pipe<128, 1, ORDER>(b, a) : launch_gather_pipe<256, 1, ORDER>(b, a);
    const int block = 256;
    long long blocks = (b->n + block - 1) / block;
    const long long cap = (long long)b->num_sms * 16;
    if (blocks > cap) blocks = cap;
    gather_kick_kernel<ORDER><<<(int)blocks, block, 0, b->stream>>>(a);
    return BT_OK;
}

int launch_gather_kick(Beam *b, const Grid *g, const double coef[3], double zscale, double h_before, double tc_before,
                       double h_after, double tc_after) {
    GatherArgs a;
    for (int c = 0; c < 6; ++c) a.q[c] = b->q[c];
    a.field = g->field;
    a.n = b->n;
    a.g = make_grid_dev(*g);
    for (int c = 0; c < 3; ++c) a.coef[c] = coef[c];
    a.zscale = zscale;
    a.hb = h_before;
    a.tcb = tc_before;
    a.ha = h_after;
    a.tca = tc_after;
    const int rc = g->order == 2 ? launch_gather_order<2>(b, a) : launch_gather_order<1>(b, a);
    if (rc != BT_OK) return rc;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_gather_kick launch: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(1);
    return BT_OK;
}

}  // namespace bt
