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

#include <math_constants.h>
#include <stdlib.h>

namespace bt {

// ---- S5 deposit, mode 0: one particle per thread, 8 global fp64 reductions (RED.E.ADD.F64) --------
__global__ void __launch_bounds__(256) deposit_atomic_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                                             const double *__restrict__ t, long long n, GridDev g,
                                                             double qw, double zscale, double *__restrict__ rho) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += stride) {
        Cic c;
        if (!cic_locate(g, x[p], y[p], t[p], zscale, c)) continue;
        const double wx[2] = {__dsub_rn(1.0, c.wx1), c.wx1};
        const double wy[2] = {__dsub_rn(1.0, c.wy1), c.wy1};
        const double wz[2] = {__dsub_rn(1.0, c.wz1), c.wz1};
        double *base = rho + ((long long)c.k * g.ny + c.j) * g.nx + c.i;
#pragma unroll
        for (int dz = 0; dz < 2; ++dz)
#pragma unroll
            for (int dy = 0; dy < 2; ++dy)
#pragma unroll
                for (int dx = 0; dx < 2; ++dx) {
                    const double w = __dmul_rn(__dmul_rn(wx[dx], wy[dy]), wz[dz]);
                    atomicAdd(base + ((long long)dz * g.ny + dy) * g.nx + dx, __dmul_rn(qw, w));
                }
    }
}

// ---- per-lane runs of R consecutive particles: 256-bit streaming access --------------------------------
// A lane owns R consecutive particles of the storage order (R = 4 or 8), i.e. 32*R/4 bytes per array = whole
// 32-byte sectors: every LDG.256 / STG.256 of a warp touches 32 distinct, fully used sectors.
__device__ __forceinline__ void ld256(const double *p, double &a, double &b, double &c, double &d) {
    asm volatile("ld.global.cs.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
__device__ __forceinline__ void st256(double *p, double a, double b, double c, double d) {
    asm volatile("st.global.cs.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
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
template <int R, bool VEC>
__device__ __forceinline__ void store_run(double *__restrict__ q, long long p0, long long n, const double (&v)[R]) {
    if (VEC && p0 + R <= n) {
#pragma unroll
        for (int r = 0; r < R; r += 4) st256(q + p0 + r, v[r], v[r + 1], v[r + 2], v[r + 3]);
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (p0 + r < n) q[p0 + r] = v[r];
    }
}

// ---- S5 deposit, mode 1 (default): run accumulation in registers + warp-segmented merge ------------
// A warp owns chunks of 32*R consecutive particles (storage order); lane L walks particles [L*R, (L+1)*R) of
// the chunk and keeps the 8 node sums of the CURRENT cell in registers, flushing them with 8 RED.E.ADD.F64 only
// when the cell changes.  At the end of the chunk the lanes' open runs are merged by a segmented shuffle
// reduction over equal cell keys (contiguous after bt_beam_sort_by_cell), so a chunk that sits in one cell costs
// 8 global reductions for 32*R particles.  Correct for ANY particle order: unsorted input just degenerates to one
// flush per particle.  Weights are the canonical R11 expression, so only the summation order differs from the
// definition.
__device__ __forceinline__ void flush_cell(double *__restrict__ rho, int key, const double (&acc)[8], int nx, long long nxy) {
    if (key < 0) return;
    double *base = rho + key;  // key = linear index of the lower-corner node
    atomicAdd(base, acc[0]);
    atomicAdd(base + 1, acc[1]);
    atomicAdd(base + nx, acc[2]);
    atomicAdd(base + nx + 1, acc[3]);
    atomicAdd(base + nxy, acc[4]);
    atomicAdd(base + nxy + 1, acc[5]);
    atomicAdd(base + nxy + nx, acc[6]);
    atomicAdd(base + nxy + nx + 1, acc[7]);
}

template <int R, bool VEC>
__global__ void __launch_bounds__(256) deposit_runs_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                                           const double *__restrict__ t, long long n, GridDev g, double qw,
                                                           double zscale, double *__restrict__ rho) {
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    const long long chunk = 32LL * R;
    const long long nxy = (long long)g.nx * g.ny;
    for (long long c0 = warp * chunk; c0 < n; c0 += nwarps * chunk) {
        const long long p0 = c0 + (long long)lane * R;
        double px_[R], py_[R], pt_[R];
        load_run<R, VEC>(x, p0, n, CUDART_NAN, px_);  // NaN => outside => contributes nothing
        load_run<R, VEC>(y, p0, n, 0.0, py_);
        load_run<R, VEC>(t, p0, n, 0.0, pt_);
        int cur = -1;
        double acc[8];
#pragma unroll
        for (int d = 0; d < 8; ++d) acc[d] = 0.0;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            Cic c;
            const bool in = cic_locate(g, px_[r], py_[r], pt_[r], zscale, c);
            const int key = in ? (c.k * g.ny + c.j) * g.nx + c.i : -1;
            const double wx0 = __dsub_rn(1.0, c.wx1), wy0 = __dsub_rn(1.0, c.wy1), wz0 = __dsub_rn(1.0, c.wz1);
            double w[8];
            w[0] = __dmul_rn(qw, __dmul_rn(__dmul_rn(wx0, wy0), wz0));
            w[1] = __dmul_rn(qw, __dmul_rn(__dmul_rn(c.wx1, wy0), wz0));
            w[2] = __dmul_rn(qw, __dmul_rn(__dmul_rn(wx0, c.wy1), wz0));
            w[3] = __dmul_rn(qw, __dmul_rn(__dmul_rn(c.wx1, c.wy1), wz0));
            w[4] = __dmul_rn(qw, __dmul_rn(__dmul_rn(wx0, wy0), c.wz1));
            w[5] = __dmul_rn(qw, __dmul_rn(__dmul_rn(c.wx1, wy0), c.wz1));
            w[6] = __dmul_rn(qw, __dmul_rn(__dmul_rn(wx0, c.wy1), c.wz1));
            w[7] = __dmul_rn(qw, __dmul_rn(__dmul_rn(c.wx1, c.wy1), c.wz1));
            if (key != cur) {
                flush_cell(rho, cur, acc, g.nx, nxy);
                cur = key;
#pragma unroll
                for (int d = 0; d < 8; ++d) acc[d] = w[d];
            } else if (in) {
#pragma unroll
                for (int d = 0; d < 8; ++d) acc[d] += w[d];
            }
        }
        // merge the lanes' open runs: segmented suffix reduction over CONTIGUOUS equal keys (after a cell
        // sort equal keys are contiguous; for arbitrary order non-adjacent equal keys stay separate runs)
        const int prev = __shfl_up_sync(0xffffffffu, cur, 1);
        const bool head = (lane == 0) || (prev != cur);
        const unsigned heads = __ballot_sync(0xffffffffu, head);
        const unsigned above = (lane == 31) ? 0u : (heads >> (lane + 1));
        const int end = above ? lane + __ffs(above) - 1 : 31;  // last lane of this lane's run
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const bool take = lane + d <= end;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const double o = __shfl_down_sync(0xffffffffu, acc[k], d);
                if (take) acc[k] += o;
            }
        }
        if (head) flush_cell(rho, cur, acc, g.nx, nxy);
    }
}

// ---- S4+S5 deposit, mode 3 (default): block-local cell binning in shared memory + run accumulation ------------
// A block owns chunks of 256*R consecutive particles (storage order).  The particles of a chunk are binned by cell
// INSIDE the block (counting sort over the chunk's bounding box of cells: one shared-memory integer atomic per
// particle gives count and rank at once, a block scan gives the offsets), so that afterwards every thread walks R
// entries of the cell-ordered list and sums same-cell particles in registers; a run is flushed with 8 RED.E.ADD.F64
// when the cell changes, and the lanes' open runs are merged by a segmented shuffle reduction first.  Global
// reductions per chunk = 8 x (distinct cells + warp seams) instead of 8 x particles, for ANY order in which a chunk
// is spatially compact (bt_beam_sort_by_cell once, then many drift/kick steps: particles wander a few cells, the
// chunk's box stays small).  Consecutive lanes flush x-adjacent cells, so the REDs of one instruction share
// 32-byte sectors (measured: 0.6-0.8 SM-cycles per RED lane against 1.55 for scattered sectors).
// A chunk whose box exceeds kBinCap cells (unsorted input, the thin tails of the bunch) takes the direct path:
// per-lane runs in storage order, as in mode 1.  Weights are the canonical R11 expression on every path.
constexpr int kBinBlock = 256;
constexpr int kBinCap = 4096;  // cells of the chunk's bounding box that the shared histogram can hold

__device__ __forceinline__ void cic_weights8(const Cic &c, double qw, double (&w)[8]) {
    const double wx0 = __dsub_rn(1.0, c.wx1), wy0 = __dsub_rn(1.0, c.wy1), wz0 = __dsub_rn(1.0, c.wz1);
    w[0] = __dmul_rn(qw, __dmul_rn(__dmul_rn(wx0, wy0), wz0));
    w[1] = __dmul_rn(qw, __dmul_rn(__dmul_rn(c.wx1, wy0), wz0));
    w[2] = __dmul_rn(qw, __dmul_rn(__dmul_rn(wx0, c.wy1), wz0));
    w[3] = __dmul_rn(qw, __dmul_rn(__dmul_rn(c.wx1, c.wy1), wz0));
    w[4] = __dmul_rn(qw, __dmul_rn(__dmul_rn(wx0, wy0), c.wz1));
    w[5] = __dmul_rn(qw, __dmul_rn(__dmul_rn(c.wx1, wy0), c.wz1));
    w[6] = __dmul_rn(qw, __dmul_rn(__dmul_rn(wx0, c.wy1), c.wz1));
    w[7] = __dmul_rn(qw, __dmul_rn(__dmul_rn(c.wx1, c.wy1), c.wz1));
}

// merge the lanes' open runs (segmented suffix reduction over CONTIGUOUS equal keys), heads flush
__device__ __forceinline__ void merge_and_flush(double *__restrict__ rho, int cur, double (&acc)[8], int nx, long long nxy) {
    const int lane = threadIdx.x & 31;
    const int prev = __shfl_up_sync(0xffffffffu, cur, 1);
    const bool head = (lane == 0) || (prev != cur);
    const unsigned heads = __ballot_sync(0xffffffffu, head);
    if (heads != 0xffffffffu) {  // warp-uniform: some run spans lanes
        const unsigned above = (lane == 31) ? 0u : (heads >> (lane + 1));
        const int end = above ? lane + __ffs(above) - 1 : 31;  // last lane of this lane's run
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const bool take = lane + d <= end;
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const double o = __shfl_down_sync(0xffffffffu, acc[k], d);
                if (take) acc[k] += o;
            }
        }
    }
    if (head) flush_cell(rho, cur, acc, nx, nxy);
}

template <int R>
struct BinSmem {
    static constexpr int CH = kBinBlock * R;
    static constexpr int PAD = CH + CH / 8;  // one pad slot per 8 entries: a thread's R-entry walk is conflict-free
    int hist[kBinCap + 1];
    int box[2][6];  // imin, jmin, kmin, imax, jmax, kmax; double-buffered by chunk parity (no extra barrier)
    int warp_tot[kBinBlock / 32];
    int key[PAD];
    double w1[3][PAD];
};

template <int R, bool VEC>
__global__ void __launch_bounds__(kBinBlock) deposit_binned_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                                                   const double *__restrict__ t, long long n, GridDev g, double qw,
                                                                   double zscale, double *__restrict__ rho) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    BinSmem<R> &sm = *reinterpret_cast<BinSmem<R> *>(smem_raw);
    constexpr int CH = BinSmem<R>::CH;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const long long nxy = (long long)g.nx * g.ny;
    const long long nchunks = (n + CH - 1) / CH;
    int parity = 0;
    for (long long ch = blockIdx.x; ch < nchunks; ch += gridDim.x, parity ^= 1) {
        int *box = sm.box[parity];
        const long long p0 = ch * CH + (long long)tid * R;
        double qx[R], qy[R], qt[R];
        load_run<R, VEC>(x, p0, n, CUDART_NAN, qx);  // NaN => outside => contributes nothing
        load_run<R, VEC>(y, p0, n, 0.0, qy);
        load_run<R, VEC>(t, p0, n, 0.0, qt);
        if (tid < 3) box[tid] = 0x7fffffff;
        else if (tid < 6) box[tid] = -1;
        __syncthreads();
        Cic c[R];
        bool in[R];
        int lo_i = 0x7fffffff, lo_j = 0x7fffffff, lo_k = 0x7fffffff, hi_i = -1, hi_j = -1, hi_k = -1;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            in[r] = cic_locate(g, qx[r], qy[r], qt[r], zscale, c[r]);
            if (in[r]) {
                lo_i = min(lo_i, c[r].i), hi_i = max(hi_i, c[r].i);
                lo_j = min(lo_j, c[r].j), hi_j = max(hi_j, c[r].j);
                lo_k = min(lo_k, c[r].k), hi_k = max(hi_k, c[r].k);
            }
        }
        lo_i = __reduce_min_sync(0xffffffffu, lo_i), hi_i = __reduce_max_sync(0xffffffffu, hi_i);
        lo_j = __reduce_min_sync(0xffffffffu, lo_j), hi_j = __reduce_max_sync(0xffffffffu, hi_j);
        lo_k = __reduce_min_sync(0xffffffffu, lo_k), hi_k = __reduce_max_sync(0xffffffffu, hi_k);
        if (lane == 0 && hi_i >= 0) {
            atomicMin(&box[0], lo_i), atomicMin(&box[1], lo_j), atomicMin(&box[2], lo_k);
            atomicMax(&box[3], hi_i), atomicMax(&box[4], hi_j), atomicMax(&box[5], hi_k);
        }
        __syncthreads();
        const int i0 = box[0], j0 = box[1], k0 = box[2];
        const int bx = box[3] - i0 + 1, by = box[4] - j0 + 1, bz = box[5] - k0 + 1;
        if (box[3] < 0) continue;  // no particle of this chunk is inside the grid (block-uniform)
        const long long ncell_ll = (long long)bx * by * bz;
        if (ncell_ll > kBinCap) {
            // direct path: runs in storage order
            int cur = -1;
            double acc[8];
#pragma unroll
            for (int d = 0; d < 8; ++d) acc[d] = 0.0;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (!in[r]) continue;
                const int key = (c[r].k * g.ny + c[r].j) * g.nx + c[r].i;
                double w[8];
                cic_weights8(c[r], qw, w);
                if (key != cur) {
                    flush_cell(rho, cur, acc, g.nx, nxy);
                    cur = key;
#pragma unroll
                    for (int d = 0; d < 8; ++d) acc[d] = w[d];
                } else {
#pragma unroll
                    for (int d = 0; d < 8; ++d) acc[d] += w[d];
                }
            }
            merge_and_flush(rho, cur, acc, g.nx, nxy);
            continue;
        }
        const int ncell = (int)ncell_ll;
        for (int s = tid; s <= ncell; s += kBinBlock) sm.hist[s] = 0;
        __syncthreads();
        int lc[R], rank[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            lc[r] = ((c[r].k - k0) * by + (c[r].j - j0)) * bx + (c[r].i - i0);
            rank[r] = in[r] ? atomicAdd(&sm.hist[lc[r]], 1) : 0;
        }
        __syncthreads();
        // exclusive scan of hist[0..ncell) in place; hist[ncell] = number of inside particles
        {
            const int ipt = (ncell + kBinBlock - 1) / kBinBlock;
            const int b0 = tid * ipt;
            int s = 0;
            for (int q = 0; q < ipt; ++q)
                if (b0 + q < ncell) s += sm.hist[b0 + q];
            int incl = s;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += o;
            }
            if (lane == 31) sm.warp_tot[wid] = incl;
            __syncthreads();
            int off = incl - s;
            for (int w = 0; w < wid; ++w) off += sm.warp_tot[w];
            for (int q = 0; q < ipt; ++q)
                if (b0 + q < ncell) {
                    const int v = sm.hist[b0 + q];
                    sm.hist[b0 + q] = off;
                    off += v;
                }
            if (tid == kBinBlock - 1) sm.hist[ncell] = off;
        }
        __syncthreads();
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
        __syncthreads();
        {
            const int total = sm.hist[ncell];
            int cur = -1;
            double acc[8];
#pragma unroll
            for (int d = 0; d < 8; ++d) acc[d] = 0.0;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int e = tid * R + r;
                if (e >= total) break;
                const int slot = e + (e >> 3);
                const int key = sm.key[slot];
                Cic cc;
                cc.i = cc.j = cc.k = 0;
                cc.wx1 = sm.w1[0][slot], cc.wy1 = sm.w1[1][slot], cc.wz1 = sm.w1[2][slot];
                double w[8];
                cic_weights8(cc, qw, w);
                if (key != cur) {
                    flush_cell(rho, cur, acc, g.nx, nxy);
                    cur = key;
#pragma unroll
                    for (int d = 0; d < 8; ++d) acc[d] = w[d];
                } else {
#pragma unroll
                    for (int d = 0; d < 8; ++d) acc[d] += w[d];
                }
            }
            merge_and_flush(rho, cur, acc, g.nx, nxy);
        }
        __syncthreads();  // the next chunk reuses box/hist/entries
    }
}

static int env_int_grid(const char *name, int dflt) {
    const char *v = getenv(name);
    return (v && *v) ? atoi(v) : dflt;
}

template <int R>
static void launch_deposit_runs(Beam *b, Grid *g, const GridDev &gd, double q_weight, double zscale) {
    const int block = 256;
    const long long per_block = (long long)block * R;
    long long blocks = (b->n + per_block - 1) / per_block;
    const long long cap = (long long)b->num_sms * 8;
    if (blocks > cap) blocks = cap;
    if (b->aligned32)
        deposit_runs_kernel<R, true><<<(int)blocks, block, 0, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight, zscale, g->rho);
    else
        deposit_runs_kernel<R, false><<<(int)blocks, block, 0, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight, zscale, g->rho);
}

template <int R>
static int launch_deposit_binned(Beam *b, Grid *g, const GridDev &gd, double q_weight, double zscale) {
    const int smem = (int)sizeof(BinSmem<R>);
    const long long nchunks = (b->n + BinSmem<R>::CH - 1) / BinSmem<R>::CH;
    long long blocks = nchunks;
    int per_sm = 1;
    if (b->aligned32) {
        BT_CUDA_TRY(cudaFuncSetAttribute(deposit_binned_kernel<R, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        BT_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, deposit_binned_kernel<R, true>, kBinBlock, smem));
    } else {
        BT_CUDA_TRY(cudaFuncSetAttribute(deposit_binned_kernel<R, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        BT_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, deposit_binned_kernel<R, false>, kBinBlock, smem));
    }
    const long long cap = (long long)b->num_sms * (per_sm > 0 ? per_sm : 1);
    if (blocks > cap) blocks = cap;
    if (b->aligned32) {
        deposit_binned_kernel<R, true><<<(int)blocks, kBinBlock, smem, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight, zscale, g->rho);
    } else {
        deposit_binned_kernel<R, false><<<(int)blocks, kBinBlock, smem, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight, zscale, g->rho);
    }
    return BT_OK;
}

int launch_deposit(Beam *b, Grid *g, double q_weight, double zscale) {
    const GridDev gd = make_grid_dev(*g);
    // mode 0: one particle per thread, 8 reductions each; 1: lane runs of 4; 2: lane runs of 8;
    // 3 (default) / 4: block-local cell binning, 4 / 8 particles per thread
    const int mode = env_int_grid("BT_DEPOSIT_MODE", 3);
    if (mode == 3 || mode == 4) {
        const int rc = mode == 3 ? launch_deposit_binned<4>(b, g, gd, q_weight, zscale) : launch_deposit_binned<8>(b, g, gd, q_weight, zscale);
        if (rc != BT_OK) return rc;
    } else if (mode == 0) {
        const int block = 256;
        long long blocks = (b->n + block - 1) / block;
        const long long cap = (long long)b->num_sms * 16;
        if (blocks > cap) blocks = cap;
        deposit_atomic_kernel<<<(int)blocks, block, 0, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight, zscale, g->rho);
    } else if (mode == 2) {
        launch_deposit_runs<8>(b, g, gd, q_weight, zscale);
    } else {
        launch_deposit_runs<4>(b, g, gd, q_weight, zscale);
    }
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

__global__ void __launch_bounds__(256) gather_kick_kernel(const __grid_constant__ GatherArgs a) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < a.n; p += stride) {
        double x = __ldcs(a.q[0] + p), px = __ldcs(a.q[1] + p), y = __ldcs(a.q[2] + p);
        double py = __ldcs(a.q[3] + p), t = __ldcs(a.q[4] + p), pt = __ldcs(a.q[5] + p);
        // R4 drift before the kick
        x = fma(a.hb, px, x);
        y = fma(a.hb, py, y);
        t = fma(a.tcb, pt, t);
        Cic c;
        if (cic_locate(a.g, x, y, t, a.zscale, c)) {
            const double wx[2] = {__dsub_rn(1.0, c.wx1), c.wx1};
            const double wy[2] = {__dsub_rn(1.0, c.wy1), c.wy1};
            const double wz[2] = {__dsub_rn(1.0, c.wz1), c.wz1};
            const double *base = a.field + 4 * (((long long)c.k * a.g.ny + c.j) * a.g.nx + c.i);
            double ex = 0.0, ey = 0.0, ez = 0.0;
#pragma unroll
            for (int dz = 0; dz < 2; ++dz)
#pragma unroll
                for (int dy = 0; dy < 2; ++dy)
#pragma unroll
                    for (int dx = 0; dx < 2; ++dx) {
                        const double w = __dmul_rn(__dmul_rn(wx[dx], wy[dy]), wz[dz]);
                        double fx, fy, fz;
                        ld_node(base + 4 * (((long long)dz * a.g.ny + dy) * a.g.nx + dx), fx, fy, fz);
                        ex = fma(w, fx, ex);
                        ey = fma(w, fy, ey);
                        ez = fma(w, fz, ez);
                    }
            px = fma(a.coef[0], ex, px);
            py = fma(a.coef[1], ey, py);
            pt = fma(a.coef[2], ez, pt);
        }
        // R4 drift after the kick
        x = fma(a.ha, px, x);
        y = fma(a.ha, py, y);
        t = fma(a.tca, pt, t);
        __stcs(a.q[0] + p, x);
        __stcs(a.q[1] + p, px);
        __stcs(a.q[2] + p, y);
        __stcs(a.q[3] + p, py);
        __stcs(a.q[4] + p, t);
        __stcs(a.q[5] + p, pt);
    }
}

// ---- S6/S7 for cell-sorted storage: lane runs of 4 consecutive particles, field of the current cell cached ----
// Same arithmetic as gather_kick_kernel per particle.  A lane keeps the 8 node records (24 doubles) of the cell it
// is in and reloads them only when the next particle of its run sits in another cell; particle I/O is one 256-bit
// streaming access per array per lane (6 loads, 6 stores per 4 particles, every sector fully used), all issued
// before the first field access, so a warp has 6 KiB of particle data in flight.
template <bool VEC>
__global__ void __launch_bounds__(128) gather_kick_runs_kernel(const __grid_constant__ GatherArgs a) {
    constexpr int R = 4;
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    const long long chunk = 32LL * R;
    for (long long c0 = warp * chunk; c0 < a.n; c0 += nwarps * chunk) {
        const long long p0 = c0 + (long long)lane * R;
        double x[R], px[R], y[R], py[R], t[R], pt[R];
        load_run<R, VEC>(a.q[0], p0, a.n, CUDART_NAN, x);
        load_run<R, VEC>(a.q[1], p0, a.n, 0.0, px);
        load_run<R, VEC>(a.q[2], p0, a.n, 0.0, y);
        load_run<R, VEC>(a.q[3], p0, a.n, 0.0, py);
        load_run<R, VEC>(a.q[4], p0, a.n, 0.0, t);
        load_run<R, VEC>(a.q[5], p0, a.n, 0.0, pt);
        int cur = -1;
        double fx[8], fy[8], fz[8];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            // R4 drift before the kick
            x[r] = fma(a.hb, px[r], x[r]);
            y[r] = fma(a.hb, py[r], y[r]);
            t[r] = fma(a.tcb, pt[r], t[r]);
            Cic c;
            if (cic_locate(a.g, x[r], y[r], t[r], a.zscale, c)) {
                const int key = (c.k * a.g.ny + c.j) * a.g.nx + c.i;
                if (key != cur) {
                    cur = key;
                    const double *base = a.field + 4 * (long long)key;
#pragma unroll
                    for (int dz = 0; dz < 2; ++dz)
#pragma unroll
                        for (int dy = 0; dy < 2; ++dy)
#pragma unroll
                            for (int dx = 0; dx < 2; ++dx)
                                ld_node(base + 4 * (((long long)dz * a.g.ny + dy) * a.g.nx + dx), fx[dz * 4 + dy * 2 + dx],
                                        fy[dz * 4 + dy * 2 + dx], fz[dz * 4 + dy * 2 + dx]);
                }
                const double wx[2] = {__dsub_rn(1.0, c.wx1), c.wx1};
                const double wy[2] = {__dsub_rn(1.0, c.wy1), c.wy1};
                const double wz[2] = {__dsub_rn(1.0, c.wz1), c.wz1};
                double ex = 0.0, ey = 0.0, ez = 0.0;
#pragma unroll
                for (int dz = 0; dz < 2; ++dz)
#pragma unroll
                    for (int dy = 0; dy < 2; ++dy)
#pragma unroll
                        for (int dx = 0; dx < 2; ++dx) {
                            const double w = __dmul_rn(__dmul_rn(wx[dx], wy[dy]), wz[dz]);
                            ex = fma(w, fx[dz * 4 + dy * 2 + dx], ex);
                            ey = fma(w, fy[dz * 4 + dy * 2 + dx], ey);
                            ez = fma(w, fz[dz * 4 + dy * 2 + dx], ez);
                        }
                px[r] = fma(a.coef[0], ex, px[r]);
                py[r] = fma(a.coef[1], ey, py[r]);
                pt[r] = fma(a.coef[2], ez, pt[r]);
            }
            // R4 drift after the kick
            x[r] = fma(a.ha, px[r], x[r]);
            y[r] = fma(a.ha, py[r], y[r]);
            t[r] = fma(a.tca, pt[r], t[r]);
        }
        store_run<R, VEC>(a.q[0], p0, a.n, x);
        store_run<R, VEC>(a.q[1], p0, a.n, px);
        store_run<R, VEC>(a.q[2], p0, a.n, y);
        store_run<R, VEC>(a.q[3], p0, a.n, py);
        store_run<R, VEC>(a.q[4], p0, a.n, t);
        store_run<R, VEC>(a.q[5], p0, a.n, pt);
    }
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
    // cell-sorted storage (bt_beam_sort_by_cell since the last upload): lane runs with the cell's field cached;
    // any other order: one particle per thread.  BT_GATHER_MODE=0/1 forces one of them (both are correct for any order).
    const int mode = env_int_grid("BT_GATHER_MODE", b->permuted ? 1 : 0);
    if (mode == 1) {
        const int block = 128;
        long long blocks = (b->n + block * 4LL - 1) / (block * 4LL);
        const long long cap = (long long)b->num_sms * 16;
        if (blocks > cap) blocks = cap;
        if (b->aligned32)
            gather_kick_runs_kernel<true><<<(int)blocks, block, 0, b->stream>>>(a);
        else
            gather_kick_runs_kernel<false><<<(int)blocks, block, 0, b->stream>>>(a);
    } else {
        const int block = 256;
        long long blocks = (b->n + block - 1) / block;
        const long long cap = (long long)b->num_sms * 16;
        if (blocks > cap) blocks = cap;
        gather_kick_kernel<<<(int)blocks, block, 0, b->stream>>>(a);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_gather_kick launch: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(1);
    return BT_OK;
}

}  // namespace bt
