// S4: cell binning.  bt_beam_sort_by_cell physically reorders the particle storage by the linear index of
// each particle's lower-corner node (R11 canonical index), so that the deposit can accumulate runs of
// same-cell particles in registers and the gather finds its 8 nodes in L1.  Counting sort in ONE data pass:
//   1. sort_count_kernel: key = (k*ny + j)*nx + i (nn for particles outside the grid) -> per-cell histogram    [24 B/particle]
//   2. exclusive scan of the histogram (three small kernels)                                                   [16 B/cell]
//   3. sort_move_kernel: rank within the cell, destination = offset[key] + rank, and ALL SIX coordinates + the original
//      index of the particle are moved to the beam's second set of arrays in the same kernel                  [52 B in, 52 B out]
//   then the two sets swap roles (ping-pong; no copy back).
// Round 1 ranked in a separate pass and then scattered each array on its own through a scratch array (6 scatters, 6 copies
// back, ids: 0.93 / 0.57 ms for 8e6 particles); here a particle's data crosses HBM once in each direction.
//
// Both kernels are warp-private (a warp owns chunks of 256 consecutive particles, 8 per lane, 256-bit loads; only
// __syncwarp).  Hot cells (the adversarial cold core puts 90 % of the bunch into 8 cells) would serialise global atomics on
// a handful of counters, so a warp first aggregates its chunk in a 512-entry direct-mapped table in shared memory (bin =
// low three bits of each cell index, tagged with the full key; a lane's run of equal keys is one shared atomic): one
// global atomic per distinct (chunk, cell), a direct global atomic only when two cells of a chunk collide in the table.
// In the move kernel the chunk is additionally grouped by cell through a 2 KiB stage in shared memory, so that the
// particles of one (chunk, cell) group leave as one contiguous run per array instead of as scattered 8-byte stores.
#include "bt_internal.h"
#include "grid_dev.cuh"

namespace bt {

constexpr int kSortBins = 512;
constexpr int kSortWarps = 4;             // warps per block

__device__ __forceinline__ void ld256s(const double *p, double &a, double &b, double &c, double &d) {
    asm volatile("ld.global.cs.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a), "=d"(b), "=d"(c), "=d"(d) : "l"(p));
}
template <int R, bool VEC>
__device__ __forceinline__ void load_lane(const double *__restrict__ q, long long p0, long long n, double fill, double (&v)[R]) {
    if (VEC && p0 + R <= n) {
#pragma unroll
        for (int r = 0; r < R; r += 4) ld256s(q + p0 + r, v[r], v[r + 1], v[r + 2], v[r + 3]);
    } else {
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = (p0 + r < n) ? q[p0 + r] : fill;
    }
}

struct SortTable {          // per warp
    alignas(16) int tag[kSortBins];   // -1 = free
    alignas(16) int cnt[kSortBins];
};

__device__ __forceinline__ int sort_bin(const Cic &c) { return ((c.k & 7) << 6) | ((c.j & 7) << 3) | (c.i & 7); }

// keys and table bins of a lane's particles; key = -1 for slots beyond n.  ORDER: the grid's particle shape -- the key is the
// lowest node of THAT shape's stencil (order 1: the cell's lower corner; order 2: nearest node - 1), so that what the sort
// brings together is what the deposit of that shape accumulates in one run (sorted by the order-1 cell, the particles of a
// cell split over up to 8 order-2 stencils)
template <int R, int ORDER>
__device__ __forceinline__ void sort_keys(long long p0, long long n, const GridDev &g, double zscale, int nn, const double (&qx)[R],
                                          const double (&qy)[R], const double (&qt)[R], int (&key)[R], int (&bin)[R]) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
        Cic c;
        const bool in = shape_locate<ORDER>(g, qx[r], qy[r], qt[r], zscale, c);
        key[r] = (p0 + r < n) ? (in ? (c.k * g.ny + c.j) * g.nx + c.i : nn) : -1;
        bin[r] = in ? sort_bin(c) : kSortBins - 1;   // outside particles share the last bin (tagged nn)
    }
}

// One shared atomic per run of equal keys of this lane: returns in rank[] the particle's rank within its (chunk, key) group
// when the key owns its table bin (ok[r] = true), else ok[r] = false (the caller goes to the global counter directly).
template <int R>
__device__ __forceinline__ void sort_claim(SortTable &tb, const int (&key)[R], const int (&bin)[R], int (&rank)[R], bool (&ok)[R],
                                           int (&len)[R]) {
    len[R - 1] = 1;
#pragma unroll
    for (int r = R - 2; r >= 0; --r) len[r] = (key[r] == key[r + 1]) ? len[r + 1] + 1 : 1;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const bool head = (r == 0) || (key[r] != key[r - 1]);
        if (head) {
            ok[r] = false;
            rank[r] = 0;
            if (key[r] >= 0) {
                const int old = atomicCAS(&tb.tag[bin[r]], -1, key[r]);
                ok[r] = (old == -1) || (old == key[r]);
                if (ok[r]) rank[r] = atomicAdd(&tb.cnt[bin[r]], len[r]);
            }
        } else {
            ok[r] = ok[r - 1];
            rank[r] = rank[r - 1] + 1;
        }
    }
}

template <int R, bool VEC, int ORDER>
__global__ void __launch_bounds__(32 * kSortWarps) sort_count_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                                                      const double *__restrict__ t, long long n, GridDev g, double zscale,
                                                                      int *__restrict__ count) {
    __shared__ SortTable tables[kSortWarps];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    SortTable &tb = tables[wid];
    constexpr int BPL = kSortBins / 32;
    const int nn = g.nx * g.ny * g.nz;
#pragma unroll
    for (int q = 0; q < BPL / 4; ++q) {
        *reinterpret_cast<int4 *>(&tb.tag[128 * q + 4 * lane]) = make_int4(-1, -1, -1, -1);
        *reinterpret_cast<int4 *>(&tb.cnt[128 * q + 4 * lane]) = make_int4(0, 0, 0, 0);
    }
    __syncwarp();
    constexpr int CW = 32 * R;
    const long long nchunks = (n + CW - 1) / CW;
    const long long warps_total = (long long)gridDim.x * kSortWarps;
    for (long long ch = (long long)blockIdx.x * kSortWarps + wid; ch < nchunks; ch += warps_total) {
        const long long p0 = ch * CW + (long long)lane * R;
        double qx[R], qy[R], qt[R];
        int key[R], bin[R], rank[R], len[R];
        bool ok[R];
        load_lane<R, VEC>(x, p0, n, 0.0, qx);
        load_lane<R, VEC>(y, p0, n, 0.0, qy);
        load_lane<R, VEC>(t, p0, n, 0.0, qt);
        sort_keys<R, ORDER>(p0, n, g, zscale, nn, qx, qy, qt, key, bin);
        sort_claim<R>(tb, key, bin, rank, ok, len);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const bool head = (r == 0) || (key[r] != key[r - 1]);
            if (head && !ok[r] && key[r] >= 0) atomicAdd(&count[key[r]], len[r]);   // table collision: straight to the counter
        }
        __syncwarp();
        // flush the table into the global histogram and free it for the next chunk
#pragma unroll
        for (int q = 0; q < BPL / 4; ++q) {
            const int b0 = 128 * q + 4 * lane;
            const int4 tg = *reinterpret_cast<const int4 *>(&tb.tag[b0]);
            const int4 cn = *reinterpret_cast<const int4 *>(&tb.cnt[b0]);
            if (cn.x) atomicAdd(&count[tg.x], cn.x);
            if (cn.y) atomicAdd(&count[tg.y], cn.y);
            if (cn.z) atomicAdd(&count[tg.z], cn.z);
            if (cn.w) atomicAdd(&count[tg.w], cn.w);
            if (cn.x | cn.y | cn.z | cn.w) {
                *reinterpret_cast<int4 *>(&tb.tag[b0]) = make_int4(-1, -1, -1, -1);
                *reinterpret_cast<int4 *>(&tb.cnt[b0]) = make_int4(0, 0, 0, 0);
            }
        }
        __syncwarp();
    }
}

struct SortMoveArgs {
    const double *in[6];
    double *out[6];
    const int *ids_in;  // nullptr: storage order == original order (ids = particle index)
    int *ids_out;
    long long n;
    GridDev g;
    double zscale;
    int *cursor;        // exclusive scan of the histogram; advanced by the groups' sizes
};

template <int R>
struct SortMoveSmem {       // per warp
    SortTable tb;
    alignas(16) int gbase[kSortBins];  // global destination of the first particle of the bin's group
    alignas(16) int lbase[kSortBins];  // position of the group in the chunk's cell-ordered list
    int spill;                          // particles that went to the global cursor directly: listed from the end
    unsigned dest[32 * R];              // destination of the e-th particle of the cell-ordered list
    double stage[2][32 * R];            // double-buffered: one __syncwarp per array
};

// R = 4: every coordinate of the lane's particles is loaded up front (7 independent streams in flight per lane), so the
// only global latencies on a chunk's critical path are that load and the cursor atomics; 96 registers, 20 warps per SM.
template <int R, bool VEC, int ORDER>
__global__ void __launch_bounds__(32 * kSortWarps, R == 4 ? 5 : 3) sort_move_kernel(const __grid_constant__ SortMoveArgs a) {
    extern __shared__ __align__(16) unsigned char sort_smem_raw[];
    constexpr int CW = 32 * R;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    SortMoveSmem<R> &sm = reinterpret_cast<SortMoveSmem<R> *>(sort_smem_raw)[wid];
    constexpr int BPL = kSortBins / 32;
    const int nn = a.g.nx * a.g.ny * a.g.nz;
#pragma unroll
    for (int q = 0; q < BPL / 4; ++q) {
        *reinterpret_cast<int4 *>(&sm.tb.tag[128 * q + 4 * lane]) = make_int4(-1, -1, -1, -1);
        *reinterpret_cast<int4 *>(&sm.tb.cnt[128 * q + 4 * lane]) = make_int4(0, 0, 0, 0);
    }
    if (lane == 0) sm.spill = 0;
    __syncwarp();
    const long long nchunks = (a.n + CW - 1) / CW;
    const long long warps_total = (long long)gridDim.x * kSortWarps;
    for (long long ch = (long long)blockIdx.x * kSortWarps + wid; ch < nchunks; ch += warps_total) {
        const long long p0 = ch * CW + (long long)lane * R;
        double v[6][R];
        int id[R];
#pragma unroll
        for (int c = 0; c < 6; ++c) load_lane<R, VEC>(a.in[c], p0, a.n, 0.0, v[c]);
#pragma unroll
        for (int r = 0; r < R; ++r) id[r] = (p0 + r < a.n) ? (a.ids_in ? a.ids_in[p0 + r] : (int)(p0 + r)) : 0;
        int key[R], bin[R], rank[R], len[R];
        bool ok[R];
        sort_keys<R, ORDER>(p0, a.n, a.g, a.zscale, nn, v[0], v[2], v[4], key, bin);
        sort_claim<R>(sm.tb, key, bin, rank, ok, len);
        const int present = (int)(a.n - ch * CW < CW ? a.n - ch * CW : CW);  // particles of this chunk
        // table collisions: the run takes its destination from the global cursor right away and places at the END of the
        // chunk's cell-ordered list (filled backwards), the groups fill it from the front
        int lpos[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const bool head = (r == 0) || (key[r] != key[r - 1]);
            lpos[r] = -1;
            if (key[r] >= 0 && !ok[r]) {
                if (head) {
                    rank[r] = atomicAdd(&a.cursor[key[r]], len[r]);          // rank[] now holds the global destination
                    lpos[r] = present - 1 - atomicAdd(&sm.spill, len[r]);
                } else {
                    rank[r] = rank[r - 1] + 1;
                    lpos[r] = lpos[r - 1] - 1;
                }
                sm.dest[lpos[r]] = (unsigned)rank[r];
            }
        }
        __syncwarp();
        // groups: reserve their ranges in the global order (one atomic per distinct cell of the chunk), scan their sizes
        {
            int4 cn[BPL / 4];
            int s = 0;
#pragma unroll
            for (int q = 0; q < BPL / 4; ++q) {
                const int b0 = 128 * q + 4 * lane;
                const int4 tg = *reinterpret_cast<const int4 *>(&sm.tb.tag[b0]);
                cn[q] = *reinterpret_cast<const int4 *>(&sm.tb.cnt[b0]);
                int4 gb = make_int4(0, 0, 0, 0);
                if (cn[q].x) gb.x = atomicAdd(&a.cursor[tg.x], cn[q].x);
                if (cn[q].y) gb.y = atomicAdd(&a.cursor[tg.y], cn[q].y);
                if (cn[q].z) gb.z = atomicAdd(&a.cursor[tg.z], cn[q].z);
                if (cn[q].w) gb.w = atomicAdd(&a.cursor[tg.w], cn[q].w);
                *reinterpret_cast<int4 *>(&sm.gbase[b0]) = gb;
                s += cn[q].x + cn[q].y + cn[q].z + cn[q].w;
                if (cn[q].x | cn[q].y | cn[q].z | cn[q].w) {
                    *reinterpret_cast<int4 *>(&sm.tb.tag[b0]) = make_int4(-1, -1, -1, -1);
                    *reinterpret_cast<int4 *>(&sm.tb.cnt[b0]) = make_int4(0, 0, 0, 0);
                }
            }
            int incl = s;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += o;
            }
            int off = incl - s;
#pragma unroll
            for (int q = 0; q < BPL / 4; ++q) {
                int4 o;
                o.x = off, off += cn[q].x;
                o.y = off, off += cn[q].y;
                o.z = off, off += cn[q].z;
                o.w = off, off += cn[q].w;
                *reinterpret_cast<int4 *>(&sm.lbase[128 * q + 4 * lane]) = o;
            }
        }
        __syncwarp();
        // position of each grouped particle in the chunk's cell-ordered list and its destination
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (key[r] >= 0 && ok[r]) {
                lpos[r] = sm.lbase[bin[r]] + rank[r];
                sm.dest[lpos[r]] = (unsigned)(sm.gbase[bin[r]] + rank[r]);
            }
        __syncwarp();
        unsigned dst[R];
#pragma unroll
        for (int m = 0; m < R; ++m) dst[m] = (m * 32 + lane < present) ? sm.dest[m * 32 + lane] : 0u;
        // move: one array at a time through the double-buffered stage (cell-ordered), contiguous runs per (chunk, cell) group
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            double *st = sm.stage[c & 1];
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (lpos[r] >= 0) st[lpos[r]] = v[c][r];
            __syncwarp();
#pragma unroll
            for (int m = 0; m < R; ++m)
                if (m * 32 + lane < present) a.out[c][dst[m]] = st[m * 32 + lane];
        }
        int *sti = reinterpret_cast<int *>(sm.stage[0]);   // free again: array 4's readers passed the __syncwarp of array 5
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (lpos[r] >= 0) sti[lpos[r]] = id[r];
        __syncwarp();
#pragma unroll
        for (int m = 0; m < R; ++m)
            if (m * 32 + lane < present) a.ids_out[dst[m]] = sti[m * 32 + lane];
        if (lane == 0) sm.spill = 0;
        __syncwarp();
    }
}

// ---- exclusive scan of m ints (three small launches; m = nx*ny*nz + 1) ---------------------------
constexpr int kScanBlock = 256;
constexpr int kScanItems = 8;  // per thread -> 2048 per block

__global__ void __launch_bounds__(kScanBlock) scan_reduce_kernel(const int *__restrict__ in, int m, int *__restrict__ block_sum) {
    __shared__ int warp_sum[kScanBlock / 32];
    const int base = blockIdx.x * (kScanBlock * kScanItems);
    int s = 0;
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) {
        const int i = base + j * kScanBlock + threadIdx.x;
        if (i < m) s += in[i];
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        int tot = 0;
        for (int w = 0; w < kScanBlock / 32; ++w) tot += warp_sum[w];
        block_sum[blockIdx.x] = tot;
    }
}

__global__ void __launch_bounds__(1024) scan_block_sums_kernel(int *__restrict__ block_sum, int nb) {
    // single block: exclusive scan of nb values in place
    __shared__ int warp_tot[32];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int start = 0; start < nb; start += 1024) {
        const int i = start + threadIdx.x;
        const int v = i < nb ? block_sum[i] : 0;
        int incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, incl, d);
            if ((threadIdx.x & 31) >= d) incl += o;
        }
        if ((threadIdx.x & 31) == 31) warp_tot[threadIdx.x >> 5] = incl;
        __syncthreads();
        if (threadIdx.x < 32) {
            int w = warp_tot[threadIdx.x];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, w, d);
                if (threadIdx.x >= d) w += o;
            }
            warp_tot[threadIdx.x] = w;  // inclusive over warps
        }
        __syncthreads();
        const int warp_off = (threadIdx.x >> 5) ? warp_tot[(threadIdx.x >> 5) - 1] : 0;
        const int c = carry;
        if (i < nb) block_sum[i] = c + warp_off + incl - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry = c + warp_off + incl;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kScanBlock) scan_apply_kernel(int *__restrict__ data, int m, const int *__restrict__ block_off) {
    // exclusive scan within the block's 2048 items (item order: i = base + t*kScanItems + j), plus block offset
    __shared__ int warp_tot[kScanBlock / 32];
    const int base = blockIdx.x * (kScanBlock * kScanItems) + threadIdx.x * kScanItems;
    int v[kScanItems];
    int s = 0;
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) {
        v[j] = (base + j < m) ? data[base + j] : 0;
        s += v[j];
    }
    int incl = s;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, incl, d);
        if ((threadIdx.x & 31) >= d) incl += o;
    }
    if ((threadIdx.x & 31) == 31) warp_tot[threadIdx.x >> 5] = incl;
    __syncthreads();
    int off = block_off[blockIdx.x] + incl - s;
    for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) off += warp_tot[w];
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) {
        if (base + j < m) data[base + j] = off;
        off += v[j];
    }
}

// NOTE: scan_reduce sums items in the strided order (j*B + t) while scan_apply uses the blocked order
// (t*items + j); both cover the same 2048-item block range, so the block totals agree.

template <typename T>
__global__ void __launch_bounds__(256) scatter_kernel(const T *__restrict__ in, const int *__restrict__ dest, long long n,
                                                      T *__restrict__ out) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n) out[dest[p]] = in[p];
}

#define BT_LAUNCH_CHECK(what)                                                                      \
    do {                                                                                           \
        cudaError_t _e = cudaGetLastError();                                                       \
        if (_e != cudaSuccess) return fail(BT_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(_e)); \
        g_launch_count.fetch_add(1);                                                               \
    } while (0)

// The beam's second set of arrays (ping-pong partner of the home arrays), the id arrays and the histogram.
int ensure_alt_storage(Beam *b) {
    const size_t n = (size_t)b->n;
    if (!b->alt[0]) {
        const size_t stride = ((n * sizeof(double)) + 255u) & ~(size_t)255u;
        double *base = nullptr;
        BT_CUDA_TRY(cudaMalloc(&base, stride * 6));
        for (int c = 0; c < 6; ++c) b->alt[c] = (double *)((char *)base + stride * c);
    }
    if (!b->ids) BT_CUDA_TRY(cudaMalloc(&b->ids, n * sizeof(int)));
    if (!b->ids_tmp) BT_CUDA_TRY(cudaMalloc(&b->ids_tmp, n * sizeof(int)));
    return BT_OK;
}

static int ensure_sort_buffers(Beam *b, long long nn) {
    int rc = ensure_alt_storage(b);
    if (rc != BT_OK) return rc;
    if (b->sort_count_cap < nn + 1) {
        if (b->sort_count) {
            BT_CUDA_TRY(cudaStreamSynchronize(b->stream));
            BT_CUDA_TRY(cudaFree(b->sort_count));
            BT_CUDA_TRY(cudaFree(b->sort_block_sum));
            b->sort_count = b->sort_block_sum = nullptr;
        }
        const long long nb = (nn + 1 + kScanBlock * kScanItems - 1) / (kScanBlock * kScanItems);
        BT_CUDA_TRY(cudaMalloc(&b->sort_count, (size_t)(nn + 1) * sizeof(int)));
        BT_CUDA_TRY(cudaMalloc(&b->sort_block_sum, (size_t)nb * sizeof(int)));
        b->sort_count_cap = nn + 1;
    }
    return BT_OK;
}

void set_current_storage(Beam *b, bool use_alt) {
    for (int c = 0; c < 6; ++c) b->q[c] = use_alt ? b->alt[c] : b->home[c];
    b->in_alt = use_alt;
    b->aligned16 = b->aligned32 = true;
    for (int c = 0; c < 6; ++c) {
        if (((uintptr_t)b->q[c]) & 15u) b->aligned16 = false;
        if (((uintptr_t)b->q[c]) & 31u) b->aligned32 = false;
    }
}

int rehome(Beam *b) {
    if (!b->in_alt) return BT_OK;
    for (int c = 0; c < 6; ++c)
        BT_CUDA_TRY(cudaMemcpyAsync(b->home[c], b->alt[c], (size_t)b->n * sizeof(double), cudaMemcpyDeviceToDevice, b->stream));
    set_current_storage(b, false);
    ++b->storage_epoch;
    return BT_OK;
}

template <int ORDER>
static int sort_by_cell_order(Beam *b, const Grid *g, double zscale) {
    if (b->n > 0x7fffffffLL) return fail(BT_ERR_UNSUPPORTED, "bt_beam_sort_by_cell: n exceeds int32");
    const long long nn = g->nn;
    int rc = ensure_sort_buffers(b, nn);
    if (rc != BT_OK) return rc;
    cudaStream_t s = b->stream;
    const GridDev gd = make_grid_dev(*g);
    const int m = (int)(nn + 1);
    const long long n = b->n;
    const int nb = (m + kScanBlock * kScanItems - 1) / (kScanBlock * kScanItems);
    constexpr int R = 4;  // particles per lane in both kernels
    const long long nchunks = (n + 32 * R - 1) / (32 * R);
    long long blocks = (long long)b->num_sms * 8;
    if (blocks > (nchunks + kSortWarps - 1) / kSortWarps) blocks = (nchunks + kSortWarps - 1) / kSortWarps;

    BT_CUDA_TRY(cudaMemsetAsync(b->sort_count, 0, (size_t)m * sizeof(int), s));
    if (b->aligned32)
        sort_count_kernel<R, true, ORDER><<<(int)blocks, 32 * kSortWarps, 0, s>>>(b->q[0], b->q[2], b->q[4], n, gd, zscale, b->sort_count);
    else
        sort_count_kernel<R, false, ORDER><<<(int)blocks, 32 * kSortWarps, 0, s>>>(b->q[0], b->q[2], b->q[4], n, gd, zscale, b->sort_count);
    BT_LAUNCH_CHECK("sort_count_kernel");
    scan_reduce_kernel<<<nb, kScanBlock, 0, s>>>(b->sort_count, m, b->sort_block_sum);
    BT_LAUNCH_CHECK("scan_reduce_kernel");
    scan_block_sums_kernel<<<1, 1024, 0, s>>>(b->sort_block_sum, nb);
    BT_LAUNCH_CHECK("scan_block_sums_kernel");
    scan_apply_kernel<<<nb, kScanBlock, 0, s>>>(b->sort_count, m, b->sort_block_sum);
    BT_LAUNCH_CHECK("scan_apply_kernel");

    SortMoveArgs a;
    const bool to_alt = !b->in_alt;
    for (int c = 0; c < 6; ++c) {
        a.in[c] = b->q[c];
        a.out[c] = to_alt ? b->alt[c] : b->home[c];
    }
    a.ids_in = b->permuted ? b->ids : nullptr;
    a.ids_out = b->ids_tmp;
    a.n = n;
    a.g = gd;
    a.zscale = zscale;
    a.cursor = b->sort_count;
    const int smem = (int)sizeof(SortMoveSmem<R>) * kSortWarps;
    static std::atomic<int> attr_set[kMaxDevices];
    if (b->device >= 0 && b->device < kMaxDevices && !attr_set[b->device].load()) {
        BT_CUDA_TRY(cudaFuncSetAttribute(sort_move_kernel<R, true, ORDER>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        BT_CUDA_TRY(cudaFuncSetAttribute(sort_move_kernel<R, false, ORDER>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        attr_set[b->device].store(1);
    }
    long long mblocks = (long long)b->num_sms * 5;
    if (mblocks > (nchunks + kSortWarps - 1) / kSortWarps) mblocks = (nchunks + kSortWarps - 1) / kSortWarps;
    if (b->aligned32)
        sort_move_kernel<R, true, ORDER><<<(int)mblocks, 32 * kSortWarps, smem, s>>>(a);
    else
        sort_move_kernel<R, false, ORDER><<<(int)mblocks, 32 * kSortWarps, smem, s>>>(a);
    BT_LAUNCH_CHECK("sort_move_kernel");
    set_current_storage(b, to_alt);
    int *tmp = b->ids;
    b->ids = b->ids_tmp;
    b->ids_tmp = tmp;
    b->permuted = true;
    ++b->storage_epoch;
    // Lent arrays (the zero-copy contract, P:l.102): whoever lent them may read them at any time, so the bunch does not stay
    // in the partner set unless the caller asked for ping-pong; one device copy (96 B per particle) brings it back.
    if (b->in_alt && !b->pingpong) return rehome(b);
    return BT_OK;
}

int sort_by_cell(Beam *b, const Grid *g, double zscale) {
    return g->order == 2 ? sort_by_cell_order<2>(b, g, zscale) : sort_by_cell_order<1>(b, g, zscale);
}

// storage order -> original order for one coordinate: out[ids[j]] = q[j]
int unpermute_to(Beam *b, int c, double *out) {
    const int sb = (int)((b->n + 255) / 256);
    scatter_kernel<double><<<sb, 256, 0, b->stream>>>(b->q[c], b->ids, b->n, out);
    BT_LAUNCH_CHECK("scatter_kernel(unpermute)");
    return BT_OK;
}

}  // namespace bt
