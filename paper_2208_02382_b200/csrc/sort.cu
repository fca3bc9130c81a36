// S4: cell binning.  bt_beam_sort_by_cell physically reorders the particle storage by the linear index of
// each particle's lower-corner node (R11 canonical index), so that the deposit can accumulate runs of
// same-cell particles in registers and the gather finds its 8 nodes in L1.  Counting sort:
//   1. key[p] = (k*ny + j)*nx + i, or nn for particles outside the grid; per-cell histogram
//   2. exclusive scan of the histogram
//   3. dest[p] = offset[key] + rank within the cell
//   4. every array (and the original-index array) is scattered through a 1-array scratch that stays in L2
// Hot cells (the adversarial cold core puts 90 % of the bunch into 8 cells) would serialise global atomics on a
// handful of counters, so steps 1 and 3 aggregate per block in a shared-memory hash table first: one global
// atomic per distinct (block, cell).
#include "bt_internal.h"
#include "grid_dev.cuh"

namespace bt {

constexpr int kSortBlock = 256;
constexpr int kSortPPT = 4;        // particles per thread -> 1024 per block
constexpr int kHashSlots = 2048;   // load factor <= 0.5
constexpr int kHashBits = 11;
constexpr int kMaxProbe = 12;

struct BlockHash {
    int keys[kHashSlots];
    int cnt[kHashSlots];
    int base[kHashSlots];
};

__device__ __forceinline__ void hash_clear(BlockHash &h) {
    for (int s = threadIdx.x; s < kHashSlots; s += blockDim.x) {
        h.keys[s] = -1;
        h.cnt[s] = 0;
    }
}

// Returns the slot of `key` (inserting it), or -1 when the probe sequence is exhausted.
__device__ __forceinline__ int hash_insert(BlockHash &h, int key) {
    unsigned s = ((unsigned)key * 0x9E3779B1u) >> (32 - kHashBits);
#pragma unroll 1
    for (int probe = 0; probe < kMaxProbe; ++probe) {
        const int prev = atomicCAS(&h.keys[s], -1, key);
        if (prev == -1 || prev == key) return (int)s;
        s = (s + 1) & (kHashSlots - 1);
    }
    return -1;
}

__global__ void __launch_bounds__(kSortBlock) cell_count_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                                                const double *__restrict__ t, long long n, GridDev g,
                                                                double zscale, int *__restrict__ key_out, int *__restrict__ count) {
    __shared__ BlockHash h;
    hash_clear(h);
    __syncthreads();
    const long long base = (long long)blockIdx.x * (kSortBlock * kSortPPT);
    const int nn = g.nx * g.ny * g.nz;
#pragma unroll
    for (int j = 0; j < kSortPPT; ++j) {
        const long long p = base + j * kSortBlock + threadIdx.x;
        if (p < n) {
            Cic c;
            const bool in = cic_locate(g, x[p], y[p], t[p], zscale, c);
            const int key = in ? (c.k * g.ny + c.j) * g.nx + c.i : nn;
            key_out[p] = key;
            const int s = hash_insert(h, key);
            if (s >= 0)
                atomicAdd(&h.cnt[s], 1);
            else
                atomicAdd(&count[key], 1);
        }
    }
    __syncthreads();
    for (int s = threadIdx.x; s < kHashSlots; s += blockDim.x)
        if (h.keys[s] >= 0) atomicAdd(&count[h.keys[s]], h.cnt[s]);
}

__global__ void __launch_bounds__(kSortBlock) cell_rank_kernel(const int *__restrict__ key_in, long long n,
                                                               int *__restrict__ cursor, int *__restrict__ dest) {
    __shared__ BlockHash h;
    hash_clear(h);
    __syncthreads();
    const long long base = (long long)blockIdx.x * (kSortBlock * kSortPPT);
    int slot[kSortPPT], rank[kSortPPT];
#pragma unroll
    for (int j = 0; j < kSortPPT; ++j) {
        const long long p = base + j * kSortBlock + threadIdx.x;
        slot[j] = -2;
        rank[j] = 0;
        if (p < n) {
            const int key = key_in[p];
            const int s = hash_insert(h, key);
            slot[j] = s;
            rank[j] = (s >= 0) ? atomicAdd(&h.cnt[s], 1) : atomicAdd(&cursor[key], 1);
        }
    }
    __syncthreads();
    for (int s = threadIdx.x; s < kHashSlots; s += blockDim.x)
        if (h.keys[s] >= 0) h.base[s] = atomicAdd(&cursor[h.keys[s]], h.cnt[s]);
    __syncthreads();
#pragma unroll
    for (int j = 0; j < kSortPPT; ++j) {
        const long long p = base + j * kSortBlock + threadIdx.x;
        if (slot[j] >= 0)
            dest[p] = h.base[slot[j]] + rank[j];
        else if (slot[j] == -1)
            dest[p] = rank[j];
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

__global__ void __launch_bounds__(256) scatter_ids_kernel(const int *__restrict__ ids_in, const int *__restrict__ dest,
                                                          long long n, int *__restrict__ out) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p < n) out[dest[p]] = ids_in ? ids_in[p] : (int)p;
}

#define BT_LAUNCH_CHECK(what)                                                                      \
    do {                                                                                           \
        cudaError_t _e = cudaGetLastError();                                                       \
        if (_e != cudaSuccess) return fail(BT_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(_e)); \
        g_launch_count.fetch_add(1);                                                               \
    } while (0)

static int ensure_sort_buffers(Beam *b, long long nn) {
    const size_t n = (size_t)b->n;
    if (!b->sort_key) BT_CUDA_TRY(cudaMalloc(&b->sort_key, n * sizeof(int)));
    if (!b->sort_dest) BT_CUDA_TRY(cudaMalloc(&b->sort_dest, n * sizeof(int)));
    if (!b->ids) BT_CUDA_TRY(cudaMalloc(&b->ids, n * sizeof(int)));
    if (!b->ids_tmp) BT_CUDA_TRY(cudaMalloc(&b->ids_tmp, n * sizeof(int)));
    if (!b->scratch) BT_CUDA_TRY(cudaMalloc(&b->scratch, n * sizeof(double)));
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

int sort_by_cell(Beam *b, const Grid *g, double zscale) {
    if (b->n > 0x7fffffffLL) return fail(BT_ERR_UNSUPPORTED, "bt_beam_sort_by_cell: n exceeds int32");
    const long long nn = g->nn;
    int rc = ensure_sort_buffers(b, nn);
    if (rc != BT_OK) return rc;
    cudaStream_t s = b->stream;
    const GridDev gd = make_grid_dev(*g);
    const int m = (int)(nn + 1);
    const long long n = b->n;
    const int pb = (int)((n + kSortBlock * kSortPPT - 1) / (kSortBlock * kSortPPT));
    const int nb = (m + kScanBlock * kScanItems - 1) / (kScanBlock * kScanItems);

    BT_CUDA_TRY(cudaMemsetAsync(b->sort_count, 0, (size_t)m * sizeof(int), s));
    cell_count_kernel<<<pb, kSortBlock, 0, s>>>(b->q[0], b->q[2], b->q[4], n, gd, zscale, b->sort_key, b->sort_count);
    BT_LAUNCH_CHECK("cell_count_kernel");
    scan_reduce_kernel<<<nb, kScanBlock, 0, s>>>(b->sort_count, m, b->sort_block_sum);
    BT_LAUNCH_CHECK("scan_reduce_kernel");
    scan_block_sums_kernel<<<1, 1024, 0, s>>>(b->sort_block_sum, nb);
    BT_LAUNCH_CHECK("scan_block_sums_kernel");
    scan_apply_kernel<<<nb, kScanBlock, 0, s>>>(b->sort_count, m, b->sort_block_sum);
    BT_LAUNCH_CHECK("scan_apply_kernel");
    cell_rank_kernel<<<pb, kSortBlock, 0, s>>>(b->sort_key, n, b->sort_count, b->sort_dest);
    BT_LAUNCH_CHECK("cell_rank_kernel");

    const int sb = (int)((n + 255) / 256);
    for (int c = 0; c < 6; ++c) {
        scatter_kernel<double><<<sb, 256, 0, s>>>(b->q[c], b->sort_dest, n, b->scratch);
        BT_LAUNCH_CHECK("scatter_kernel");
        BT_CUDA_TRY(cudaMemcpyAsync(b->q[c], b->scratch, (size_t)n * sizeof(double), cudaMemcpyDeviceToDevice, s));
    }
    scatter_ids_kernel<<<sb, 256, 0, s>>>(b->permuted ? b->ids : nullptr, b->sort_dest, n, b->ids_tmp);
    BT_LAUNCH_CHECK("scatter_ids_kernel");
    int *tmp = b->ids;
    b->ids = b->ids_tmp;
    b->ids_tmp = tmp;
    b->permuted = true;
    return BT_OK;
}

// storage order -> original order for one coordinate: out[ids[j]] = q[j]
int unpermute_to(Beam *b, int c, double *out) {
    const int sb = (int)((b->n + 255) / 256);
    scatter_kernel<double><<<sb, 256, 0, b->stream>>>(b->q[c], b->ids, b->n, out);
    BT_LAUNCH_CHECK("scatter_kernel(unpermute)");
    return BT_OK;
}

}  // namespace bt
