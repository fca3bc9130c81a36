// Beam statistics ("beam statistics", l.112 "beam second moments ... emittances",
// l.61 slice-step diagnostics): means and the 6x6 second moments about the mean, ONE pass over the particles.
//
//   mean_i = (1/n) sum q_i ,   cov_ij = (1/n) sum (q_i - mean_i)(q_j - mean_j)
//
// One pass needs a provisional centre k (a two-pass scheme would read the bunch twice): with d = q - k,
//   S_i = sum d_i , P_ij = sum d_i d_j  =>  mean_i = k_i + S_i/n , cov_ij = P_ij/n - (S_i/n)(S_j/n),
// which is the definition exactly (algebraically) and loses no digits as long as |k - mean| is of the order of the rms
// size: k is the mean of min(n, 256) particles sampled at a stride of n/256 through the storage (every block recomputes
// it), so the subtracted term is ~ cov/256 in any storage order, cell-sorted included.
// HBM-bound: 48 bytes and 33 FP64 issue slots per particle.  Deterministic: fixed partition, fixed reduction trees,
// the per-block partials are combined in block order by the last block to finish.  Fixed costs are kept small because a
// 16e6-particle bunch is only 119 us of HBM time: the grid is exactly the resident blocks (one wave), the centre and the 27
// block totals each take ONE barrier pair (all values shuffled first, then exchanged through shared memory at once), and
// bt_beam_moments' 42 results are written straight into mapped pinned host memory (no copy, one stream synchronisation).
#include <mutex>

#include "bt_internal.h"

namespace bt {

constexpr int kMomBlock = 256;
constexpr int kMomVals = 27;  // 6 sums + 21 products (upper triangle, row-major)
constexpr int kCentreSample = kMomBlock;

struct MomArgs {
    const double *q[6];
    long long n;
    double *partial;   // [gridDim.x][27]
    double *out;       // [6 mean][36 cov]
    unsigned int *ticket;
};

__device__ __forceinline__ double block_sum(double v, double *scratch /*[kMomBlock/32]*/) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();  // scratch free
    if (lane == 0) scratch[wid] = v;
    __syncthreads();
    double tot = 0.0;
#pragma unroll
    for (int w = 0; w < kMomBlock / 32; ++w) tot += scratch[w];  // same order in every thread
    return tot;
}

// block totals of NV values at once: warp shuffles, one exchange through shared memory ([NV][warps]), one barrier pair;
// every thread returns with all NV totals (same summation order everywhere)
template <int NV>
__device__ __forceinline__ void block_sum_all(double (&v)[NV], double *scratch /*[NV * kMomBlock/32]*/) {
    constexpr int NWARP = kMomBlock / 32;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v[i] += __shfl_xor_sync(0xffffffffu, v[i], d);
    }
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();  // scratch free
    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < NV; ++i) scratch[i * NWARP + wid] = v[i];
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        double tot = 0.0;
#pragma unroll
        for (int w = 0; w < NWARP; ++w) tot += scratch[i * NWARP + w];
        v[i] = tot;
    }
}

__device__ __forceinline__ void accumulate(const double (&d)[6], double (&s)[6], double (&pr)[21]) {
    int k = 0;
#pragma unroll
    for (int i = 0; i < 6; ++i) {
        s[i] += d[i];
#pragma unroll
        for (int j = i; j < 6; ++j) pr[k] = fma(d[i], d[j], pr[k]), ++k;
    }
}

template <bool VEC2>
__global__ void __launch_bounds__(kMomBlock, 2) moments_kernel(const __grid_constant__ MomArgs a) {
    __shared__ double scratch[kMomVals * (kMomBlock / 32)];
    __shared__ bool is_last;
    // provisional centre: mean of min(n, 256) particles taken at a stride of n/256 through the storage -- representative in
    // any storage order (after bt_beam_sort_by_cell the FIRST 256 particles all sit in one corner of the grid, several
    // sigma from the mean) -- computed by every block in the same order (bitwise identical everywhere; L2 hits after the
    // first block)
    double k[6];
    {
        const long long m = a.n < kCentreSample ? a.n : kCentreSample;
        const long long stride = a.n / m;
        double v[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) v[c] = threadIdx.x < m ? a.q[c][threadIdx.x * stride] : 0.0;
        block_sum_all<6>(v, scratch);
#pragma unroll
        for (int c = 0; c < 6; ++c) k[c] = v[c] / (double)m;
    }
    double s[6], pr[21];
#pragma unroll
    for (int c = 0; c < 6; ++c) s[c] = 0.0;
#pragma unroll
    for (int c = 0; c < 21; ++c) pr[c] = 0.0;
    const long long tid = (long long)blockIdx.x * kMomBlock + threadIdx.x;
    const long long nthreads = (long long)gridDim.x * kMomBlock;
    if (VEC2) {  // arrays 16-byte aligned: 128-bit streaming loads, two particles per thread per trip
        const long long n2 = a.n >> 1;
        for (long long i = tid; i < n2; i += nthreads) {
            double2 v[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) v[c] = __ldcs(reinterpret_cast<const double2 *>(a.q[c]) + i);
            double d0[6], d1[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) d0[c] = v[c].x - k[c], d1[c] = v[c].y - k[c];
            accumulate(d0, s, pr);
            accumulate(d1, s, pr);
        }
        if ((a.n & 1) && tid == 0) {
            double d[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) d[c] = a.q[c][a.n - 1] - k[c];
            accumulate(d, s, pr);
        }
    } else {
        for (long long p = tid; p < a.n; p += nthreads) {
            double d[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) d[c] = __ldcs(a.q[c] + p) - k[c];
            accumulate(d, s, pr);
        }
    }
    // block reduction of the 27 sums at once
    {
        double all[kMomVals];
#pragma unroll
        for (int c = 0; c < 6; ++c) all[c] = s[c];
#pragma unroll
        for (int c = 0; c < 21; ++c) all[6 + c] = pr[c];
        block_sum_all<kMomVals>(all, scratch);
        double *mine = a.partial + (long long)blockIdx.x * kMomVals;
        if (threadIdx.x == 0) {
#pragma unroll
            for (int c = 0; c < kMomVals; ++c) mine[c] = all[c];
        }
    }
    // the last block to finish combines the partials in block order
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int t = atomicAdd(a.ticket, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    // warp w adds the partials of blocks w, w + 8, ... (lane = value), then the eight sums are added in warp order: a fixed
    // order for a given grid, with 8 x 27 independent load streams instead of 27 serial ones
    __shared__ double total[kMomVals];
    {
        const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
        double tot = 0.0;
        if (lane < kMomVals)
            for (unsigned int b = wid; b < gridDim.x; b += kMomBlock / 32) tot += __ldcg(a.partial + (long long)b * kMomVals + lane);
        __syncthreads();  // scratch free
        if (lane < kMomVals) scratch[lane * (kMomBlock / 32) + wid] = tot;
        __syncthreads();
        if (threadIdx.x < kMomVals) {
            double t = 0.0;
#pragma unroll
            for (int w = 0; w < kMomBlock / 32; ++w) t += scratch[threadIdx.x * (kMomBlock / 32) + w];
            total[threadIdx.x] = t;
        }
    }
    __syncthreads();
    const double inv_n = 1.0 / (double)a.n;
    __shared__ double centre[6];
    if (threadIdx.x == 0) {
#pragma unroll
        for (int c = 0; c < 6; ++c) centre[c] = k[c];
    }
    __syncthreads();
    if (threadIdx.x < 6) a.out[threadIdx.x] = centre[threadIdx.x] + total[threadIdx.x] * inv_n;
    if (threadIdx.x < 36) {
        const int i = threadIdx.x / 6, j = threadIdx.x % 6;
        const int lo = i < j ? i : j, hi = i < j ? j : i;
        const int idx = 6 + lo * 6 - lo * (lo - 1) / 2 + (hi - lo);  // position of (lo, hi) in the packed upper triangle
        a.out[6 + threadIdx.x] = total[idx] * inv_n - (total[lo] * inv_n) * (total[hi] * inv_n);
    }
    if (threadIdx.x == 0) *a.ticket = 0u;  // ready for the next call
}

// k[6] = mean of min(n, 256) particles sampled at a stride of n/256: the provisional centre of the diagnostics walk, which
// needs it BEFORE the walk overwrites the bunch (moments_kernel computes the same sample itself, per block).
__global__ void __launch_bounds__(kMomBlock) moments_centre_kernel(const __grid_constant__ MomArgs a) {
    __shared__ double scratch[kMomBlock / 32];
    const long long m = a.n < kCentreSample ? a.n : kCentreSample;
    const long long stride = a.n / m;
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        const double v = threadIdx.x < m ? a.q[c][threadIdx.x * stride] : 0.0;
        const double k = block_sum(v, scratch) / (double)m;
        if (threadIdx.x == 0) a.out[c] = k;
    }
}

int launch_moments_centre(Beam *b, double *dev_centre) {
    MomArgs a;
    for (int c = 0; c < 6; ++c) a.q[c] = b->q[c];
    a.n = b->n;
    a.out = dev_centre;
    a.partial = nullptr;
    a.ticket = nullptr;
    moments_centre_kernel<<<1, kMomBlock, 0, b->stream>>>(a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_track_diagnostics centre: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(1);
    return BT_OK;
}

// Enqueues the reduction; the 42 results (mean[6], cov[36]) land in dev_out on the beam's stream (device memory, or the
// device address of mapped host memory).
int launch_moments_async(Beam *b, double *dev_out) {
    if (b->mom_blocks == 0) {  // one wave: the grid is what is resident at once
        int per_sm_v = 1, per_sm_s = 1;
        BT_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_v, moments_kernel<true>, kMomBlock, 0));
        BT_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_s, moments_kernel<false>, kMomBlock, 0));
        const int per_sm = per_sm_v < per_sm_s ? per_sm_v : per_sm_s;
        b->mom_blocks = b->num_sms * (per_sm > 0 ? per_sm : 1);
    }
    const int max_blocks = b->mom_blocks;
    if (!b->mom_buf) {
        const size_t bytes = (size_t)(6 + 42 + (size_t)max_blocks * kMomVals) * sizeof(double) + 16;
        BT_CUDA_TRY(cudaMalloc(&b->mom_buf, bytes));
        BT_CUDA_TRY(cudaMemsetAsync(b->mom_buf, 0, bytes, b->stream));
    }
    MomArgs a;
    for (int c = 0; c < 6; ++c) a.q[c] = b->q[c];
    a.n = b->n;
    a.out = dev_out ? dev_out : b->mom_buf;
    a.partial = b->mom_buf + 48;
    a.ticket = reinterpret_cast<unsigned int *>(b->mom_buf + 48 + (size_t)max_blocks * kMomVals);
    long long blocks = (b->n / 2 + kMomBlock - 1) / kMomBlock;
    if (blocks > max_blocks) blocks = max_blocks;
    if (blocks < 1) blocks = 1;
    if (b->aligned16)
        moments_kernel<true><<<(int)blocks, kMomBlock, 0, b->stream>>>(a);
    else
        moments_kernel<false><<<(int)blocks, kMomBlock, 0, b->stream>>>(a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_beam_moments launch: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(1);
    return BT_OK;
}

int launch_moments(Beam *b, double host_mean[6], double host_cov[36]) {
    if (!b->mom_host) {
        BT_CUDA_TRY(cudaHostAlloc(&b->mom_host, 42 * sizeof(double), cudaHostAllocMapped));
        BT_CUDA_TRY(cudaHostGetDevicePointer(&b->mom_host_dev, b->mom_host, 0));
    }
    const int rc = launch_moments_async(b, b->mom_host_dev);
    if (rc != BT_OK) return rc;
    BT_CUDA_TRY(cudaStreamSynchronize(b->stream));  // the kernel's writes to mapped host memory are complete
    for (int i = 0; i < 6; ++i) host_mean[i] = b->mom_host[i];
    for (int i = 0; i < 36; ++i) host_cov[i] = b->mom_host[6 + i];
    return BT_OK;
}

// ---- bt_moments_static: the same statistics for callers that must not allocate device memory -------------------------------
//
// Who needs this.  bt_beam_moments / bt_beam_moments_device cudaMalloc their partial-sum buffer on a beam's first call, and
// bt_beam_create itself creates library state.  Some hosts of this library cannot afford that:
//   - an application whose own arena has already claimed (nearly) all of HBM at start-up -- the block-structured mesh
//     frameworks the paper builds on work this way -- so that a cudaMalloc from a plug-in library fails, or succeeds only
//     by taking memory the arena expected to grow into;
//   - a time-critical step loop that keeps several streams busy: cudaMalloc and cudaFree synchronise the whole device, so
//     one stray allocation stalls every stream;
//   - code running under a memory checker / allocator hook that counts every device allocation as a leak or an error.
// Such a caller already owns the six coordinate arrays and a 42-double result buffer.  The only other memory the reduction
// needs is the table of per-block partial sums and a completion counter; here that lives in a fixed array in the library's
// own device data segment, so this entry point makes no cudaMalloc, cudaFree, cudaHostAlloc or other allocating call.
//
// The price, all of which the header repeats:
//   - the array has a fixed capacity (kStaticRows rows of 27 doubles).  The launch uses one block, and so one row, per
//     kStaticSlab particles (a grid that depends on n only, not on the GPU model), hence the limit
//     n <= BT_MOMENTS_STATIC_MAX_PARTICLES; larger n is refused;
//   - every GPU that loads libbt.so carries the array (432.25 KiB) until the process exits, whether or not it is used;
//   - there is ONE array per device, shared by all calls: two calls whose kernels may overlap on the same GPU (different
//     streams, different host threads) race on it.  Order them on one stream or with events;
//   - the array keeps whatever the previous call left.  Rows are always written before they are read, and the completion
//     counter is cleared on the caller's stream before every launch, so a call that died half-way cannot poison the next.
//
// In host code the name g_static_scratch is only a handle to the symbol, not an address the GPU can use.  The device
// address is fetched with cudaGetSymbolAddress, once per device with that device current, and cached; that happens in the
// first call on each device (so make that first call outside any stream capture).
constexpr long long kStaticSlab = 32768;  // particles reduced by one block = one row of partial sums
constexpr long long kStaticRows = BT_MOMENTS_STATIC_MAX_PARTICLES / kStaticSlab;  // 2048
static_assert(kStaticRows * kStaticSlab == BT_MOMENTS_STATIC_MAX_PARTICLES, "the limit must be a whole number of slabs");
constexpr long long kStaticDoubles = kStaticRows * kMomVals + 32;  // rows, then 256 bytes holding the completion counter

static __device__ __align__(256) double g_static_scratch[kStaticDoubles];

static std::mutex g_static_mutex;
static double *g_static_addr[kMaxDevices];  // device address of g_static_scratch per device ordinal, nullptr = not asked yet

// device address of this device's copy of the array (the current device's); no allocation
static int static_scratch_address(double **out) {
    int dev = -1;
    BT_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(BT_ERR_UNSUPPORTED, "bt_moments_static: device ordinal beyond the library's table");
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[dev]) {
        double *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_static_scratch);
        if (e != cudaSuccess || !p)
            return fail(BT_ERR_CUDA, std::string("bt_moments_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        g_static_addr[dev] = p;
    }
    *out = g_static_addr[dev];
    return BT_OK;
}

}  // namespace bt

extern "C" int bt_moments_static(const double *const dev_q[6], int64_t n, double *dev_out, void *cuda_stream) {
    using namespace bt;
    if (!dev_q || !dev_out) return fail(BT_ERR_INVALID, "bt_moments_static: NULL argument");
    if (n < 1) return fail(BT_ERR_INVALID, "bt_moments_static: n must be >= 1");
    if (n > BT_MOMENTS_STATIC_MAX_PARTICLES)
        return fail(BT_ERR_INVALID, "bt_moments_static: n = " + std::to_string((long long)n) + " exceeds BT_MOMENTS_STATIC_MAX_PARTICLES = " +
                                        std::to_string((long long)BT_MOMENTS_STATIC_MAX_PARTICLES) +
                                        " (the fixed scratch array has one row per 32768 particles and 2048 rows); "
                                        "use bt_beam_moments_device, which allocates, for larger bunches");
    bool vec = true;
    for (int c = 0; c < 6; ++c) {
        if (!dev_q[c]) return fail(BT_ERR_INVALID, "bt_moments_static: NULL coordinate array");
        if (reinterpret_cast<uintptr_t>(dev_q[c]) & 7) return fail(BT_ERR_INVALID, "bt_moments_static: coordinate arrays must be 8-byte aligned");
        vec = vec && !(reinterpret_cast<uintptr_t>(dev_q[c]) & 15);
    }
    if (reinterpret_cast<uintptr_t>(dev_out) & 7) return fail(BT_ERR_INVALID, "bt_moments_static: dev_out must be 8-byte aligned");
    double *scratch = nullptr;
    const int rc = static_scratch_address(&scratch);
    if (rc != BT_OK) return rc;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    MomArgs a;
    for (int c = 0; c < 6; ++c) a.q[c] = dev_q[c];
    a.n = n;
    a.out = dev_out;
    a.partial = scratch;
    a.ticket = reinterpret_cast<unsigned int *>(scratch + kStaticRows * kMomVals);
    // the counter must read zero when the first block arrives, whatever an earlier (possibly failed) launch left there
    BT_CUDA_TRY(cudaMemsetAsync(a.ticket, 0, sizeof(unsigned int), stream));
    const int blocks = (int)((n + kStaticSlab - 1) / kStaticSlab);  // <= kStaticRows: every block owns one row
    if (vec)
        moments_kernel<true><<<blocks, kMomBlock, 0, stream>>>(a);
    else
        moments_kernel<false><<<blocks, kMomBlock, 0, stream>>>(a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_moments_static launch: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(1);
    return BT_OK;
}
