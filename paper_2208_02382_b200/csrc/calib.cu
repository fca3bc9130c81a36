// Measurement utilities: the two roofline denominators of the fused walk, measured on the box.
//   bt_calib_fp64: FP64 pipe issue-slot peak (independent DFMA chains, registers only).
//   bt_calib_rw6 : stream ceiling for bt_track's access pattern (6 arrays in, 6 arrays out).
#include "bt_internal.h"

namespace bt {

constexpr int kChains = 8;   // independent (x, p) pairs per thread
constexpr int kInner = 32;   // unrolled pair updates per loop trip: 2 * kChains * kInner DFMAs

// The instruction mix of the fused walk, without its interpreter: DFMAs with TWO vector operands and ONE uniform
// (kernel-parameter) operand, the form `x = fma(c, p, x)` of every map.  (Round 1's version fed all three operands from
// vector registers, which costs FP64 issue rate -- it read 0.92 of 148 x 64 x clock while the walk itself held 0.95.)
__global__ void __launch_bounds__(256) fp64_peak_kernel(double *out, int iters, double a, double b) {
    double x[kChains], p[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) x[c] = (double)(threadIdx.x + c) * 1e-3, p[c] = (double)(c + 1) * 1e-3;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < kInner; ++k)
#pragma unroll
            for (int c = 0; c < kChains; ++c) {
                x[c] = fma(a, p[c], x[c]);
                p[c] = fma(b, x[c], p[c]);
            }
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += x[c] + p[c];
    if (s == 123.456) out[0] = s;  // never true for the chosen a, b; keeps the chains alive
}

__global__ void __launch_bounds__(256) rw6_kernel(double2 *const __restrict__ q0, double2 *const __restrict__ q1,
                                                  double2 *const __restrict__ q2, double2 *const __restrict__ q3,
                                                  double2 *const __restrict__ q4, double2 *const __restrict__ q5,
                                                  long long n2) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n2) return;
    double2 a = __ldcs(q0 + i), b = __ldcs(q1 + i), c = __ldcs(q2 + i), d = __ldcs(q3 + i), e = __ldcs(q4 + i), f = __ldcs(q5 + i);
    a.x = fma(1e-3, b.x, a.x), a.y = fma(1e-3, b.y, a.y);
    c.x = fma(1e-3, d.x, c.x), c.y = fma(1e-3, d.y, c.y);
    e.x = fma(1e-3, f.x, e.x), e.y = fma(1e-3, f.y, e.y);
    __stcs(q0 + i, a), __stcs(q1 + i, b), __stcs(q2 + i, c), __stcs(q3 + i, d), __stcs(q4 + i, e), __stcs(q5 + i, f);
}

}  // namespace bt

using namespace bt;

extern "C" int bt_calib_fp64(void *cuda_stream, double min_ms, double *slots_per_s) {
    if (!slots_per_s) return fail(BT_ERR_INVALID, "bt_calib_fp64: NULL argument");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    BT_CUDA_TRY(cudaGetDevice(&dev));
    BT_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double *d_out = nullptr;
    BT_CUDA_TRY(cudaMalloc(&d_out, sizeof(double)));
    cudaEvent_t e0, e1;
    BT_CUDA_TRY(cudaEventCreate(&e0));
    BT_CUDA_TRY(cudaEventCreate(&e1));
    const int grid = sms * 8, block = 256, iters = 2000;
    const double per_launch = (double)grid * block * (double)iters * kInner * kChains * 2.0;
    fp64_peak_kernel<<<grid, block, 0, s>>>(d_out, 50, 1e-3, -1e-3);  // warm-up
    g_launch_count.fetch_add(1);
    double best = 0.0, total_ms = 0.0;
    int rc = BT_OK;
    while (total_ms < min_ms || best == 0.0) {
        cudaEventRecord(e0, s);
        fp64_peak_kernel<<<grid, block, 0, s>>>(d_out, iters, 1e-3, -1e-3);
        cudaEventRecord(e1, s);
        g_launch_count.fetch_add(1);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) {
            rc = fail(BT_ERR_CUDA, std::string("bt_calib_fp64: ") + cudaGetErrorString(e));
            break;
        }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        total_ms += ms;
        const double rate = per_launch / (ms * 1e-3);
        if (rate > best) best = rate;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_out);
    *slots_per_s = best;
    return rc;
}

extern "C" int bt_calib_rw6(void *cuda_stream, int64_t n, int32_t reps, double *gbytes_per_s) {
    if (!gbytes_per_s || n < 2 || reps < 1) return fail(BT_ERR_INVALID, "bt_calib_rw6: invalid argument");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    n &= ~(int64_t)1;
    double *buf = nullptr;
    const size_t stride = (((size_t)n * sizeof(double)) + 255u) & ~(size_t)255u;
    BT_CUDA_TRY(cudaMalloc(&buf, stride * 6));
    cudaMemsetAsync(buf, 0, stride * 6, s);
    double2 *q[6];
    for (int c = 0; c < 6; ++c) q[c] = (double2 *)((char *)buf + stride * c);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const long long n2 = n / 2;
    const int block = 256;
    const int grid = (int)((n2 + block - 1) / block);
    double best = 0.0;
    int rc = BT_OK;
    for (int r = 0; r < reps + 1; ++r) {
        cudaEventRecord(e0, s);
        rw6_kernel<<<grid, block, 0, s>>>(q[0], q[1], q[2], q[3], q[4], q[5], n2);
        cudaEventRecord(e1, s);
        g_launch_count.fetch_add(1);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) {
            rc = fail(BT_ERR_CUDA, std::string("bt_calib_rw6: ") + cudaGetErrorString(e));
            break;
        }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r == 0) continue;  // warm-up
        const double gbs = 96.0 * (double)n / (ms * 1e-3) * 1e-9;
        if (gbs > best) best = gbs;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(buf);
    *gbytes_per_s = best;
    return rc;
}
