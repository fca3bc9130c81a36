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

// ---- S5 deposit, mode 1 (default): run accumulation in registers + warp-segmented merge ------------
// A warp owns chunks of 32*kRun consecutive particles (storage order); lane L walks particles
// [L*kRun, (L+1)*kRun) of the chunk and keeps the 8 node sums of the CURRENT cell in registers, flushing
// them with 8 RED.E.ADD.F64 only when the cell changes.  At the end of the chunk the lanes' open runs are
// merged by a segmented shuffle reduction over equal cell keys (contiguous after bt_beam_sort_by_cell), so a
// chunk that sits in one cell costs 8 global reductions for 256 particles.  Correct for ANY particle order:
// unsorted input just degenerates to one flush per particle.  Weights are the canonical R11 expression, so
// only the summation order differs from the definition.
constexpr int kRun = 8;

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

template <bool VEC>
__global__ void __launch_bounds__(256) deposit_runs_kernel(const double *__restrict__ x, const double *__restrict__ y,
                                                           const double *__restrict__ t, long long n, GridDev g, double qw,
                                                           double zscale, double *__restrict__ rho) {
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    const long long chunk = 32LL * kRun;
    const long long nxy = (long long)g.nx * g.ny;
    for (long long c0 = warp * chunk; c0 < n; c0 += nwarps * chunk) {
        const long long p0 = c0 + (long long)lane * kRun;
        double px_[kRun], py_[kRun], pt_[kRun];
        if (VEC && p0 + kRun <= n) {
#pragma unroll
            for (int r = 0; r < kRun; r += 2) {
                const double2 a = __ldcs(reinterpret_cast<const double2 *>(x + p0 + r));
                const double2 b = __ldcs(reinterpret_cast<const double2 *>(y + p0 + r));
                const double2 c = __ldcs(reinterpret_cast<const double2 *>(t + p0 + r));
                px_[r] = a.x, px_[r + 1] = a.y, py_[r] = b.x, py_[r + 1] = b.y, pt_[r] = c.x, pt_[r + 1] = c.y;
            }
        } else {
#pragma unroll
            for (int r = 0; r < kRun; ++r) {
                const bool live = p0 + r < n;
                px_[r] = live ? x[p0 + r] : CUDART_NAN;  // NaN => outside => contributes nothing
                py_[r] = live ? y[p0 + r] : 0.0;
                pt_[r] = live ? t[p0 + r] : 0.0;
            }
        }
        int cur = -1;
        double acc[8];
#pragma unroll
        for (int d = 0; d < 8; ++d) acc[d] = 0.0;
#pragma unroll
        for (int r = 0; r < kRun; ++r) {
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

static int env_int_grid(const char *name, int dflt) {
    const char *v = getenv(name);
    return (v && *v) ? atoi(v) : dflt;
}

int launch_deposit(Beam *b, Grid *g, double q_weight, double zscale) {
    const GridDev gd = make_grid_dev(*g);
    const int mode = env_int_grid("BT_DEPOSIT_MODE", 1);
    const int block = 256;
    if (mode == 0) {
        long long blocks = (b->n + block - 1) / block;
        const long long cap = (long long)b->num_sms * 16;
        if (blocks > cap) blocks = cap;
        deposit_atomic_kernel<<<(int)blocks, block, 0, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight, zscale, g->rho);
    } else {
        const long long per_block = (long long)block * kRun;
        long long blocks = (b->n + per_block - 1) / per_block;
        const long long cap = (long long)b->num_sms * 8;
        if (blocks > cap) blocks = cap;
        if (b->aligned16)
            deposit_runs_kernel<true><<<(int)blocks, block, 0, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight, zscale, g->rho);
        else
            deposit_runs_kernel<false><<<(int)blocks, block, 0, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight, zscale, g->rho);
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
    const int block = 256;
    long long blocks = (b->n + block - 1) / block;
    const long long cap = (long long)b->num_sms * 16;
    if (blocks > cap) blocks = cap;
    gather_kick_kernel<<<(int)blocks, block, 0, b->stream>>>(a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_gather_kick launch: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(1);
    return BT_OK;
}

}  // namespace bt
