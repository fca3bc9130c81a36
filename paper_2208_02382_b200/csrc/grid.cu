// S4-S7: particle-grid kernels -- CIC deposit and trilinear gather + kick (+ adjacent drifts).
//
// Canonical index/weights (R11), identical expression on every path so that only the summation
// order of the deposit differs from the definition:
//   u = (q - lo) * inv_d   (one rounded subtract, one rounded multiply; explicit _rn intrinsics so
//                           that nvcc can never contract zscale*t - lo into an FMA)
//   i = floor(u), w1 = u - i (exact), w0 = 1 - w1 ; node weight (wx*wy)*wz.
// Inside iff 0 <= i <= n-2 on all axes, tested as (u >= 0 && u < n-1) so NaN is outside (R13).
#include "bt_internal.h"

#include <stdlib.h>

namespace bt {

struct GridDev {
    double lo[3], inv_d[3];
    double umax[3];  // (double)(n-1)
    int nx, ny, nz;
};

static GridDev make_grid_dev(const Grid &g) {
    GridDev d;
    for (int a = 0; a < 3; ++a) {
        d.lo[a] = g.lo[a];
        d.inv_d[a] = g.inv_d[a];
    }
    d.umax[0] = (double)(g.nx - 1);
    d.umax[1] = (double)(g.ny - 1);
    d.umax[2] = (double)(g.nz - 1);
    d.nx = g.nx;
    d.ny = g.ny;
    d.nz = g.nz;
    return d;
}

struct Cic {
    int i, j, k;
    double wx1, wy1, wz1;
};

__device__ __forceinline__ bool cic_axis(double q, double lo, double inv_d, double umax, int &i, double &w1) {
    const double u = __dmul_rn(__dsub_rn(q, lo), inv_d);
    const bool in = (u >= 0.0) && (u < umax);
    const double fl = floor(u);
    i = in ? __double2int_rd(u) : 0;
    w1 = __dsub_rn(u, fl);
    return in;
}

__device__ __forceinline__ bool cic_locate(const GridDev &g, double x, double y, double t, double zscale, Cic &c) {
    const double zeta = __dmul_rn(zscale, t);
    const bool ix = cic_axis(x, g.lo[0], g.inv_d[0], g.umax[0], c.i, c.wx1);
    const bool iy = cic_axis(y, g.lo[1], g.inv_d[1], g.umax[1], c.j, c.wy1);
    const bool iz = cic_axis(zeta, g.lo[2], g.inv_d[2], g.umax[2], c.k, c.wz1);
    return ix && iy && iz;
}

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

int launch_deposit(Beam *b, Grid *g, double q_weight, double zscale) {
    const GridDev gd = make_grid_dev(*g);
    const int block = 256;
    long long blocks = (b->n + block - 1) / block;
    const long long cap = (long long)b->num_sms * 16;
    if (blocks > cap) blocks = cap;
    deposit_atomic_kernel<<<(int)blocks, block, 0, b->stream>>>(b->q[0], b->q[2], b->q[4], b->n, gd, q_weight, zscale, g->rho);
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
    double pad;
    asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(ex), "=d"(ey), "=d"(ez), "=d"(pad) : "l"(f));
    (void)pad;
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
