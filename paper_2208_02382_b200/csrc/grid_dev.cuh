// Device-side grid description and the canonical CIC index/weights (R11, R13), shared by grid.cu and sort.cu.
//   u = (q - lo) * inv_d   (one rounded subtract, one rounded multiply; explicit _rn intrinsics so that nvcc
//                           can never contract zscale*t - lo into an FMA)
//   i = floor(u), w1 = u - i (exact), w0 = 1 - w1 ; node weight (wx*wy)*wz.
// Inside iff 0 <= i <= n-2 on all axes, tested as (u >= 0 && u < n-1) so NaN is outside.
#pragma once
#include "bt_internal.h"

namespace bt {

struct GridDev {
    double lo[3], inv_d[3];
    int nm1[3];  // n - 1 per axis
    int nx, ny, nz;
};

static inline GridDev make_grid_dev(const Grid &g) {
    GridDev d;
    for (int a = 0; a < 3; ++a) {
        d.lo[a] = g.lo[a];
        d.inv_d[a] = g.inv_d[a];
    }
    d.nm1[0] = g.nx - 1;
    d.nm1[1] = g.ny - 1;
    d.nm1[2] = g.nz - 1;
    d.nx = g.nx;
    d.ny = g.ny;
    d.nz = g.nz;
    return d;
}

struct Cic {
    int i, j, k;
    double wx1, wy1, wz1;
};

// floor(u) without the conversion pipe: for 0 <= u < 2^32, u + 1.5*2^52 rounded toward -inf is exactly
// 1.5*2^52 + floor(u) (the ulp there is 1): its HIGH word is that of the magic constant and its low mantissa word is
// floor(u) as an integer; subtracting the constant back is exact.  Two DADDs on the FP64 pipe instead of FRND.F64 +
// F2I.F64 (quarter-rate conversions).  The range test is done on those two words with integer compares (no DSETP on the
// FP64 pipe): u < 0 (floor(u) <= -1 borrows from the high word), u >= 2^32, Inf and NaN all change the high word, so
//   inside  <=>  hi == hi(magic)  &&  (unsigned)floor(u) < n - 1        <=>  u >= 0 && u < n-1   (R13; -0.0 is inside).
// The index of an outside particle is whatever the low word holds and must not be used.
constexpr int kMagicHi = 0x43380000;
__device__ __forceinline__ bool cic_axis(double q, double lo, double inv_d, int nm1, int &i, double &w1) {
    const double kMagic = 6755399441055744.0;  // 1.5 * 2^52 = 0x4338000000000000
    const double u = __dmul_rn(__dsub_rn(q, lo), inv_d);
    const double tt = __dadd_rd(u, kMagic);
    i = __double2loint(tt);
    w1 = __dsub_rn(u, __dsub_rn(tt, kMagic));
    return (__double2hiint(tt) == kMagicHi) && ((unsigned)i < (unsigned)nm1);
}

__device__ __forceinline__ bool cic_locate(const GridDev &g, double x, double y, double t, double zscale, Cic &c) {
    const double zeta = __dmul_rn(zscale, t);
    const bool ix = cic_axis(x, g.lo[0], g.inv_d[0], g.nm1[0], c.i, c.wx1);
    const bool iy = cic_axis(y, g.lo[1], g.inv_d[1], g.nm1[1], c.j, c.wy1);
    const bool iz = cic_axis(zeta, g.lo[2], g.inv_d[2], g.nm1[2], c.k, c.wz1);
    return ix && iy && iz;
}

// ---- order-2 shape (reading R16, quadratic B-spline; P:l.60 set_particle_shape(2)) ---------------------------------
//   v = u + 0.5, j = floor(v) (nearest node), delta = u - j; nodes j-1, j, j+1 carry
//   (1/2)(1/2 - delta)^2, 3/4 - delta^2, (1/2)(1/2 + delta)^2, every operation rounded once in this order.
// Inside iff 1 <= j <= n-2, tested as (v >= 1 && v < n-1).  The struct holds the BASE node j-1 and delta.
__device__ __forceinline__ bool tsc_axis(double q, double lo, double inv_d, int nm1, int &base, double &delta) {
    const double kMagic = 6755399441055744.0;  // 1.5 * 2^52, see cic_axis
    const double u = __dmul_rn(__dsub_rn(q, lo), inv_d);
    const double v = __dadd_rn(u, 0.5);
    const double tt = __dadd_rd(v, kMagic);
    base = __double2loint(tt) - 1;
    delta = __dsub_rn(u, __dsub_rn(tt, kMagic));
    return (__double2hiint(tt) == kMagicHi) && ((unsigned)base < (unsigned)(nm1 - 1));  // 1 <= floor(v) <= n-2
}

// Generic view used by the templated kernels: (i, j, k) = lowest node of the stencil, (wx1, wy1, wz1) = the per-axis
// fraction the weights are built from (order 1: w1 of R11; order 2: delta of R16).
template <int ORDER>
__device__ __forceinline__ bool shape_locate(const GridDev &g, double x, double y, double t, double zscale, Cic &c) {
    if (ORDER == 1) return cic_locate(g, x, y, t, zscale, c);
    const double zeta = __dmul_rn(zscale, t);
    const bool ix = tsc_axis(x, g.lo[0], g.inv_d[0], g.nm1[0], c.i, c.wx1);
    const bool iy = tsc_axis(y, g.lo[1], g.inv_d[1], g.nm1[1], c.j, c.wy1);
    const bool iz = tsc_axis(zeta, g.lo[2], g.inv_d[2], g.nm1[2], c.k, c.wz1);
    return ix && iy && iz;
}

template <int ORDER>
__device__ __forceinline__ void axis_weights(double f, double (&w)[ORDER + 1]) {
    if (ORDER == 1) {
        w[0] = __dsub_rn(1.0, f);
        w[1] = f;
    } else {
        const double a = __dsub_rn(0.5, f), b = __dadd_rn(0.5, f);
        w[0] = __dmul_rn(0.5, __dmul_rn(a, a));
        w[1] = __dsub_rn(0.75, __dmul_rn(f, f));
        w[ORDER] = __dmul_rn(0.5, __dmul_rn(b, b));
    }
}

// (wx*wy)*wz for the (ORDER+1)^3 nodes of the stencil (no q_weight: the deposit scales a run's sum once, at the flush)
template <int ORDER>
__device__ __forceinline__ void node_weights_unscaled(const Cic &c, double (&w)[(ORDER + 1) * (ORDER + 1) * (ORDER + 1)]) {
    constexpr int NW = ORDER + 1;
    double wx[NW], wy[NW], wz[NW];
    axis_weights<ORDER>(c.wx1, wx);
    axis_weights<ORDER>(c.wy1, wy);
    axis_weights<ORDER>(c.wz1, wz);
#pragma unroll
    for (int dy = 0; dy < NW; ++dy)
#pragma unroll
        for (int dx = 0; dx < NW; ++dx) {
            const double wxy = __dmul_rn(wx[dx], wy[dy]);
#pragma unroll
            for (int dz = 0; dz < NW; ++dz) w[(dz * NW + dy) * NW + dx] = __dmul_rn(wxy, wz[dz]);
        }
}

// q_weight * ((wx*wy)*wz) for the (ORDER+1)^3 nodes of the stencil, dz outermost, dx innermost
template <int ORDER>
__device__ __forceinline__ void node_weights(const Cic &c, double qw, double (&w)[(ORDER + 1) * (ORDER + 1) * (ORDER + 1)]) {
    constexpr int NW = ORDER + 1;
    double wx[NW], wy[NW], wz[NW];
    axis_weights<ORDER>(c.wx1, wx);
    axis_weights<ORDER>(c.wy1, wy);
    axis_weights<ORDER>(c.wz1, wz);
#pragma unroll
    for (int dy = 0; dy < NW; ++dy)
#pragma unroll
        for (int dx = 0; dx < NW; ++dx) {
            const double wxy = __dmul_rn(wx[dx], wy[dy]);
#pragma unroll
            for (int dz = 0; dz < NW; ++dz) w[(dz * NW + dy) * NW + dx] = __dmul_rn(qw, __dmul_rn(wxy, wz[dz]));
        }
}

}  // namespace bt
