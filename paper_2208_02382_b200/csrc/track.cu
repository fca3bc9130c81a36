// S2: the fused lattice walk.  One launch: every particle is loaded once (coalesced, 16-byte
// vector loads when aligned), every record of the launch's table is applied in registers (all
// turns x elements x slices that fit one table), and it is stored once -> 96 B of HBM traffic per
// particle per launch.  Arithmetic is pure FP64 DFMA/DMUL: every transcendental is an element
// parameter and was folded into the per-slice coefficients on the host (bt_api.cu: build_turn_table).
//
// Thread mapping: each thread owns P particles (P = 1, 2 or 4); one warp = one task of 32*P particles
// that walks the whole record table.
//
// Record table: KERNEL PARAMETER space (a __grid_constant__ struct of up to 32 764 bytes = 510 records of 64 B).
// Parameters live in constant bank 0, so -- exactly as with a __constant__ array -- the warp-uniform walk fetches every
// record word with a uniform-datapath constant load (SASS: LDCU UR, c[0x0][UR+off]) straight into a uniform register and
// uses it as the UR operand of the DFMAs: no vector-register traffic, no R2UR moves, and the dispatch is uniform
// compares + uniform branches.  Unlike a __constant__ array the table belongs to the LAUNCH: nothing on the device is
// shared between beams, streams or launches, so beams on different streams / host threads and the chunk streams of
// bt_track_host need no serialisation, and a lattice whose RF changes the reference energy simply passes a different
// table with every launch.  (Round 1 kept one 64 KiB __constant__ table per device behind a mutex and an event.)
// Measured on B200 against the alternatives (shared-memory table, global table through L1, either with
// software-prefetched records in vector registers): vector-register coefficients cost FP64 issue rate (three 64-bit
// vector operands per DFMA), and R2UR of loaded words sits on the dependency chain of every element.
// Lattices x turns longer than one table are walked in several launches (bt_api.cu plans them).
//
// Opcodes are one-hot bits, tested with a short uniform compare tree ordered by how often the kinds occur;
// the host specialises single-slice elements (no loop control), groups of five quad slices (unrolled) and runs of
// [single-slice quad, sextupole, octupole, single-slice drift] half cells (one dispatch for the whole run).
#include "bt_internal.h"

#include <stdlib.h>
#include <string.h>

namespace bt {

constexpr int kMaxBlock = 128;  // launch bound; the default block is 64 threads (fine-grained balance over SMs)

// Register budget per instantiation (128-thread blocks per SM the compiler must allow): the per-record latency
// (constant loads, compare tree, branch) is covered by other warps, so P <= 4 is held to 80 registers
// (6 warps per sub-partition).
template <int P>
constexpr int kMinBlocks = P <= 2 ? 8 : 6;

// Kernel parameters: launch geometry + the record table itself.  Two capacities, so that short lattices (configs[0]:
// 5 records) do not push 32 KiB of parameters through every launch.
template <int NREC>
struct TrackArgs {
    double *q[6];
    long long n;
    long long tail_start;  // first particle handled by the guarded P=1 blocks
    int n_full_blocks;     // blocks [0, n_full_blocks) run the unguarded P-particle path
    int n_ops;             // records of tab[] in use
    int nturns;            // passes over those records
    int pad_;
    DevOp tab[NREC];
};
static_assert(sizeof(TrackArgs<kTableRecords>) <= 32764, "kernel parameter space is 32 764 bytes");

template <int P>
struct Ptc {
    double x[P], px[P], y[P], py[P], t[P], pt[P];
};

#define BT_FORP _Pragma("unroll") for (int j = 0; j < P; ++j)

// R5: one slice of a thick quad, 9 slots (4 DMUL + 5 DFMA)
template <int P>
__device__ __forceinline__ void quad_slice(Ptc<P> &p, double c0, double c1, double c2, double c3, double c4, double c5, double c6) {
    BT_FORP {
        const double x = p.x[j], px = p.px[j], y = p.y[j], py = p.py[j];
        p.x[j] = fma(c1, px, c0 * x);
        p.px[j] = fma(c0, px, c2 * x);
        p.y[j] = fma(c4, py, c3 * y);
        p.py[j] = fma(c3, py, c5 * y);
        p.t[j] = fma(c6, p.pt[j], p.t[j]);
    }
}
// R4: 3 slots
template <int P>
__device__ __forceinline__ void drift_slice(Ptc<P> &p, double c0, double c1) {
    BT_FORP {
        p.x[j] = fma(c0, p.px[j], p.x[j]);
        p.y[j] = fma(c0, p.py[j], p.y[j]);
        p.t[j] = fma(c1, p.pt[j], p.t[j]);
    }
}
// R8, m = 3, Ks = 0: 5 slots.  ca = Kn/2, cb = Kn
template <int P>
__device__ __forceinline__ void sext_kick(Ptc<P> &p, double ca, double cb) {
    BT_FORP {
        const double x = p.x[j], y = p.y[j];
        const double re = fma(-y, y, x * x);  // Re (x+iy)^2
        const double xy = x * y;              // Im (x+iy)^2 / 2
        p.px[j] = fma(-ca, re, p.px[j]);
        p.py[j] = fma(cb, xy, p.py[j]);
    }
}
// R8, m = 4, Ks = 0: 8 slots.  c = Kn/6
template <int P>
__device__ __forceinline__ void oct_kick(Ptc<P> &p, double c) {
    BT_FORP {
        const double x = p.x[j], y = p.y[j];
        const double x2 = x * x, y2 = y * y;
        const double a = fma(-3.0, y2, x2);  // Re (x+iy)^3 = x (x^2 - 3y^2)
        const double b = fma(3.0, x2, -y2);  // Im (x+iy)^3 = y (3x^2 - y^2)
        p.px[j] = fma(-c, x * a, p.px[j]);
        p.py[j] = fma(c, y * b, p.py[j]);
    }
}

// R7 thin dipole edge: 2 slots
template <int P>
__device__ __forceinline__ void edge_kick(Ptc<P> &p, double c0, double c1) {
    BT_FORP {
        p.px[j] = fma(c0, p.x[j], p.px[j]);
        p.py[j] = fma(c1, p.y[j], p.py[j]);
    }
}
// R6 sector bend: 10 slots per slice (2 DMUL + 8 DFMA)
template <int P>
__device__ __forceinline__ void sbend_slice(Ptc<P> &p, double c0, double c1, double c2, double c3, double c4, double c5, double c6) {
    BT_FORP {
        const double x = p.x[j], px = p.px[j], pt = p.pt[j];
        p.x[j] = fma(c3, pt, fma(c1, px, c0 * x));
        p.px[j] = fma(c4, pt, fma(c0, px, c2 * x));
        p.y[j] = fma(c6, p.py[j], p.y[j]);
        // t += r51 x + r52 px + r56 pt with r51 = -r26 = -c4, r52 = -r16 = -c3
        p.t[j] = fma(c5, pt, fma(-c3, px, fma(-c4, x, p.t[j])));
    }
}
// R9 short RF, linearised: 4 slots
template <int P>
__device__ __forceinline__ void rf_kick(Ptc<P> &p, double c0, double c1) {
    BT_FORP {
        p.px[j] *= c0;
        p.py[j] *= c0;
        p.pt[j] = fma(c0, p.pt[j], c1 * p.t[j]);
    }
}
// R17 exact drift: straight line with the exact time of flight; c0 = h, c1 = 1/beta0
template <int P>
__device__ __forceinline__ void driftx_slice(Ptc<P> &p, double c0, double c1) {
    BT_FORP {
        const double px = p.px[j], py = p.py[j], pt = p.pt[j];
        const double a = fma(pt, pt, fma(-2.0 * pt, c1, 1.0)) - fma(px, px, py * py);
        const double ips = 1.0 / sqrt(a);  // p0 / p_s
        p.x[j] = fma(c0 * px, ips, p.x[j]);
        p.y[j] = fma(c0 * py, ips, p.y[j]);
        p.t[j] = fma(c0, fma(c1 - pt, ips, -c1), p.t[j]);
    }
}
// R18 sinusoidal short RF: the energy kick qV cos(k t + phi) without the expansion in t
template <int P>
__device__ __forceinline__ void rfsin_kick(Ptc<P> &p, double c0, double c1, double c2, double c3, double c4) {
    BT_FORP {
        p.px[j] *= c0;
        p.py[j] *= c0;
        p.pt[j] = fma(c1, cos(fma(c2, p.t[j], c3)) - c4, c0 * p.pt[j]);
    }
}
// R8 general order: repeated complex multiplication
template <int P>
__device__ __forceinline__ void mult_kick(Ptc<P> &p, double c0, double c1, int m) {
    BT_FORP {
        const double x = p.x[j], y = p.y[j];
        double zr = 1.0, zi = 0.0;
#pragma unroll 1
        for (int k = 1; k < m; ++k) {
            const double nr = fma(-zi, y, zr * x);
            const double ni = fma(zi, x, zr * y);
            zr = nr;
            zi = ni;
        }
        p.px[j] -= fma(-c1, zi, c0 * zr);
        p.py[j] += fma(c1, zr, c0 * zi);
    }
}

// R20 chromatic quad for ONE particle: per-particle focusing strength k/(1+delta), closed-form flow of
// H = -(1+d) + (px^2+py^2)/(2(1+d)) + k(x^2-y^2)/2 - pt/beta0.  Deliberately NOT inlined: two square roots, sincos, exp and
// a reciprocal need ~100 registers of their own; as a real call they do not weigh on the register allocation of the
// DFMA-only maps that share the kernel (inlined, the P = 4 instantiation spilled 800 bytes).
struct ChrOut {
    double x, px, y, py, t;
};
__device__ __noinline__ ChrOut quadchr_one(double x, double px, double y, double py, double t, double pt, double h, double ib, double ak,
                                           double sgn) {
    const double opd = sqrt(fma(pt, pt, fma(-2.0 * pt, ib, 1.0)));  // 1 + delta = P/p0
    double integral;
    ChrOut o;
    if (sgn == 0.0) {
        integral = fma(px, px, py * py) * h;
        o.x = fma(h / opd, px, x), o.px = px;
        o.y = fma(h / opd, py, y), o.py = py;
    } else {
        const double w = sqrt(ak / opd), a = opd * w, wh = w * h;
        double sn, cs;
        sincos(wh, &sn, &cs);
        const double ex = exp(wh), exi = 1.0 / ex;
        const double ch = 0.5 * (ex + exi), sh = 0.5 * (ex - exi);
        const bool fx = sgn > 0.0;
        const double qf = fx ? x : y, pf = fx ? px : py;
        const double qd = fx ? y : x, pd = fx ? py : px;
        const double A = pf, B = -a * qf, C = pd, D = a * qd;
        // sin(2wh) = 2 s c, sinh(2wh) = 2 sh ch
        const double IF = 0.5 * h * fma(A, A, B * B) + (fma(A, A, -B * B) * (0.5 * sn * cs) + A * B * (sn * sn)) / w;
        const double ID = 0.5 * h * fma(C, C, -D * D) + (fma(C, C, D * D) * (0.5 * sh * ch) + C * D * (sh * sh)) / w;
        integral = IF + ID;
        const double qf1 = fma(sn / a, pf, cs * qf), pf1 = fma(-a * sn, qf, cs * pf);
        const double qd1 = fma(sh / a, pd, ch * qd), pd1 = fma(a * sh, qd, ch * pd);
        o.x = fx ? qf1 : qd1, o.px = fx ? pf1 : pd1;
        o.y = fx ? qd1 : qf1, o.py = fx ? pd1 : pf1;
    }
    o.t = t + (((ib - pt) / opd) * fma(integral, 0.5 / (opd * opd), h) - h * ib);
    return o;
}

// R20 chromatic quad, one slice: a call per particle (see quadchr_one)
template <int P>
__device__ __forceinline__ void quadchr_slice(Ptc<P> &p, double h, double ib, double ak, double sgn) {
    BT_FORP {
        const ChrOut o = quadchr_one(p.x[j], p.px[j], p.y[j], p.py[j], p.t[j], p.pt[j], h, ib, ak, sgn);
        p.x[j] = o.x, p.px[j] = o.px, p.y[j] = o.y, p.py[j] = o.py, p.t[j] = o.t;
    }
}

// ---- the record at tab[e] applied to the P particles of this thread; returns how many records it consumed ----------
// NL: this instantiation also knows the non-linearised maps (R17, R18, R20).  They need square roots, sincos and exp;
// compiled into the same kernel they cost the DFMA-only maps registers (configs[1]: 2.61 -> 3.19 ms per step, measured), so
// lattices without them run the NL = false kernel, which is the linear walk exactly as before.
template <int P, bool NL>
__device__ __forceinline__ int apply(Ptc<P> &p, const DevOp *__restrict__ tab, const int e) {
    const DevOp &r = tab[e];
    const int op = r.op;
    if (op & (OP_HALFCELL | OP_QUAD5 | OP_QUAD1 | OP_QUAD)) {
        if (op & OP_HALFCELL) {
            // a run of `count` half cells [quad (one slice), sextupole, octupole, drift (one slice)]: records e, e+1 hold the
            // first one (quad coefficients; kick and drift coefficients), e+2, e+3 the second, ...  Same arithmetic and order
            // as the four maps dispatched one by one; one dispatch for the whole run.
            const int cnt = r.count;
#pragma unroll 1
            for (int s = 0; s < cnt; ++s) {
                const DevOp &qa = tab[e + 2 * s];
                const DevOp &kb = tab[e + 2 * s + 1];
                quad_slice<P>(p, qa.c[0], qa.c[1], qa.c[2], qa.c[3], qa.c[4], qa.c[5], qa.c[6]);
                sext_kick<P>(p, kb.c[0], kb.c[1]);
                oct_kick<P>(p, kb.c[2]);
                drift_slice<P>(p, kb.c[3], kb.c[4]);
            }
            return 2 * cnt;
        }
        const double c0 = r.c[0], c1 = r.c[1], c2 = r.c[2], c3 = r.c[3], c4 = r.c[4], c5 = r.c[5], c6 = r.c[6];
        if (op & OP_QUAD5) {  // count groups of five slices
            const int cnt = r.count;
#pragma unroll 1
            for (int s = 0; s < cnt; ++s) {
#pragma unroll
                for (int u = 0; u < 5; ++u) quad_slice<P>(p, c0, c1, c2, c3, c4, c5, c6);
            }
        } else if (op & OP_QUAD1) {
            quad_slice<P>(p, c0, c1, c2, c3, c4, c5, c6);
        } else {
            const int cnt = r.count;
#pragma unroll 1
            for (int s = 0; s < cnt; ++s) quad_slice<P>(p, c0, c1, c2, c3, c4, c5, c6);
        }
    } else if (op & (OP_DRIFT1 | OP_DRIFT)) {
        const double c0 = r.c[0], c1 = r.c[1];
        if (op & OP_DRIFT1) {
            drift_slice<P>(p, c0, c1);
        } else {
            const int cnt = r.count;
#pragma unroll 1
            for (int s = 0; s < cnt; ++s) drift_slice<P>(p, c0, c1);
        }
    } else if (op & (OP_SEXTOCT | OP_SEXT | OP_OCT)) {
        // OP_SEXTOCT = a sextupole kick followed by an octupole kick at the same place, in one dispatch;
        // the arithmetic is exactly the two separate kicks in order.
        if (op & (OP_SEXTOCT | OP_SEXT)) sext_kick<P>(p, r.c[0], r.c[1]);
        if (op & (OP_SEXTOCT | OP_OCT)) oct_kick<P>(p, r.c[2]);
        if (op & OP_TAILDRIFT) drift_slice<P>(p, r.c[3], r.c[4]);  // the single-slice drift that follows, same dispatch
    } else if (op & (OP_SBEND | OP_EDGE)) {
        if (op & OP_EDGE) {
            edge_kick<P>(p, r.c[0], r.c[1]);
        } else {
            const double c0 = r.c[0], c1 = r.c[1], c2 = r.c[2], c3 = r.c[3], c4 = r.c[4], c5 = r.c[5], c6 = r.c[6];
            const int cnt = r.count;
#pragma unroll 1
            for (int s = 0; s < cnt; ++s) sbend_slice<P>(p, c0, c1, c2, c3, c4, c5, c6);
        }
    } else if (op & OP_RF) {
        rf_kick<P>(p, r.c[0], r.c[1]);
    } else if (NL && (op & OP_DRIFTX)) {
        const double c0 = r.c[0], c1 = r.c[1];
        const int cnt = r.count;
#pragma unroll 1
        for (int s = 0; s < cnt; ++s) driftx_slice<P>(p, c0, c1);
    } else if (NL && (op & OP_QUADCHR)) {
        const double h = r.c[0], ib = r.c[1], ak = r.c[2], sgn = r.c[3];
        const int cnt = r.count;
#pragma unroll 1
        for (int s = 0; s < cnt; ++s) quadchr_slice<P>(p, h, ib, ak, sgn);
    } else if (NL && (op & OP_RFSIN)) {
        rfsin_kick<P>(p, r.c[0], r.c[1], r.c[2], r.c[3], r.c[4]);
    } else if (op & OP_MULT) {
        mult_kick<P>(p, r.c[0], r.c[1], r.count);
    }
    return 1;
}

template <int P, bool NL>
__device__ __forceinline__ void walk(Ptc<P> &p, const DevOp *__restrict__ tab, const int n_ops, const int nturns) {
#pragma unroll 1
    for (int turn = 0; turn < nturns; ++turn) {
#pragma unroll 1
        for (int e = 0; e < n_ops;) e += apply<P, NL>(p, tab, e);
    }
}

// ---- streaming particle access: read once, written once ------------------------------------------
__device__ __forceinline__ double2 ld_stream2(const double *p) {
    double2 v;
    asm volatile("ld.global.cs.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_stream2(double *p, double2 v) {
    asm volatile("st.global.cs.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ double ld_stream1(const double *p) {
    double v;
    asm volatile("ld.global.cs.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_stream1(double *p, double v) { asm volatile("st.global.cs.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory"); }

template <int P>
__device__ __forceinline__ void load_ptc(Ptc<P> &p, double *const (&q)[6], const int B) {
    if constexpr (P >= 2) {  // q[] already point at this thread's first pair
#pragma unroll
        for (int j = 0; j < P / 2; ++j) {
            const int off = j * 2 * B;
            double2 v;
            v = ld_stream2(q[0] + off), p.x[2 * j] = v.x, p.x[2 * j + 1] = v.y;
            v = ld_stream2(q[1] + off), p.px[2 * j] = v.x, p.px[2 * j + 1] = v.y;
            v = ld_stream2(q[2] + off), p.y[2 * j] = v.x, p.y[2 * j + 1] = v.y;
            v = ld_stream2(q[3] + off), p.py[2 * j] = v.x, p.py[2 * j + 1] = v.y;
            v = ld_stream2(q[4] + off), p.t[2 * j] = v.x, p.t[2 * j + 1] = v.y;
            v = ld_stream2(q[5] + off), p.pt[2 * j] = v.x, p.pt[2 * j + 1] = v.y;
        }
    } else {
        p.x[0] = ld_stream1(q[0]);
        p.px[0] = ld_stream1(q[1]);
        p.y[0] = ld_stream1(q[2]);
        p.py[0] = ld_stream1(q[3]);
        p.t[0] = ld_stream1(q[4]);
        p.pt[0] = ld_stream1(q[5]);
    }
}
template <int P>
__device__ __forceinline__ void store_ptc(const Ptc<P> &p, double *const (&q)[6], const int B) {
    if constexpr (P >= 2) {
#pragma unroll
        for (int j = 0; j < P / 2; ++j) {
            const int off = j * 2 * B;
            st_stream2(q[0] + off, make_double2(p.x[2 * j], p.x[2 * j + 1]));
            st_stream2(q[1] + off, make_double2(p.px[2 * j], p.px[2 * j + 1]));
            st_stream2(q[2] + off, make_double2(p.y[2 * j], p.y[2 * j + 1]));
            st_stream2(q[3] + off, make_double2(p.py[2 * j], p.py[2 * j + 1]));
            st_stream2(q[4] + off, make_double2(p.t[2 * j], p.t[2 * j + 1]));
            st_stream2(q[5] + off, make_double2(p.pt[2 * j], p.pt[2 * j + 1]));
        }
    } else {
        st_stream1(q[0], p.x[0]);
        st_stream1(q[1], p.px[0]);
        st_stream1(q[2], p.y[0]);
        st_stream1(q[3], p.py[0]);
        st_stream1(q[4], p.t[0]);
        st_stream1(q[5], p.pt[0]);
    }
}

// P particles per thread (P even: 16-byte vector access; requires 16-byte aligned arrays).
template <int P, bool NL, int NREC>
__global__ void __launch_bounds__(kMaxBlock, kMinBlocks<P>) track_kernel(const __grid_constant__ TrackArgs<NREC> a) {
    const int tid = threadIdx.x;
    const int B = blockDim.x;
    if ((int)blockIdx.x < a.n_full_blocks) {
        // ---- unguarded path: this block owns particles [blk*P*B, (blk+1)*P*B) ----
        Ptc<P> p;
        const long long first = (long long)blockIdx.x * (P * B) + (P >= 2 ? 2 * tid : tid);
        double *q[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) q[c] = a.q[c] + first;
        load_ptc<P>(p, q, B);
        walk<P, NL>(p, a.tab, a.n_ops, a.nturns);
        store_ptc<P>(p, q, B);
    } else {
        // ---- guarded tail: one particle per thread ----
        Ptc<1> p;
        const long long i = a.tail_start + (long long)((int)blockIdx.x - a.n_full_blocks) * B + tid;
        if (i >= a.n) return;
        double *q[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) q[c] = a.q[c] + i;
        load_ptc<1>(p, q, B);
        walk<1, NL>(p, a.tab, a.n_ops, a.nturns);
        store_ptc<1>(p, q, B);
    }
}

// ---- slice-step / element-step diagnostics INSIDE the walk (P:l.61 set_slice_step_diagnostics) ---------------
// The same walk, on tables built WITHOUT record fusion (one record per element, `count` slices of one kind), and after every
// slice (slice granularity) or after the last slice of every element (element granularity) each warp reduces the 27 sums
//   S_i = sum (q_i - k_i),  P_ij = sum (q_i - k_i)(q_j - k_j)   (i <= j; k = a provisional centre, moments.cu)
// of its 32*P particles and writes them as one 216-byte row: no extra pass over the particles, 96 B per particle per launch
// as in bt_track.  The reduction across lanes is a transposition through shared memory: lane L adds the 32 lanes' copies of
// value L.  diag_combine_kernel then adds the rows of one boundary in a fixed
// order (bit-reproducible) and forms mean = k + S/n, cov = P/n - (S/n)(S/n)^T.
constexpr int kDiagVals = 27;

// one slice map of the record's kind; `count` is the diagnostics walk's business
template <int P, bool NL>
__device__ __forceinline__ void apply_one_slice(Ptc<P> &p, const DevOp &r) {
    const int op = r.op;
    if (op & OP_QUAD) {
        quad_slice<P>(p, r.c[0], r.c[1], r.c[2], r.c[3], r.c[4], r.c[5], r.c[6]);
    } else if (op & OP_DRIFT) {
        drift_slice<P>(p, r.c[0], r.c[1]);
    } else if (op & (OP_SEXT | OP_OCT)) {
        if (op & OP_SEXT) sext_kick<P>(p, r.c[0], r.c[1]);
        else oct_kick<P>(p, r.c[2]);
    } else if (op & (OP_SBEND | OP_EDGE)) {
        if (op & OP_EDGE) edge_kick<P>(p, r.c[0], r.c[1]);
        else sbend_slice<P>(p, r.c[0], r.c[1], r.c[2], r.c[3], r.c[4], r.c[5], r.c[6]);
    } else if (op & OP_RF) {
        rf_kick<P>(p, r.c[0], r.c[1]);
    } else if (NL && (op & OP_DRIFTX)) {
        driftx_slice<P>(p, r.c[0], r.c[1]);
    } else if (NL && (op & OP_QUADCHR)) {
        quadchr_slice<P>(p, r.c[0], r.c[1], r.c[2], r.c[3]);
    } else if (NL && (op & OP_RFSIN)) {
        rfsin_kick<P>(p, r.c[0], r.c[1], r.c[2], r.c[3], r.c[4]);
    } else if (op & OP_MULT) {
        mult_kick<P>(p, r.c[0], r.c[1], r.count);
    }
}

template <int NREC>
struct DiagArgs {
    double *q[6];
    long long n;
    const double *centre;  // k[6], device memory (moments_centre_kernel)
    double *rows;          // [boundary][warp][27]
    long long nwarps;      // warps of the launch = rows per boundary
    int n_ops;
    int slice_gran;        // 1: a row after every slice; 0: after every element
    DevOp tab[NREC];
};
static_assert(sizeof(DiagArgs<kTableRecords>) <= 32764, "kernel parameter space is 32 764 bytes");

constexpr int kDiagPitch = 33;  // doubles per value row of a warp's transposition buffer (32 lanes + 1 pad)

template <int P>
__device__ __forceinline__ void diag_emit(const Ptc<P> &p, const double (&k)[6], const bool (&valid)[P], double *__restrict__ row,
                                          double *__restrict__ tr) {
    double v[kDiagVals];
#pragma unroll
    for (int i = 0; i < kDiagVals; ++i) v[i] = 0.0;
    BT_FORP {
        double d[6];
        d[0] = p.x[j] - k[0], d[1] = p.px[j] - k[1], d[2] = p.y[j] - k[2];
        d[3] = p.py[j] - k[3], d[4] = p.t[j] - k[4], d[5] = p.pt[j] - k[5];
        if (!valid[j]) {
#pragma unroll
            for (int c = 0; c < 6; ++c) d[c] = 0.0;
        }
        int idx = 6;
#pragma unroll
        for (int a = 0; a < 6; ++a) {
            v[a] += d[a];
#pragma unroll
            for (int b = a; b < 6; ++b) v[idx] = fma(d[a], d[b], v[idx]), ++idx;
        }
    }
    // transposition through the warp's shared buffer: every lane parks its 27 sums (conflict-free: consecutive lanes,
    // consecutive words), then lane L adds the 32 lanes' copies of value L in a fixed order (four chains for ILP) --
    // 27 STS + 32 LDS + 31 DADD per lane and boundary (a shuffle butterfly needs 62 SHFL + 124 SEL + 31 DADD)
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int i = 0; i < kDiagVals; ++i) tr[i * kDiagPitch + lane] = v[i];
    __syncwarp();
    if (lane < kDiagVals) {
        const double *src = tr + lane * kDiagPitch;
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
        for (int j = 0; j < 32; j += 4) s0 += src[j], s1 += src[j + 1], s2 += src[j + 2], s3 += src[j + 3];
        row[lane] = (s0 + s1) + (s2 + s3);
    }
    __syncwarp();
}

// The same emission with the lane reduction done by a transposing shuffle butterfly (31 exchanges of doubles leave the total of
// value L in lane L).  Used at SLICE granularity, where an emission follows every slice map and the L1 data pipe, not the
// FP64 pipe, is what the emissions load: 62 SHFL cost it less than 27 STS.64 + 32 LDS.64 (measured on configs[1], 5 300
// boundaries: 34.5 ms against 44.0 ms); at element granularity the shared-memory transposition wins (4.64 against 5.59 ms).
template <int P>
__device__ __forceinline__ void diag_emit_shfl(const Ptc<P> &p, const double (&k)[6], const bool (&valid)[P], double *__restrict__ row) {
    double v[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = 0.0;
    BT_FORP {
        double d[6];
        d[0] = p.x[j] - k[0], d[1] = p.px[j] - k[1], d[2] = p.y[j] - k[2];
        d[3] = p.py[j] - k[3], d[4] = p.t[j] - k[4], d[5] = p.pt[j] - k[5];
        if (!valid[j]) {
#pragma unroll
            for (int c = 0; c < 6; ++c) d[c] = 0.0;
        }
        int idx = 6;
#pragma unroll
        for (int a = 0; a < 6; ++a) {
            v[a] += d[a];
#pragma unroll
            for (int b = a; b < 6; ++b) v[idx] = fma(d[a], d[b], v[idx]), ++idx;
        }
    }
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {  // after the round with distance d a lane keeps the half of its values selected by its bit d
        const bool up = (lane & d) != 0;
#pragma unroll
        for (int i = 0; i < d; ++i) {
            const double send = up ? v[i] : v[i + d];
            const double keep = up ? v[i + d] : v[i];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, d);
        }
    }
    if (lane < kDiagVals) row[lane] = v[0];  // lane L holds the warp's total of value L
}

// SLICE = false (element granularity): records are applied by the regular apply() -- whole elements, five-slice quad groups
// included -- and a row follows every record marked OP_MARK (the last record of an element); SLICE = true: one slice at a
// time, a row after each.
template <int P, bool NL, int NREC, bool SLICE>
__global__ void __launch_bounds__(128, P == 8 ? 2 : P == 4 ? 3 : 4) track_diag_kernel(const __grid_constant__ DiagArgs<NREC> a) {
    const int tid = threadIdx.x, B = blockDim.x;
    const long long gw = (long long)blockIdx.x * (B >> 5) + (tid >> 5);
    const long long base = (long long)blockIdx.x * (P * B);
    // particle j of this thread (same assignment as track_kernel: pairs 2 tid, 2 tid + 1 of every 2B-particle group)
    long long idx[P];
    bool valid[P];
    BT_FORP {
        idx[j] = P >= 2 ? base + (long long)(j / 2) * 2 * B + 2 * tid + (j & 1) : base + tid;
        valid[j] = idx[j] < a.n;
    }
    Ptc<P> p;
    const bool full = base + (long long)P * B <= a.n;  // block-uniform
    if (full) {
        double *q[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) q[c] = a.q[c] + base + (P >= 2 ? 2 * tid : tid);
        load_ptc<P>(p, q, B);
    } else {
        BT_FORP {
            p.x[j] = valid[j] ? a.q[0][idx[j]] : 0.0, p.px[j] = valid[j] ? a.q[1][idx[j]] : 0.0;
            p.y[j] = valid[j] ? a.q[2][idx[j]] : 0.0, p.py[j] = valid[j] ? a.q[3][idx[j]] : 0.0;
            p.t[j] = valid[j] ? a.q[4][idx[j]] : 0.0, p.pt[j] = valid[j] ? a.q[5][idx[j]] : 0.0;
        }
    }
    double k[6];
#pragma unroll
    for (int c = 0; c < 6; ++c) k[c] = a.centre[c];
    double *row = a.rows + gw * kDiagVals;
    const long long row_stride = a.nwarps * kDiagVals;
    __shared__ double tr_all[SLICE ? 1 : 4][SLICE ? 1 : kDiagVals * kDiagPitch];  // blocks of 128 threads: one buffer per warp
    double *tr = SLICE ? tr_all[0] : tr_all[tid >> 5];
    (void)tr;
    if constexpr (SLICE) {
#pragma unroll 1
        for (int e = 0; e < a.n_ops; ++e) {
            const DevOp &r = a.tab[e];
            const int cnt = (r.op & (OP_DRIFT | OP_QUAD | OP_SBEND | OP_DRIFTX | OP_QUADCHR)) ? r.count : 1;
#pragma unroll 1
            for (int sl = 0; sl < cnt; ++sl) {
                apply_one_slice<P, NL>(p, r);
                diag_emit_shfl<P>(p, k, valid, row);
                row += row_stride;
            }
        }
    } else {
#pragma unroll 1
        for (int e = 0; e < a.n_ops;) {
            const int mark = a.tab[e].op & OP_MARK;
            e += apply<P, NL>(p, a.tab, e);
            if (mark) {
                diag_emit<P>(p, k, valid, row, tr);
                row += row_stride;
            }
        }
    }
    if (full) {
        double *q[6];
#pragma unroll
        for (int c = 0; c < 6; ++c) q[c] = a.q[c] + base + (P >= 2 ? 2 * tid : tid);
        store_ptc<P>(p, q, B);
    } else {
        BT_FORP {
            if (valid[j]) {
                a.q[0][idx[j]] = p.x[j], a.q[1][idx[j]] = p.px[j], a.q[2][idx[j]] = p.y[j];
                a.q[3][idx[j]] = p.py[j], a.q[4][idx[j]] = p.t[j], a.q[5][idx[j]] = p.pt[j];
            }
        }
    }
}

// rows of one boundary -> mean[6], cov[36]; one block per boundary, fixed summation order
__global__ void __launch_bounds__(256) diag_combine_kernel(const double *__restrict__ rows, long long nwarps, const double *__restrict__ centre,
                                                           long long n, double *__restrict__ out) {
    __shared__ double part[8][32];
    __shared__ double total[32];
    const int lane = threadIdx.x & 31, grp = threadIdx.x >> 5;
    const double *r = rows + (long long)blockIdx.x * nwarps * kDiagVals;
    double s = 0.0;
    if (lane < kDiagVals)
        for (long long w = grp; w < nwarps; w += 8) s += r[w * kDiagVals + lane];
    part[grp][lane] = s;
    __syncthreads();
    if (threadIdx.x < 32) {
        double t = 0.0;
#pragma unroll
        for (int g = 0; g < 8; ++g) t += part[g][threadIdx.x];
        total[threadIdx.x] = t;
    }
    __syncthreads();
    const double inv_n = 1.0 / (double)n;
    double *o = out + (long long)blockIdx.x * 42;
    if (threadIdx.x < 6) o[threadIdx.x] = centre[threadIdx.x] + total[threadIdx.x] * inv_n;
    if (threadIdx.x < 36) {
        const int i = threadIdx.x / 6, j = threadIdx.x % 6;
        const int lo = i < j ? i : j, hi = i < j ? j : i;
        const int idx = 6 + lo * 6 - lo * (lo - 1) / 2 + (hi - lo);  // position of (lo, hi) in the packed upper triangle
        o[6 + threadIdx.x] = total[idx] * inv_n - (total[lo] * inv_n) * (total[hi] * inv_n);
    }
}

template <int P, bool NL, int NREC>
static cudaError_t launch_one(const TrackArgs<NREC> &a, int grid, int block, cudaStream_t stream) {
    track_kernel<P, NL, NREC><<<grid, block, 0, stream>>>(a);
    return cudaGetLastError();
}

template <int NREC>
static cudaError_t launch_sized(TrackArgs<NREC> &a, const DevOp *h_table, int n_ops, int P, bool nl, int grid, int block, cudaStream_t stream) {
    memcpy(a.tab, h_table, (size_t)n_ops * sizeof(DevOp));
    switch (P) {
        case 4: return nl ? launch_one<4, true, NREC>(a, grid, block, stream) : launch_one<4, false, NREC>(a, grid, block, stream);
        case 2: return nl ? launch_one<2, true, NREC>(a, grid, block, stream) : launch_one<2, false, NREC>(a, grid, block, stream);
        default: return nl ? launch_one<1, true, NREC>(a, grid, block, stream) : launch_one<1, false, NREC>(a, grid, block, stream);
    }
}

int launch_track(Beam *b, const DevOp *h_table, int32_t n_ops, int32_t nturns, double slots_per_record) {
    if (n_ops < 1 || n_ops > kTableRecords) return fail(BT_ERR_INVALID, "launch_track: table size");
    // ---- launch geometry -------------------------------------------------------------------------
    // One warp = one task of 32*P particles walking the whole table.  P amortises the interpreter's per-record
    // work (what matters when records are short: slots_per_record small) but coarsens the tasks: the last tasks
    // of a launch run with few warps per SM sub-partition and cannot fill the FP64 pipe, so with long records
    // (per-record work negligible) P is lowered until every sub-partition gets >= 24 tasks.  Measured on B200:
    // config 1 (10^6 particles, 92 slots/record) 0.913 of the FP64 roofline at P = 4, 0.945 at P = 2; config 3
    // (12 slots/record) 0.83 at P = 4, 0.76 at P = 2.  Small blocks keep the tasks balanced over SMs.
    const long long n = b->range ? b->range->n : b->n;
    const long long off = b->range ? b->range->off : 0;
    const long long geom_n = b->range ? b->range->geom_n : b->n;  // chunks of one bunch run concurrently on several streams
    cudaStream_t stream = b->range ? b->range->stream : b->stream;
    const int sms = b->num_sms > 0 ? b->num_sms : 148;
    const long long sched = (long long)sms * 4;
    auto tasks = [&](int p) { return geom_n / (32LL * p) / sched; };  // tasks per sub-partition
    int P = 1;
    if (b->aligned16) {
        if (slots_per_record < 40.0) P = tasks(4) >= 4 ? 4 : tasks(2) >= 4 ? 2 : 1;
        else P = tasks(4) >= 24 ? 4 : tasks(2) >= 12 ? 2 : 1;
    }
    int block = 64;
    while (block > 32 && geom_n / ((long long)P * block) < 2LL * sms) block >>= 1;
    P = knob(KNOB_TRACK_PPT, P);
    block = knob(KNOB_TRACK_BLOCK, block);
    if (!(P == 1 || ((P == 2 || P == 4) && b->aligned16)))
        return fail(BT_ERR_INVALID, "knob track_ppt must be 1, 2 or 4 (2, 4 need 16-byte aligned arrays)");
    if (block < 32 || block > kMaxBlock || (block & 31)) return fail(BT_ERR_INVALID, "knob track_block must be a multiple of 32 in [32,128]");

    const long long per_block = (long long)P * block;
    const long long full = n / per_block;
    const long long tail_start = full * per_block;
    const long long rem = n - tail_start;
    const long long grid_ll = full + (rem + block - 1) / block;
    if (grid_ll > 0x7fffffffLL) return fail(BT_ERR_UNSUPPORTED, "bt_track: grid too large");
    const int grid = (int)grid_ll;
    bool nl = false;  // any non-linearised record in this table?
    for (int32_t e = 0; e < n_ops; ++e) nl = nl || (h_table[e].op & (OP_DRIFTX | OP_RFSIN | OP_QUADCHR));

    auto fill = [&](auto &a) {
        for (int c = 0; c < 6; ++c) a.q[c] = b->q[c] + off;
        a.n = n;
        a.tail_start = tail_start;
        a.n_full_blocks = (int)full;
        a.n_ops = n_ops;
        a.nturns = nturns;
        a.pad_ = 0;
    };
    cudaError_t e;
    if (n_ops <= kTableRecordsSmall) {
        TrackArgs<kTableRecordsSmall> a;
        fill(a);
        e = launch_sized(a, h_table, n_ops, P, nl, grid, block, stream);
    } else {
        TrackArgs<kTableRecords> a;
        fill(a);
        e = launch_sized(a, h_table, n_ops, P, nl, grid, block, stream);
    }
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_track launch: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(1);
    b->last_launch.grid = grid;
    b->last_launch.block = block;
    b->last_launch.ppt = P;
    b->last_launch.smem = 0;
    b->last_launch.launches += 1;
    return BT_OK;
}

// ---- diagnostics walk: one launch over `n_ops` un-fused records, rows for `nb` boundaries, then their combination ----------
int diag_warps(const Beam *b, int *P_out, int *block_out) {
    // The lane reduction and the 216-byte row are per warp and boundary, so they are amortised over the 32 P particles of a
    // warp: P = 8 where the bunch still fills the machine (configs[1], 10^6 particles: element granularity 1.77 -> 1.69 x the
    // plain walk, slice granularity 10.4 -> 8.7 x, rows 834 -> 417 MB; P = 2 and 1 measured 2.04 / 3.51 x and 15.2 / 27.2 x)
    int P = !b->aligned16 ? 1 : b->n >= 524288 ? 8 : b->n >= 65536 ? 4 : 1;
    P = knob(KNOB_TRACK_PPT, P);
    if (P != 1 && !(b->aligned16 && (P == 2 || P == 4 || P == 8))) P = 1;
    int block = knob(KNOB_TRACK_BLOCK, 128);
    if (block != 64 && block != 128) block = 128;
    *P_out = P;
    *block_out = block;
    const long long per_block = (long long)P * block;
    return (int)((b->n + per_block - 1) / per_block) * (block / 32);
}

template <int P, int NREC>
static cudaError_t launch_diag_p(const DiagArgs<NREC> &a, bool nl, bool slice, int grid, int block, cudaStream_t s) {
    if (slice) {
        if (nl) track_diag_kernel<P, true, NREC, true><<<grid, block, 0, s>>>(a);
        else track_diag_kernel<P, false, NREC, true><<<grid, block, 0, s>>>(a);
    } else {
        if (nl) track_diag_kernel<P, true, NREC, false><<<grid, block, 0, s>>>(a);
        else track_diag_kernel<P, false, NREC, false><<<grid, block, 0, s>>>(a);
    }
    return cudaGetLastError();
}

template <int NREC>
static cudaError_t launch_diag_sized(DiagArgs<NREC> &a, const DevOp *h_table, int n_ops, int P, bool nl, int grid, int block, cudaStream_t s) {
    memcpy(a.tab, h_table, (size_t)n_ops * sizeof(DevOp));
    return P == 8 ? launch_diag_p<8, NREC>(a, nl, a.slice_gran != 0, grid, block, s)
         : P == 4 ? launch_diag_p<4, NREC>(a, nl, a.slice_gran != 0, grid, block, s)
         : P == 2 ? launch_diag_p<2, NREC>(a, nl, a.slice_gran != 0, grid, block, s)
                  : launch_diag_p<1, NREC>(a, nl, a.slice_gran != 0, grid, block, s);
}

int launch_track_diag(Beam *b, const DevOp *h_table, int32_t n_ops, int slice_gran, int nb, const double *centre, double *rows, double *out) {
    if (n_ops < 1 || n_ops > kTableRecords) return fail(BT_ERR_INVALID, "launch_track_diag: table size");
    int P, block;
    const long long nwarps = diag_warps(b, &P, &block);
    const int grid = (int)(nwarps / (block / 32));
    bool nl = false;
    for (int32_t e = 0; e < n_ops; ++e) nl = nl || (h_table[e].op & (OP_DRIFTX | OP_RFSIN | OP_QUADCHR));
    auto fill = [&](auto &a) {
        for (int c = 0; c < 6; ++c) a.q[c] = b->q[c];
        a.n = b->n;
        a.centre = centre;
        a.rows = rows;
        a.nwarps = nwarps;
        a.n_ops = n_ops;
        a.slice_gran = slice_gran;
    };
    cudaError_t e;
    if (n_ops <= kTableRecordsSmall) {
        DiagArgs<kTableRecordsSmall> a;
        fill(a);
        e = launch_diag_sized(a, h_table, n_ops, P, nl, grid, block, b->stream);
    } else {
        DiagArgs<kTableRecords> a;
        fill(a);
        e = launch_diag_sized(a, h_table, n_ops, P, nl, grid, block, b->stream);
    }
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_track_diagnostics launch: ") + cudaGetErrorString(e));
    if (nb > 0) diag_combine_kernel<<<nb, 256, 0, b->stream>>>(rows, nwarps, centre, b->n, out);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_track_diagnostics combine: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(2);
    b->last_launch.grid = grid;
    b->last_launch.block = block;
    b->last_launch.ppt = P;
    b->last_launch.launches += 1;
    return BT_OK;
}

}  // namespace bt
