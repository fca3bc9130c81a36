// S2: the fused lattice walk.  One launch: every particle is loaded once (coalesced, 16-byte
// vector loads when aligned), all turns x elements x slices are applied in registers, and it is
// stored once -> 96 B of HBM traffic per particle per launch.  Arithmetic is pure FP64
// DFMA/DMUL: every transcendental is an element parameter and was folded into the per-slice
// coefficients on the host (bt_api.cu: build_turn_table).
//
// Thread mapping: each thread owns P particles (P = 1, 2 or 4).  The op table is warp-uniform, so
// the interpreter overhead (header load, dispatch, coefficient loads, loop control) is paid once
// per warp-instruction stream and amortised over P particles; with the FP64 pipe accepting one
// warp-instruction every second issue cycle of an SM sub-partition, P = 4 leaves that overhead
// hidden behind the DFMA stream.  The P independent particles also give the ILP that covers the
// DFMA latency at low occupancy.
//
// Op table source: shared memory (staged per CTA, re-staged per turn when an RF cavity changes the
// reference energy) when it fits, else global memory through the read-only path.
#include "bt_internal.h"

#include <stdlib.h>

namespace bt {

constexpr int kMaxBlock = 128;

struct TrackArgs {
    double *q[6];
    const DevOp *table;
    long long n;
    long long tail_start;  // first particle handled by the guarded P=1 blocks
    int n_full_blocks;     // blocks [0, n_full_blocks) run the unguarded P-particle path
    int n_ops;
    int nturns;
    int turn_stride;  // DevOps between consecutive turns' tables (0: same table every turn)
};

// ---- table access -------------------------------------------------------------------------------
template <bool SMEM>
struct Tab;

template <>
struct Tab<true> {
    uint32_t base;  // shared-space address
    __device__ __forceinline__ void hdr(int e, int &op, int &ns, double &c0) const {
        uint32_t a, b, lo, hi;
        asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(a), "=r"(b), "=r"(lo), "=r"(hi) : "r"(base + e * 64));
        op = (int)a;
        ns = (int)b;
        c0 = __hiloint2double((int)hi, (int)lo);
    }
    // k = 1,2,3 -> (c[2k-1], c[2k])
    __device__ __forceinline__ void pair(int e, int k, double &u, double &v) const {
        asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(u), "=d"(v) : "r"(base + e * 64 + k * 16));
    }
};

template <>
struct Tab<false> {
    const char *base;
    __device__ __forceinline__ void hdr(int e, int &op, int &ns, double &c0) const {
        uint32_t a, b, lo, hi;
        asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(a), "=r"(b), "=r"(lo), "=r"(hi) : "l"(base + (size_t)e * 64));
        op = (int)a;
        ns = (int)b;
        c0 = __hiloint2double((int)hi, (int)lo);
    }
    __device__ __forceinline__ void pair(int e, int k, double &u, double &v) const {
        asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(u), "=d"(v) : "l"(base + (size_t)e * 64 + k * 16));
    }
};

template <int P>
struct Ptc {
    double x[P], px[P], y[P], py[P], t[P], pt[P];
};

// ---- one pass over the op table (one turn) -------------------------------------------------------
template <int P, bool SMEM>
__device__ __forceinline__ void walk_turn(Ptc<P> &p, const Tab<SMEM> tab, const int n_ops) {
#pragma unroll 1
    for (int e = 0; e < n_ops; ++e) {
        int op, ns;
        double c0;
        tab.hdr(e, op, ns, c0);
        switch (op) {
            case OP_DRIFT: {  // R4: 3 slots
                double c1, c2;
                tab.pair(e, 1, c1, c2);
#pragma unroll 1
                for (int s = 0; s < ns; ++s) {
#pragma unroll
                    for (int j = 0; j < P; ++j) {
                        p.x[j] = fma(c0, p.px[j], p.x[j]);
                        p.y[j] = fma(c0, p.py[j], p.y[j]);
                        p.t[j] = fma(c1, p.pt[j], p.t[j]);
                    }
                }
                break;
            }
            case OP_QUAD: {  // R5: 9 slots (4 DMUL + 5 DFMA)
                double c1, c2, c3, c4, c5, c6;
                tab.pair(e, 1, c1, c2);
                tab.pair(e, 2, c3, c4);
                tab.pair(e, 3, c5, c6);
#pragma unroll 5
                for (int s = 0; s < ns; ++s) {
#pragma unroll
                    for (int j = 0; j < P; ++j) {
                        const double x = p.x[j], px = p.px[j], y = p.y[j], py = p.py[j];
                        p.x[j] = fma(c1, px, c0 * x);
                        p.px[j] = fma(c0, px, c2 * x);
                        p.y[j] = fma(c4, py, c3 * y);
                        p.py[j] = fma(c3, py, c5 * y);
                        p.t[j] = fma(c6, p.pt[j], p.t[j]);
                    }
                }
                break;
            }
            case OP_SBEND: {  // R6: 10 slots (2 DMUL + 8 DFMA)
                double c1, c2, c3, c4, c5, c6;
                tab.pair(e, 1, c1, c2);
                tab.pair(e, 2, c3, c4);
                tab.pair(e, 3, c5, c6);
#pragma unroll 2
                for (int s = 0; s < ns; ++s) {
#pragma unroll
                    for (int j = 0; j < P; ++j) {
                        const double x = p.x[j], px = p.px[j], pt = p.pt[j];
                        p.x[j] = fma(c3, pt, fma(c1, px, c0 * x));
                        p.px[j] = fma(c4, pt, fma(c0, px, c2 * x));
                        p.y[j] = fma(c6, p.py[j], p.y[j]);
                        // t += r51 x + r52 px + r56 pt with r51 = -r26 = -c4, r52 = -r16 = -c3
                        p.t[j] = fma(c5, pt, fma(-c3, px, fma(-c4, x, p.t[j])));
                    }
                }
                break;
            }
            case OP_EDGE: {  // R7: 2 slots
                double c1, c2;
                tab.pair(e, 1, c1, c2);
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    p.px[j] = fma(c0, p.x[j], p.px[j]);
                    p.py[j] = fma(c1, p.y[j], p.py[j]);
                }
                break;
            }
            case OP_SEXT: {  // R8, m = 3, Ks = 0: 5 slots
                double c1, c2;
                tab.pair(e, 1, c1, c2);
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    const double x = p.x[j], y = p.y[j];
                    const double re = fma(-y, y, x * x);  // Re (x+iy)^2
                    const double xy = x * y;              // Im (x+iy)^2 / 2
                    p.px[j] = fma(-c0, re, p.px[j]);
                    p.py[j] = fma(c1, xy, p.py[j]);
                }
                break;
            }
            case OP_OCT: {  // R8, m = 4, Ks = 0: 8 slots
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    const double x = p.x[j], y = p.y[j];
                    const double x2 = x * x, y2 = y * y;
                    const double a = fma(-3.0, y2, x2);  // Re (x+iy)^3 = x (x^2 - 3y^2)
                    const double b = fma(3.0, x2, -y2);  // Im (x+iy)^3 = y (3x^2 - y^2)
                    p.px[j] = fma(-c0, x * a, p.px[j]);
                    p.py[j] = fma(c0, y * b, p.py[j]);
                }
                break;
            }
            case OP_MULT: {  // R8 general order: repeated complex multiplication
                double c1, c2;
                tab.pair(e, 1, c1, c2);
                const int m = (int)c0;
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    const double x = p.x[j], y = p.y[j];
                    double zr = 1.0, zi = 0.0;
                    for (int k = 1; k < m; ++k) {
                        const double nr = fma(-zi, y, zr * x);
                        const double ni = fma(zi, x, zr * y);
                        zr = nr;
                        zi = ni;
                    }
                    p.px[j] -= fma(-c2, zi, c1 * zr);
                    p.py[j] += fma(c2, zr, c1 * zi);
                }
                break;
            }
            case OP_RF: {  // R9: 4 slots
                double c1, c2;
                tab.pair(e, 1, c1, c2);
#pragma unroll
                for (int j = 0; j < P; ++j) {
                    p.px[j] *= c0;
                    p.py[j] *= c0;
                    p.pt[j] = fma(c0, p.pt[j], c1 * p.t[j]);
                }
                break;
            }
            default:
                break;
        }
    }
}

// ---- streaming particle access: read once, written once -> keep them out of the way of the table --
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

template <int P, bool SMEM>
__device__ __forceinline__ void run_turns(Ptc<P> &p, const TrackArgs &a, uint32_t smem_addr, uint4 *smem_ptr) {
#pragma unroll 1
    for (int turn = 0; turn < a.nturns; ++turn) {
        const DevOp *gt = a.table + (size_t)turn * a.turn_stride;
        if constexpr (SMEM) {
            if (turn == 0 || a.turn_stride != 0) {
                if (turn != 0) __syncthreads();  // everyone is done with the previous turn's table
                const uint4 *src = reinterpret_cast<const uint4 *>(gt);
                for (int i = threadIdx.x; i < a.n_ops * 4; i += blockDim.x) smem_ptr[i] = __ldg(src + i);
                __syncthreads();
            }
            Tab<true> tab{smem_addr};
            walk_turn<P, true>(p, tab, a.n_ops);
        } else {
            Tab<false> tab{reinterpret_cast<const char *>(gt)};
            walk_turn<P, false>(p, tab, a.n_ops);
        }
    }
}

// P particles per thread (P even: 16-byte vector access; requires 16-byte aligned arrays).
template <int P, bool SMEM>
__global__ void __launch_bounds__(kMaxBlock) track_kernel(const __grid_constant__ TrackArgs a) {
    extern __shared__ uint4 smem_tab[];
    const uint32_t smem_addr = (uint32_t)__cvta_generic_to_shared(smem_tab);
    const int tid = threadIdx.x;
    const int B = blockDim.x;

    if ((int)blockIdx.x < a.n_full_blocks) {
        // ---- unguarded path: this block owns particles [blk*P*B, (blk+1)*P*B) ----
        Ptc<P> p;
        const long long base = (long long)blockIdx.x * (P * B);
        if constexpr (P >= 2) {
            double *q[6];
#pragma unroll
            for (int c = 0; c < 6; ++c) q[c] = a.q[c] + base + 2 * tid;
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
            run_turns<P, SMEM>(p, a, smem_addr, smem_tab);
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
            const long long i = base + tid;
            p.x[0] = ld_stream1(a.q[0] + i);
            p.px[0] = ld_stream1(a.q[1] + i);
            p.y[0] = ld_stream1(a.q[2] + i);
            p.py[0] = ld_stream1(a.q[3] + i);
            p.t[0] = ld_stream1(a.q[4] + i);
            p.pt[0] = ld_stream1(a.q[5] + i);
            run_turns<P, SMEM>(p, a, smem_addr, smem_tab);
            st_stream1(a.q[0] + i, p.x[0]);
            st_stream1(a.q[1] + i, p.px[0]);
            st_stream1(a.q[2] + i, p.y[0]);
            st_stream1(a.q[3] + i, p.py[0]);
            st_stream1(a.q[4] + i, p.t[0]);
            st_stream1(a.q[5] + i, p.pt[0]);
        }
    } else {
        // ---- guarded tail: one particle per thread ----
        Ptc<1> p;
        const long long i = a.tail_start + (long long)((int)blockIdx.x - a.n_full_blocks) * B + tid;
        const bool live = i < a.n;
        p.x[0] = live ? ld_stream1(a.q[0] + i) : 0.0;
        p.px[0] = live ? ld_stream1(a.q[1] + i) : 0.0;
        p.y[0] = live ? ld_stream1(a.q[2] + i) : 0.0;
        p.py[0] = live ? ld_stream1(a.q[3] + i) : 0.0;
        p.t[0] = live ? ld_stream1(a.q[4] + i) : 0.0;
        p.pt[0] = live ? ld_stream1(a.q[5] + i) : 0.0;
        run_turns<1, SMEM>(p, a, smem_addr, smem_tab);  // every thread walks: the table staging has barriers
        if (live) {
            st_stream1(a.q[0] + i, p.x[0]);
            st_stream1(a.q[1] + i, p.px[0]);
            st_stream1(a.q[2] + i, p.y[0]);
            st_stream1(a.q[3] + i, p.py[0]);
            st_stream1(a.q[4] + i, p.t[0]);
            st_stream1(a.q[5] + i, p.pt[0]);
        }
    }
}

static int env_int(const char *name, int dflt) {
    const char *v = getenv(name);
    return (v && *v) ? atoi(v) : dflt;
}

template <int P, bool SMEM>
static cudaError_t do_launch(const TrackArgs &a, int grid, int block, size_t smem, cudaStream_t s) {
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(track_kernel<P, SMEM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    track_kernel<P, SMEM><<<grid, block, smem, s>>>(a);
    return cudaGetLastError();
}

int launch_track(Beam *b, const DevOp *d_table, int32_t n_ops, int32_t nturns, int32_t turn_stride) {
    // ---- launch geometry -------------------------------------------------------------------------
    // Enough threads to give every SM sub-partition >= 2 warps decides P; small bunches shrink the block
    // so that the grid still covers all SMs (config 0: 10^4 particles is latency-bound whatever we do).
    const long long n = b->n;
    const int sms = b->num_sms > 0 ? b->num_sms : 148;
    int P = 1;
    const long long per = n / ((long long)sms * 8 * 32);
    if (per >= 4) P = 4;
    else if (per >= 2) P = 2;
    if (!b->aligned16) P = 1;
    int block = kMaxBlock;
    while (block > 32 && n / ((long long)P * block) < 2LL * sms) block >>= 1;
    P = env_int("BT_TRACK_PPT", P);
    block = env_int("BT_TRACK_BLOCK", block);
    if (!(P == 1 || ((P == 2 || P == 4) && b->aligned16))) return fail(BT_ERR_INVALID, "BT_TRACK_PPT must be 1, 2 or 4 (2, 4 need 16-byte aligned arrays)");
    if (block < 32 || block > kMaxBlock || (block & 31)) return fail(BT_ERR_INVALID, "BT_TRACK_BLOCK must be a multiple of 32 in [32,128]");

    const size_t table_bytes = (size_t)n_ops * sizeof(DevOp);
    const size_t smem_budget = b->max_smem_optin > 0 ? (size_t)b->max_smem_optin : (size_t)48 * 1024;
    bool use_smem = table_bytes <= smem_budget / 2;  // keep >= 2 CTAs per SM resident
    const int src = env_int("BT_TRACK_SRC", -1);  // 0: global, 1: shared
    if (src == 0) use_smem = false;
    if (src == 1 && table_bytes <= smem_budget) use_smem = true;

    TrackArgs a;
    for (int c = 0; c < 6; ++c) a.q[c] = b->q[c];
    a.table = d_table;
    a.n = n;
    a.n_ops = n_ops;
    a.nturns = nturns;
    a.turn_stride = turn_stride;
    const long long per_block = (long long)P * block;
    const long long full = n / per_block;
    a.n_full_blocks = (int)full;
    a.tail_start = full * per_block;
    const long long rem = n - a.tail_start;
    const long long grid_ll = full + (rem + block - 1) / block;
    if (grid_ll > 0x7fffffffLL) return fail(BT_ERR_UNSUPPORTED, "bt_track: grid too large");
    const int grid = (int)grid_ll;
    const size_t smem = use_smem ? table_bytes : 0;

    cudaError_t e;
    if (use_smem) {
        e = P == 4 ? do_launch<4, true>(a, grid, block, smem, b->stream)
          : P == 2 ? do_launch<2, true>(a, grid, block, smem, b->stream)
                   : do_launch<1, true>(a, grid, block, smem, b->stream);
    } else {
        e = P == 4 ? do_launch<4, false>(a, grid, block, smem, b->stream)
          : P == 2 ? do_launch<2, false>(a, grid, block, smem, b->stream)
                   : do_launch<1, false>(a, grid, block, smem, b->stream);
    }
    if (e != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_track launch: ") + cudaGetErrorString(e));
    g_launch_count.fetch_add(1);
    b->last_launch.grid = grid;
    b->last_launch.block = block;
    b->last_launch.ppt = P;
    b->last_launch.smem = (int32_t)smem;
    return BT_OK;
}

}  // namespace bt
