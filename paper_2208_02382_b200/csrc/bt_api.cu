// C-ABI entry points of libbt.so (include/bt.h): handles, validation, host-side coefficient
// precompute (S1, S3) and the call sequence of the hot path.  All particle work runs in the
// kernels of track.cu / grid.cu.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "bt_internal.h"

namespace bt {

static thread_local std::string t_last_error;
std::atomic<int64_t> g_launch_count{0};

void set_error(const std::string &msg) { t_last_error = msg; }
int fail(int code, const std::string &msg) {
    t_last_error = msg;
    return code;
}

static const double kPi = 3.14159265358979323846264338327950288;
static const double kCLight = 299792458.0;

// ---- validation (SURVEY 8b "Errors") ------------------------------------------------------------
static int validate_element(const bt_element &e, int idx) {
    auto bad = [&](const char *why) {
        return fail(BT_ERR_INVALID, "element " + std::to_string(idx) + ": " + why);
    };
    if (e.nslice < 1) return bad("nslice < 1");
    if (!(e.ds >= 0.0) || !isfinite(e.ds)) return bad("ds < 0 or not finite");
    switch (e.type) {
        case BT_DRIFT:
        case BT_DRIFT_EXACT:
            break;
        case BT_QUAD_CHROMATIC:
        case BT_QUAD:
            if (!isfinite(e.p[0])) return bad("k not finite");
            break;
        case BT_SBEND:
            if (e.p[0] == 0.0 || !isfinite(e.p[0])) return bad("rc == 0 or not finite");
            break;
        case BT_DIPEDGE:
            if (e.nslice != 1) return bad("thin element needs nslice == 1");
            if (e.p[1] == 0.0 || !isfinite(e.p[1])) return bad("rc == 0 or not finite");
            if (!isfinite(e.p[0]) || cos(e.p[0]) == 0.0) return bad("cos(psi) == 0");
            if (!isfinite(e.p[2]) || !isfinite(e.p[3])) return bad("g or K not finite");
            break;
        case BT_MULTIPOLE:
            if (e.nslice != 1) return bad("thin element needs nslice == 1");
            if (!(e.p[0] >= 1.0 && e.p[0] <= 10.0) || e.p[0] != floor(e.p[0])) return bad("m not an integer in [1,10]");
            if (!isfinite(e.p[1]) || !isfinite(e.p[2])) return bad("Kn or Ks not finite");
            break;
        case BT_SHORTRF:
        case BT_SHORTRF_SIN:
            if (e.nslice != 1) return bad("thin element needs nslice == 1");
            if (!isfinite(e.p[0]) || !isfinite(e.p[1]) || !isfinite(e.p[2])) return bad("RF parameter not finite");
            break;
        default:
            return bad("unknown element type");
    }
    return BT_OK;
}

// ---- debug knobs (bt_debug_knob): process-wide, typed, default -1 = "the measured default" ---------------------------
std::atomic<int32_t> g_knob[KNOB_COUNT] = {{-1}, {-1}, {-1}, {-1}, {-1}, {-1}};
static const char *const kKnobNames[KNOB_COUNT] = {"track_ppt", "track_block", "track_fuse", "deposit_mode", "gather_mode", "plan_window"};

// Runs of half cells [QUAD1][SEXTOCT|TAILDRIFT] among the records appended since `start` become one dispatch: the first
// record of a run is relabelled OP_HALFCELL with count = pairs in the run; the coefficients stay where they are, so the
// table keeps its size and the walk applies exactly the same maps in the same order.  A run never crosses a multiple of
// kTableRecords counted from `start` (where bt_track cuts a turn that is longer than one launch's table).
static void fuse_halfcell_runs(std::vector<DevOp> &out, size_t start) {
    const size_t K = (size_t)kTableRecords;
    size_t i = start;
    while (i + 1 < out.size()) {
        size_t head = i, pairs = 0;
        while (i + 1 < out.size() && out[i].op == OP_QUAD1 && out[i + 1].op == (OP_SEXTOCT | OP_TAILDRIFT) &&
               (i - start) / K == (i + 1 - start) / K && (i - start) / K == (head - start) / K) {
            ++pairs;
            i += 2;
        }
        if (pairs >= 1) {
            out[head].op = OP_HALFCELL;
            out[head].count = (int32_t)pairs;
        } else {
            ++i;
        }
    }
}

// ---- S1/S3: coefficients of one slice map per element, for one pass at reference gamma ----------
// diag != 0: tables of the diagnostics walk -- no record spans two elements (no fusion) and the last record of every element
// is marked OP_MARK; diag == 2 (slice granularity): exactly one looped record per element (no five-slice groups either).
// The coefficients are the same expressions, so the walk is bit-identical to bt_track's.
double build_turn_table(const std::vector<bt_element> &lat, double gamma, std::vector<DevOp> &out, double *slots, int diag) {
    double nslots = 0.0;
    const bool fuse = !diag && g_knob[KNOB_TRACK_FUSE].load() != 0;  // 0: one record per element (A/B measurements, bit-identity test)
    const size_t start = out.size();
    for (size_t i = 0; i < lat.size(); ++i) {
        if (diag && i > 0) out.back().op |= OP_MARK;  // the previous element ended with the last record pushed so far
        const bt_element &e = lat[i];
        DevOp o;
        memset(&o, 0, sizeof(o));
        o.count = e.nslice;
        const double bg = sqrt(gamma * gamma - 1.0);
        const double beta = bg / gamma;
        const double h = e.ds / (double)e.nslice;  // R3: one rounded division
        const double tc = h / (bg * bg);
        switch (e.type) {
            case BT_DRIFT:
                nslots += 3.0 * e.nslice;
                // peephole: a single-slice drift right behind a normal sextupole/octupole kick shares its dispatch
                if (fuse && e.nslice == 1 && i > 0 && !out.empty() && lat[i - 1].type == BT_MULTIPOLE &&
                    (out.back().op == OP_SEXT || out.back().op == OP_OCT || out.back().op == OP_SEXTOCT)) {
                    out.back().op |= OP_TAILDRIFT;
                    out.back().c[3] = h;
                    out.back().c[4] = tc;
                    break;
                }
                o.op = (e.nslice == 1 && diag != 2) ? OP_DRIFT1 : OP_DRIFT;
                o.c[0] = h;
                o.c[1] = tc;
                out.push_back(o);
                break;
            case BT_QUAD: {
                const double k = e.p[0];
                if (k == 0.0) {  // R5: k = 0 is a drift
                    o.op = (e.nslice == 1 && diag != 2) ? OP_DRIFT1 : OP_DRIFT;
                    o.c[0] = h;
                    o.c[1] = tc;
                    nslots += 3.0 * e.nslice;
                    out.push_back(o);
                    break;
                }
                const double w = sqrt(fabs(k));
                const double c = cos(w * h), s = sin(w * h), ch = cosh(w * h), sh = sinh(w * h);
                const double f[3] = {c, s / w, -w * s};
                const double d[3] = {ch, sh / w, w * sh};
                const double *xb = k > 0.0 ? f : d, *yb = k > 0.0 ? d : f;
                o.c[0] = xb[0];
                o.c[1] = xb[1];
                o.c[2] = xb[2];
                o.c[3] = yb[0];
                o.c[4] = yb[1];
                o.c[5] = yb[2];
                o.c[6] = tc;
                nslots += 9.0 * e.nslice;
                if (diag == 2) {
                    o.op = OP_QUAD;
                    out.push_back(o);
                    break;
                }
                // nslice = 5a + b: a groups of five slices, then b single slices (same slice map, same order)
                if (e.nslice / 5 > 0) {
                    o.op = OP_QUAD5;
                    o.count = e.nslice / 5;
                    out.push_back(o);
                }
                if (e.nslice % 5 > 0) {
                    o.op = e.nslice % 5 == 1 ? OP_QUAD1 : OP_QUAD;
                    o.count = e.nslice % 5;
                    out.push_back(o);
                }
                break;
            }
            case BT_SBEND: {
                const double rho = e.p[0];
                const double th = h / rho;
                const double C = cos(th), S = sin(th);
                o.op = OP_SBEND;
                o.c[0] = C;
                o.c[1] = rho * S;
                o.c[2] = -(S / rho);
                o.c[3] = -(rho * (1.0 - C)) / beta;
                o.c[4] = -S / beta;
                o.c[5] = rho * (S / (beta * beta) - th);
                o.c[6] = h;
                nslots += 10.0 * e.nslice;
                out.push_back(o);
                break;
            }
            case BT_DIPEDGE: {
                const double psi = e.p[0], rho = e.p[1], g = e.p[2], K = e.p[3];
                const double sp = sin(psi), cp = cos(psi);
                const double psi_c = K * (g / rho) * (1.0 + sp * sp) / cp;
                o.op = OP_EDGE;
                o.c[0] = tan(psi) / rho;
                o.c[1] = -tan(psi - psi_c) / rho;
                nslots += 2.0;
                out.push_back(o);
                break;
            }
            case BT_MULTIPOLE: {
                const int m = (int)e.p[0];
                const double Kn = e.p[1], Ks = e.p[2];
                double fact = 1.0;
                for (int j = 2; j <= m - 1; ++j) fact *= (double)j;
                if (m == 3 && Ks == 0.0) {
                    o.op = OP_SEXT;
                    o.c[0] = Kn / 2.0;
                    o.c[1] = Kn;
                    nslots += 5.0;
                } else if (m == 4 && Ks == 0.0) {
                    nslots += 8.0;
                    // peephole: a normal octupole right behind a normal sextupole shares its dispatch
                    if (fuse && i > 0 && !out.empty() && out.back().op == OP_SEXT && lat[i - 1].type == BT_MULTIPOLE) {
                        out.back().op = OP_SEXTOCT;
                        out.back().c[2] = Kn / 6.0;
                        break;
                    }
                    o.op = OP_OCT;
                    o.c[2] = Kn / 6.0;
                } else {
                    o.op = OP_MULT;
                    o.count = m;
                    o.c[0] = Kn / fact;
                    o.c[1] = Ks / fact;
                    nslots += 4.0 * (m - 1) + 6.0;
                }
                out.push_back(o);
                break;
            }
            case BT_SHORTRF: {
                const double Vhat = e.p[0], freq = e.p[1], phi = e.p[2] * (kPi / 180.0);
                const double gamma_f = gamma + Vhat * cos(phi);
                const double bg_f = sqrt(gamma_f * gamma_f - 1.0);
                const double krf = 2.0 * kPi * freq / kCLight;
                o.op = OP_RF;
                o.c[0] = bg / bg_f;
                o.c[1] = Vhat * krf * sin(phi) / bg_f;
                gamma = gamma_f;  // S3: later elements see the new reference energy
                nslots += 4.0;
                out.push_back(o);
                break;
            }
            case BT_DRIFT_EXACT:  // R17
                o.op = OP_DRIFTX;
                o.c[0] = h;
                o.c[1] = 1.0 / beta;
                nslots += 26.0 * e.nslice;  // 12 DFMA/DMUL/DADD + reciprocal square root (~14 FP64-pipe instructions)
                out.push_back(o);
                break;
            case BT_QUAD_CHROMATIC:  // R20
                o.op = OP_QUADCHR;
                o.c[0] = h;
                o.c[1] = 1.0 / beta;
                o.c[2] = fabs(e.p[0]);
                o.c[3] = e.p[0] > 0.0 ? 1.0 : e.p[0] < 0.0 ? -1.0 : 0.0;
                nslots += 200.0 * e.nslice;  // two square roots, sincos, exp, a reciprocal and ~60 DFMA/DMUL: order of magnitude
                out.push_back(o);
                break;
            case BT_SHORTRF_SIN: {  // R18
                const double Vhat = e.p[0], freq = e.p[1], phi = e.p[2] * (kPi / 180.0);
                const double cphi = cos(phi);
                const double gamma_f = gamma + Vhat * cphi;
                const double bg_f = sqrt(gamma_f * gamma_f - 1.0);
                o.op = OP_RFSIN;
                o.c[0] = bg / bg_f;
                o.c[1] = -(Vhat / bg_f);
                o.c[2] = 2.0 * kPi * freq / kCLight;
                o.c[3] = phi;
                o.c[4] = cphi;
                gamma = gamma_f;
                nslots += 40.0;  // fp64 cosine ~ 35 FP64-pipe instructions on the fast path
                out.push_back(o);
                break;
            }
        }
    }
    if (fuse) fuse_halfcell_runs(out, start);
    if (diag && out.size() > start) out.back().op |= OP_MARK;
    if (slots) *slots = nslots;
    return gamma;
}

// ---- grids are shared between streams: order their operations with one event ------------------------------------------
int grid_acquire(Grid *g, cudaStream_t s) {
    if (g->done_valid && s != g->last_stream) BT_CUDA_TRY(cudaStreamWaitEvent(s, g->done, 0));
    return BT_OK;
}
int grid_release(Grid *g, cudaStream_t s) {
    if (!g->done) BT_CUDA_TRY(cudaEventCreateWithFlags(&g->done, cudaEventDisableTiming));
    BT_CUDA_TRY(cudaEventRecord(g->done, s));
    g->done_valid = true;
    g->last_stream = s;
    return BT_OK;
}

// ---- the launches of one bt_track(nturns) call ---------------------------------------------------------------------
// A plan is a list of (records, passes) launches over record storage it owns or borrows.  Static lattices: one table,
// walked nturns times by one launch (or, when a turn needs more than kTableRecords records, its segments turn after turn).
// Lattices whose RF changes the reference energy (S3): every turn has its own coefficients; as many whole turns as fit
// one launch's table go into it.
// A plan covers a WINDOW of turns, not necessarily the whole call: per-turn tables cost 64 bytes per record and turn
// (bt_track(10^6 turns) of a 200-record ring would be 12.8 GB of host memory if built at once), so plan_walk stops after
// kPlanWindowRecords records (whole turns, at least one) and the caller asks again from the reference energy the window
// ends at.  The records of a launch are copied into its parameters when it is enqueued, so a window's storage is reused at
// once, and the host builds window k+1 (cos/sinh per turn) while the GPU walks window k.
struct WalkPlan {
    struct Launch {
        size_t lo;
        int32_t len, nturns;
        double spr;  // FP64 slots per record (geometry heuristic)
    };
    const std::vector<DevOp> *ops = nullptr;
    std::vector<DevOp> own;
    std::vector<Launch> launches;
    double gamma_after = 0.0;
};

constexpr int kPlanWindowRecords = 128 * kTableRecords;  // 65 280 records = 4 MiB of host memory per window

// Plans the next window of a walk of `nturns` turns that starts at reference energy `gamma`; returns the turns it covers
// (1..nturns) and leaves the energy after them in plan.gamma_after.
static int32_t plan_walk(Beam &b, double gamma, int32_t nturns, WalkPlan &plan) {
    const size_t K = (size_t)kTableRecords;
    const size_t window = (size_t)knob(KNOB_PLAN_WINDOW, kPlanWindowRecords);
    plan.own.clear();
    plan.launches.clear();
    auto add_segments = [&](size_t lo, size_t len, double spr) {
        for (size_t o = 0; o < len; o += K) plan.launches.push_back({lo + o, (int32_t)(len - o < K ? len - o : K), 1, spr});
    };
    if (!b.energy_changes) {
        const int fuse_now = knob(KNOB_TRACK_FUSE, 1) != 0;
        if (!b.table_valid || b.table_fuse != fuse_now) {  // the cached table was built under the knob's value at the time
            b.h_table.clear();
            build_turn_table(b.lattice, gamma, b.h_table, &b.table_slots);
            b.table_valid = true;
            b.table_fuse = fuse_now;
        }
        plan.ops = &b.h_table;
        plan.gamma_after = gamma;
        const double spr = b.table_slots / (double)b.h_table.size();
        // A periodic channel (configs[1]: one FODO cell x 100) is one period walked repeats x nturns times: the same
        // records in the same order, a table of 5 instead of 500 records in the launch's parameters.
        size_t period = b.h_table.size();
        for (size_t p = 1; p <= b.h_table.size() / 2; ++p) {
            if (b.h_table.size() % p) continue;
            if (memcmp(b.h_table.data(), b.h_table.data() + p, (b.h_table.size() - p) * sizeof(DevOp)) == 0) {
                period = p;
                break;
            }
        }
        const long long passes = (long long)nturns * (long long)(b.h_table.size() / period);
        if (period <= K && passes <= 0x7fffffffLL) {
            plan.launches.push_back({0, (int32_t)period, (int32_t)passes, spr});
            return nturns;
        }
        if (b.h_table.size() <= K) {
            plan.launches.push_back({0, (int32_t)b.h_table.size(), nturns, spr});
            return nturns;
        }
        // a turn longer than one table: its segments turn after turn, a window's worth of records at a time
        long long turns = (long long)(window / b.h_table.size());
        if (turns < 1) turns = 1;
        if (turns > nturns) turns = nturns;
        for (long long t = 0; t < turns; ++t) add_segments(0, b.h_table.size(), spr);
        return (int32_t)turns;
    }
    plan.ops = &plan.own;
    size_t pend_lo = 0;  // records [pend_lo, own.size()) = whole turns not yet assigned to a launch
    double pend_spr = 0.0;
    int32_t t = 0;
    while (t < nturns && (t == 0 || plan.own.size() < window)) {
        const size_t turn_lo = plan.own.size();
        double slots = 0.0;
        gamma = build_turn_table(b.lattice, gamma, plan.own, &slots);
        ++t;
        const size_t turn_len = plan.own.size() - turn_lo;
        const double spr = slots / (double)turn_len;
        if (turn_len > K) {  // a single turn exceeds one table: flush what is pending, then its segments
            if (turn_lo > pend_lo) plan.launches.push_back({pend_lo, (int32_t)(turn_lo - pend_lo), 1, pend_spr});
            add_segments(turn_lo, turn_len, spr);
            pend_lo = plan.own.size();
            continue;
        }
        if (plan.own.size() - pend_lo > K) {  // this turn no longer fits with the pending ones
            plan.launches.push_back({pend_lo, (int32_t)(turn_lo - pend_lo), 1, pend_spr});
            pend_lo = turn_lo;
        }
        pend_spr = spr;
    }
    if (plan.own.size() > pend_lo) plan.launches.push_back({pend_lo, (int32_t)(plan.own.size() - pend_lo), 1, pend_spr});
    plan.gamma_after = gamma;
    return t;
}

static int run_plan(Beam &b, const WalkPlan &plan) {  // on b.range's stream when set, else on the beam's
    for (const WalkPlan::Launch &l : plan.launches) {
        const int rc = launch_track(&b, plan.ops->data() + l.lo, l.len, l.nturns, l.spr);
        if (rc != BT_OK) return rc;
    }
    return BT_OK;
}

// All windows of a walk of nturns turns from the beam's current reference energy, on b.range's stream when set, else on
// the beam's; *gamma_after = the reference energy at the end.  `plan` is working storage (reused window after window).
static int run_walk(Beam &b, int32_t nturns, WalkPlan &plan, double *gamma_after) {
    double gamma = b.gamma;
    for (int32_t left = nturns; left > 0;) {
        const int32_t did = plan_walk(b, gamma, left, plan);
        const int rc = run_plan(b, plan);
        if (rc != BT_OK) return rc;
        gamma = plan.gamma_after;
        left -= did;
    }
    *gamma_after = gamma;
    return BT_OK;
}

}  // namespace bt

using namespace bt;

extern "C" {

const char *bt_last_error(void) { return t_last_error.c_str(); }

int bt_debug_knob(const char *name, int32_t value) {
    if (!name) return fail(BT_ERR_INVALID, "bt_debug_knob: name is NULL");
    for (int k = 0; k < KNOB_COUNT; ++k)
        if (strcmp(name, kKnobNames[k]) == 0) {
            g_knob[k].store(value < 0 ? -1 : value);
            return BT_OK;
        }
    return fail(BT_ERR_INVALID, std::string("bt_debug_knob: unknown knob ") + name);
}
int bt_version(void) { return BT_VERSION; }
int64_t bt_launch_count(void) { return g_launch_count.load(); }

int bt_beam_create(bt_beam **out, int64_t n, double *const dev_ptrs[6], void *cuda_stream) {
    if (!out) return fail(BT_ERR_INVALID, "bt_beam_create: out is NULL");
    *out = nullptr;
    if (n <= 0) return fail(BT_ERR_INVALID, "bt_beam_create: n <= 0");
    if (n > ((int64_t)1 << 40)) return fail(BT_ERR_INVALID, "bt_beam_create: n too large");
    if (dev_ptrs)
        for (int i = 0; i < 6; ++i) {
            if (!dev_ptrs[i]) return fail(BT_ERR_INVALID, "bt_beam_create: dev_ptrs has a NULL entry");
            if (((uintptr_t)dev_ptrs[i]) & 7u) return fail(BT_ERR_INVALID, "bt_beam_create: device pointer not 8-byte aligned");
        }
    int dev = 0;
    BT_CUDA_TRY(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    BT_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    bt_beam *h = new (std::nothrow) bt_beam();
    if (!h) return fail(BT_ERR_OOM, "bt_beam_create: host allocation failed");
    Beam &b = h->b;
    b.n = n;
    b.device = dev;
    b.num_sms = prop.multiProcessorCount;
    b.max_smem_optin = (int)prop.sharedMemPerBlockOptin;
    b.stream = (cudaStream_t)cuda_stream;
    if (dev_ptrs) {
        for (int i = 0; i < 6; ++i) b.q[i] = b.home[i] = dev_ptrs[i];
        b.owns = false;
        b.pingpong = false;  // lent arrays always hold the bunch unless bt_beam_set_sort_pingpong says otherwise
    } else {
        // one allocation, 6 slices, each 256-byte aligned (S0)
        const size_t stride = (((size_t)n * sizeof(double)) + 255u) & ~(size_t)255u;
        double *base = nullptr;
        cudaError_t e = cudaMalloc(&base, stride * 6);
        if (e != cudaSuccess) {
            delete h;
            return fail(e == cudaErrorMemoryAllocation ? BT_ERR_OOM : BT_ERR_CUDA,
                        std::string("bt_beam_create: cudaMalloc: ") + cudaGetErrorString(e));
        }
        for (int i = 0; i < 6; ++i) b.q[i] = b.home[i] = (double *)((char *)base + stride * i);
        b.owns = true;
        b.pingpong = true;
    }
    b.aligned16 = b.aligned32 = true;
    for (int i = 0; i < 6; ++i) {
        if (((uintptr_t)b.q[i]) & 15u) b.aligned16 = false;
        if (((uintptr_t)b.q[i]) & 31u) b.aligned32 = false;
    }
    *out = h;
    return BT_OK;
}

void bt_beam_destroy(bt_beam *beam) {
    if (!beam) return;
    Beam &b = beam->b;
    cudaStreamSynchronize(b.stream);
    if (b.owns && b.home[0]) cudaFree(b.home[0]);
    if (b.alt[0]) cudaFree(b.alt[0]);
    int *ibufs[] = {b.ids, b.ids_tmp, b.sort_count, b.sort_block_sum};
    for (int *p : ibufs)
        if (p) cudaFree(p);
    if (b.dl_tmp) cudaFree(b.dl_tmp);
    if (b.mom_buf) cudaFree(b.mom_buf);
    if (b.mom_host) cudaFreeHost(b.mom_host);
    if (b.diag_rows) cudaFree(b.diag_rows);
    if (b.diag_out) cudaFree(b.diag_out);
    for (int i = 0; i < 3; ++i) {
        if (b.pipe_stream[i]) cudaStreamDestroy(b.pipe_stream[i]);
        if (b.pipe_event[i]) cudaEventDestroy(b.pipe_event[i]);
    }
    delete beam;
}

int bt_beam_set_ref(bt_beam *beam, double kin_energy_MeV, double mass_MeV, double charge_qe) {
    if (!beam) return fail(BT_ERR_INVALID, "bt_beam_set_ref: beam is NULL");
    if (!(kin_energy_MeV > 0.0) || !isfinite(kin_energy_MeV)) return fail(BT_ERR_INVALID, "bt_beam_set_ref: energy <= 0");
    if (!(mass_MeV > 0.0) || !isfinite(mass_MeV)) return fail(BT_ERR_INVALID, "bt_beam_set_ref: mass <= 0");
    Beam &b = beam->b;
    b.gamma = 1.0 + kin_energy_MeV / mass_MeV;  // R2: kinetic energy
    if (!(b.gamma > 1.0)) return fail(BT_ERR_INVALID, "bt_beam_set_ref: gamma == 1 in fp64");
    b.mass_MeV = mass_MeV;
    b.charge_qe = charge_qe;
    b.s = 0.0;
    b.turn = 0;
    b.has_ref = true;
    b.table_valid = false;
    return BT_OK;
}

int bt_beam_get_ref(const bt_beam *beam, double *gamma, double *s, int64_t *turn) {
    if (!beam) return fail(BT_ERR_INVALID, "bt_beam_get_ref: beam is NULL");
    if (!beam->b.has_ref) return fail(BT_ERR_STATE, "bt_beam_get_ref: bt_beam_set_ref not called");
    if (gamma) *gamma = beam->b.gamma;
    if (s) *s = beam->b.s;
    if (turn) *turn = beam->b.turn;
    return BT_OK;
}

int64_t bt_beam_size(const bt_beam *beam) { return beam ? beam->b.n : 0; }

int bt_beam_upload(bt_beam *beam, const double *const host[6]) {
    if (!beam || !host) return fail(BT_ERR_INVALID, "bt_beam_upload: NULL argument");
    for (int i = 0; i < 6; ++i)
        if (!host[i]) return fail(BT_ERR_INVALID, "bt_beam_upload: host has a NULL entry");
    Beam &b = beam->b;
    set_current_storage(&b, false);  // back in the home arrays, in the caller's order
    for (int i = 0; i < 6; ++i)
        BT_CUDA_TRY(cudaMemcpyAsync(b.q[i], host[i], (size_t)b.n * sizeof(double), cudaMemcpyHostToDevice, b.stream));
    b.permuted = false;
    b.deposits_since_sort = 0;
    ++b.storage_epoch;
    return BT_OK;
}

int bt_beam_download(const bt_beam *beam, double *const host[6]) {
    if (!beam || !host) return fail(BT_ERR_INVALID, "bt_beam_download: NULL argument");
    for (int i = 0; i < 6; ++i)
        if (!host[i]) return fail(BT_ERR_INVALID, "bt_beam_download: host has a NULL entry");
    Beam &b = const_cast<Beam &>(beam->b);
    for (int i = 0; i < 6; ++i) {
        const double *src = b.q[i];
        if (b.permuted) {  // storage is cell-sorted: restore the original order through the idle partner array --
            // never through arrays the caller lent (their owner may be reading them): those get a scratch of the library's
            double *tmp = b.in_alt ? b.home[i] : b.alt[i];
            if (b.in_alt && !b.owns) {
                if (!b.dl_tmp) BT_CUDA_TRY(cudaMalloc(&b.dl_tmp, (size_t)b.n * sizeof(double)));
                tmp = b.dl_tmp;
            }
            int rc = unpermute_to(&b, i, tmp);
            if (rc != BT_OK) return rc;
            src = tmp;
        }
        BT_CUDA_TRY(cudaMemcpyAsync(host[i], src, (size_t)b.n * sizeof(double), cudaMemcpyDeviceToHost, b.stream));
    }
    BT_CUDA_TRY(cudaStreamSynchronize(b.stream));
    return BT_OK;
}

int bt_beam_ptrs(bt_beam *beam, double *dev_ptrs_out[6]) {
    if (!beam || !dev_ptrs_out) return fail(BT_ERR_INVALID, "bt_beam_ptrs: NULL argument");
    for (int i = 0; i < 6; ++i) dev_ptrs_out[i] = beam->b.q[i];
    return BT_OK;
}

int bt_beam_sort_by_cell(bt_beam *beam, const bt_grid *grid, double zscale) {
    if (!beam || !grid) return fail(BT_ERR_INVALID, "bt_beam_sort_by_cell: NULL argument");
    if (!isfinite(zscale)) return fail(BT_ERR_INVALID, "bt_beam_sort_by_cell: zscale not finite");
    return sort_by_cell(&beam->b, &grid->g, zscale);
}

int bt_beam_set_sort_pingpong(bt_beam *beam, int enable) {
    if (!beam) return fail(BT_ERR_INVALID, "bt_beam_set_sort_pingpong: beam is NULL");
    beam->b.pingpong = enable != 0;
    return enable ? BT_OK : rehome(&beam->b);
}

int bt_beam_rehome(bt_beam *beam) {
    if (!beam) return fail(BT_ERR_INVALID, "bt_beam_rehome: beam is NULL");
    return rehome(&beam->b);
}

int bt_beam_storage(const bt_beam *beam, int32_t *in_home, int64_t *epoch) {
    if (!beam) return fail(BT_ERR_INVALID, "bt_beam_storage: beam is NULL");
    if (in_home) *in_home = beam->b.in_alt ? 0 : 1;
    if (epoch) *epoch = beam->b.storage_epoch;
    return BT_OK;
}

int bt_beam_ids(bt_beam *beam, int32_t **dev_ids_out) {
    if (!beam || !dev_ids_out) return fail(BT_ERR_INVALID, "bt_beam_ids: NULL argument");
    *dev_ids_out = beam->b.permuted ? beam->b.ids : nullptr;
    return BT_OK;
}

int bt_sync(bt_beam *beam) {
    if (!beam) return fail(BT_ERR_INVALID, "bt_sync: beam is NULL");
    BT_CUDA_TRY(cudaStreamSynchronize(beam->b.stream));
    return BT_OK;
}

int bt_lattice_set(bt_beam *beam, const bt_element *elems, int32_t n_elems) {
    if (!beam || !elems) return fail(BT_ERR_INVALID, "bt_lattice_set: NULL argument");
    if (n_elems < 1) return fail(BT_ERR_INVALID, "bt_lattice_set: n_elems < 1");
    bool energy_changes = false;
    double length = 0.0;
    for (int32_t i = 0; i < n_elems; ++i) {
        int rc = validate_element(elems[i], i);
        if (rc != BT_OK) return rc;
        if ((elems[i].type == BT_SHORTRF || elems[i].type == BT_SHORTRF_SIN) && elems[i].p[0] * cos(elems[i].p[2] * (kPi / 180.0)) != 0.0)
            energy_changes = true;
        length += elems[i].ds;
    }
    Beam &b = beam->b;
    b.lattice.assign(elems, elems + n_elems);
    b.energy_changes = energy_changes;
    b.lattice_length = length;
    b.table_valid = false;
    return BT_OK;
}

int bt_track(bt_beam *beam, int32_t nturns) {
    if (!beam) return fail(BT_ERR_INVALID, "bt_track: beam is NULL");
    if (nturns < 0) return fail(BT_ERR_INVALID, "bt_track: nturns < 0");
    Beam &b = beam->b;
    if (b.lattice.empty()) return fail(BT_ERR_STATE, "bt_track: bt_lattice_set not called");
    if (!b.has_ref) return fail(BT_ERR_STATE, "bt_track: bt_beam_set_ref not called");
    if (nturns == 0) return BT_OK;
    WalkPlan plan;
    double gamma_after = b.gamma;
    const int rc = run_walk(b, nturns, plan, &gamma_after);
    if (rc != BT_OK) return rc;
    b.gamma = gamma_after;  // S3
    b.s += b.lattice_length * (double)nturns;
    b.turn += nturns;
    return BT_OK;
}

// Slice-step / element-step diagnostics fused into the walk (P:l.61 set_slice_step_diagnostics): O(1)
// launches per table -- the diagnostics walk writes one 216-byte row per (warp, boundary), a combine kernel turns the
// rows of a launch into records.  Launches are cut where the record table (510 records) or the row buffer (1 GiB) is full.
int bt_track_diagnostics_records(const bt_beam *beam, int32_t nturns, int32_t granularity, int64_t *n_records) {
    if (!beam || !n_records) return fail(BT_ERR_INVALID, "bt_track_diagnostics_records: NULL argument");
    if (nturns < 0) return fail(BT_ERR_INVALID, "bt_track_diagnostics_records: nturns < 0");
    if (granularity != BT_DIAG_ELEMENT && granularity != BT_DIAG_SLICE) return fail(BT_ERR_INVALID, "bt_track_diagnostics_records: granularity must be BT_DIAG_ELEMENT or BT_DIAG_SLICE");
    if (beam->b.lattice.empty()) return fail(BT_ERR_STATE, "bt_track_diagnostics_records: bt_lattice_set not called");
    long long per_turn = 0;
    for (const bt_element &e : beam->b.lattice) per_turn += granularity == BT_DIAG_SLICE ? e.nslice : 1;
    *n_records = per_turn * nturns;
    return BT_OK;
}

int bt_track_diagnostics_n(bt_beam *beam, int32_t nturns, int32_t granularity, double *host_moments, int64_t capacity_records) {
    int64_t need = 0;
    const int rc = bt_track_diagnostics_records(beam, nturns, granularity, &need);
    if (rc != BT_OK) return rc;
    if (capacity_records < need)
        return fail(BT_ERR_INVALID, "bt_track_diagnostics_n: host_moments holds " + std::to_string((long long)capacity_records) +
                                        " records of 42 doubles, the call writes " + std::to_string((long long)need));
    return bt_track_diagnostics(beam, nturns, granularity, host_moments);
}

int bt_beam_release_scratch(bt_beam *beam) {
    if (!beam) return fail(BT_ERR_INVALID, "bt_beam_release_scratch: beam is NULL");
    Beam &b = beam->b;
    BT_CUDA_TRY(cudaStreamSynchronize(b.stream));
    if (b.diag_rows) cudaFree(b.diag_rows);
    if (b.diag_out) cudaFree(b.diag_out);
    if (b.dl_tmp) cudaFree(b.dl_tmp);
    b.diag_rows = b.diag_out = b.dl_tmp = nullptr;
    b.diag_rows_bytes = b.diag_out_bytes = 0;
    return BT_OK;
}

int bt_track_diagnostics(bt_beam *beam, int32_t nturns, int32_t granularity, double *host_moments) {
    if (!beam || !host_moments) return fail(BT_ERR_INVALID, "bt_track_diagnostics: NULL argument");
    if (nturns < 0) return fail(BT_ERR_INVALID, "bt_track_diagnostics: nturns < 0");
    if (granularity != BT_DIAG_ELEMENT && granularity != BT_DIAG_SLICE) return fail(BT_ERR_INVALID, "bt_track_diagnostics: granularity must be BT_DIAG_ELEMENT or BT_DIAG_SLICE");
    Beam &b = beam->b;
    if (b.lattice.empty()) return fail(BT_ERR_STATE, "bt_track_diagnostics: bt_lattice_set not called");
    if (!b.has_ref) return fail(BT_ERR_STATE, "bt_track_diagnostics: bt_beam_set_ref not called");
    const bool slice = granularity == BT_DIAG_SLICE;
    long long per_turn = 0;
    for (const bt_element &e : b.lattice) per_turn += slice ? e.nslice : 1;
    const long long nrec = per_turn * nturns;
    if (nrec == 0) return BT_OK;
    int P = 1, block = 128;
    const long long nwarps = diag_warps(&b, &P, &block);
    const long long row_bytes = nwarps * 27 * (long long)sizeof(double);      // one boundary
    const long long budget = 1LL << 30;
    long long cap = budget / row_bytes;                                       // boundaries per launch
    if (cap < 1) cap = 1;
    if (cap > nrec) cap = nrec;
    double *dev_out = nullptr, *centre = nullptr;
    if (b.diag_rows_bytes < (size_t)(cap * row_bytes)) {  // the row buffer stays with the beam (up to 1 GiB)
        if (b.diag_rows) {
            BT_CUDA_TRY(cudaStreamSynchronize(b.stream));
            BT_CUDA_TRY(cudaFree(b.diag_rows));
            b.diag_rows = nullptr, b.diag_rows_bytes = 0;
        }
        BT_CUDA_TRY(cudaMalloc(&b.diag_rows, (size_t)(cap * row_bytes)));
        b.diag_rows_bytes = (size_t)(cap * row_bytes);
    }
    double *rows = b.diag_rows;
    const size_t out_bytes = (size_t)nrec * 42 * sizeof(double) + 64;
    if (b.diag_out_bytes < out_bytes) {  // the record buffer stays with the beam as well (no allocation on repeated calls)
        if (b.diag_out) {
            BT_CUDA_TRY(cudaStreamSynchronize(b.stream));
            BT_CUDA_TRY(cudaFree(b.diag_out));
            b.diag_out = nullptr, b.diag_out_bytes = 0;
        }
        BT_CUDA_TRY(cudaMalloc(&b.diag_out, out_bytes));
        b.diag_out_bytes = out_bytes;
    }
    dev_out = b.diag_out;
    centre = dev_out + nrec * 42;
    int rc = launch_moments_centre(&b, centre);
    std::vector<DevOp> ops, pend;
    long long pend_b = 0, done_b = 0;
    auto flush = [&]() -> int {
        if (pend.empty()) return BT_OK;
        const int r = launch_track_diag(&b, pend.data(), (int32_t)pend.size(), slice ? 1 : 0, (int)pend_b, centre, rows, dev_out + done_b * 42);
        done_b += pend_b;
        pend.clear();
        pend_b = 0;
        return r;
    };
    double gamma = b.gamma;
    for (int32_t t = 0; t < nturns && rc == BT_OK; ++t) {
        ops.clear();
        gamma = build_turn_table(b.lattice, gamma, ops, nullptr, slice ? 2 : 1);
        for (size_t i = 0; i < ops.size() && rc == BT_OK; ++i) {
            DevOp o = ops[i];
            const bool looped = (o.op & (OP_DRIFT | OP_QUAD | OP_SBEND | OP_DRIFTX | OP_QUADCHR)) != 0;
            if (!(slice && looped)) {  // an indivisible record: a thin element, or any record at element granularity
                const long long owes = slice ? 1 : ((o.op & OP_MARK) ? 1 : 0);
                if (pend_b + owes > cap || (long long)pend.size() == kTableRecords) rc = flush();
                if (rc != BT_OK) break;
                pend.push_back(o);
                pend_b += owes;
                continue;
            }
            long long left = o.count;  // slice granularity: one row per slice; a long element may be cut between two launches
            while (left > 0 && rc == BT_OK) {
                if (pend_b == cap || (long long)pend.size() == kTableRecords) rc = flush();
                if (rc != BT_OK) break;
                const long long take = left < cap - pend_b ? left : cap - pend_b;
                o.count = (int32_t)take;
                pend.push_back(o);
                pend_b += take;
                left -= take;
            }
        }
    }
    if (rc == BT_OK) rc = flush();
    if (rc == BT_OK) {
        b.gamma = gamma;
        b.s += b.lattice_length * (double)nturns;
        b.turn += nturns;
        if (cudaMemcpyAsync(host_moments, dev_out, (size_t)nrec * 42 * sizeof(double), cudaMemcpyDeviceToHost, b.stream) != cudaSuccess)
            rc = fail(BT_ERR_CUDA, "bt_track_diagnostics: copy of the records failed");
    }
    if (cudaStreamSynchronize(b.stream) != cudaSuccess && rc == BT_OK) rc = fail(BT_ERR_CUDA, "bt_track_diagnostics: stream synchronisation failed");
    return rc;
}

// Host-to-host walk: chunks of the bunch ride three streams, so that the H2D copy of chunk k+1, the walk of chunk k and
// the D2H copy of chunk k-1 overlap (PCIe is full duplex; particles are independent, so any partition is exact).  Every
// chunk runs the same plan of launches; a launch carries its record table as kernel parameters, so chunks on different
// streams may be at different launches of the plan (lattices whose RF changes the reference energy included).
int bt_track_host(bt_beam *beam, const double *const host_in[6], double *const host_out[6], int32_t nturns, int32_t nchunks) {
    if (!beam || !host_in || !host_out) return fail(BT_ERR_INVALID, "bt_track_host: NULL argument");
    for (int i = 0; i < 6; ++i)
        if (!host_in[i] || !host_out[i]) return fail(BT_ERR_INVALID, "bt_track_host: host array list has a NULL entry");
    if (nturns < 0) return fail(BT_ERR_INVALID, "bt_track_host: nturns < 0");
    if (nchunks < 1 || nchunks > 256) return fail(BT_ERR_INVALID, "bt_track_host: nchunks must be in [1, 256]");
    Beam &b = beam->b;
    if (b.lattice.empty()) return fail(BT_ERR_STATE, "bt_track_host: bt_lattice_set not called");
    if (!b.has_ref) return fail(BT_ERR_STATE, "bt_track_host: bt_beam_set_ref not called");
    if (nturns == 0 || nchunks == 1) {
        int rc = bt_beam_upload(beam, host_in);
        if (rc == BT_OK) rc = bt_track(beam, nturns);
        if (rc == BT_OK) rc = bt_beam_download(beam, host_out);
        return rc;
    }
    for (int i = 0; i < 3; ++i) {
        if (!b.pipe_stream[i]) BT_CUDA_TRY(cudaStreamCreateWithFlags(&b.pipe_stream[i], cudaStreamNonBlocking));
        if (!b.pipe_event[i]) BT_CUDA_TRY(cudaEventCreateWithFlags(&b.pipe_event[i], cudaEventDisableTiming));
    }
    // One plan serves every chunk when the whole call fits one window (the usual case).  Otherwise each chunk walks the
    // windows on its own, rebuilding them (bounded host memory; the tables are cheap next to a chunk's copies).
    WalkPlan plan;
    const bool whole = plan_walk(b, b.gamma, nturns, plan) == nturns;
    double gamma_after = plan.gamma_after;
    set_current_storage(&b, false);  // the result lives in the home arrays, in the caller's order
    // the chunk streams start after everything already queued on the beam's stream
    BT_CUDA_TRY(cudaEventRecord(b.pipe_event[0], b.stream));
    for (int i = 0; i < 3; ++i) BT_CUDA_TRY(cudaStreamWaitEvent(b.pipe_stream[i], b.pipe_event[0], 0));
    const long long gran = 1024;  // keeps every chunk's arrays as aligned as the whole arrays
    const long long len = ((b.n + nchunks - 1) / nchunks + gran - 1) / gran * gran;
    int rc = BT_OK;
    cudaError_t ce = cudaSuccess;
    int k = 0;
    for (long long off = 0; off < b.n && rc == BT_OK && ce == cudaSuccess; off += len, ++k) {
        const long long m = b.n - off < len ? b.n - off : len;
        cudaStream_t st = b.pipe_stream[k % 3];
        for (int i = 0; i < 6 && ce == cudaSuccess; ++i)
            ce = cudaMemcpyAsync(b.q[i] + off, host_in[i] + off, (size_t)m * sizeof(double), cudaMemcpyHostToDevice, st);
        if (ce != cudaSuccess) break;
        TrackRange r;
        r.off = off, r.n = m, r.geom_n = b.n, r.stream = st;
        b.range = &r;
        rc = whole ? run_plan(b, plan) : run_walk(b, nturns, plan, &gamma_after);
        b.range = nullptr;
        for (int i = 0; i < 6 && rc == BT_OK && ce == cudaSuccess; ++i)
            ce = cudaMemcpyAsync(host_out[i] + off, b.q[i] + off, (size_t)m * sizeof(double), cudaMemcpyDeviceToHost, st);
    }
    // join the chunk streams on every path (an error above must not leave them running behind the caller's back)
    for (int i = 0; i < 3; ++i) {
        if (cudaEventRecord(b.pipe_event[i], b.pipe_stream[i]) == cudaSuccess) cudaStreamWaitEvent(b.stream, b.pipe_event[i], 0);
    }
    const cudaError_t se = cudaStreamSynchronize(b.stream);
    b.permuted = false;  // storage order = the caller's order
    b.deposits_since_sort = 0;
    ++b.storage_epoch;
    if (rc != BT_OK) return rc;
    if (ce != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_track_host: copy: ") + cudaGetErrorString(ce));
    if (se != cudaSuccess) return fail(BT_ERR_CUDA, std::string("bt_track_host: ") + cudaGetErrorString(se));
    b.gamma = gamma_after;
    b.s += b.lattice_length * (double)nturns;
    b.turn += nturns;
    return BT_OK;
}

int bt_track_last_launch(const bt_beam *beam, int32_t *grid_dim, int32_t *block_dim, int32_t *ppt, int32_t *smem) {
    if (!beam) return fail(BT_ERR_INVALID, "bt_track_last_launch: beam is NULL");
    const TrackLaunchInfo &li = beam->b.last_launch;
    if (grid_dim) *grid_dim = li.grid;
    if (block_dim) *block_dim = li.block;
    if (ppt) *ppt = li.ppt;
    if (smem) *smem = li.smem;
    return BT_OK;
}

// ---- grid ---------------------------------------------------------------------------------------

int bt_grid_create(bt_grid **out, int32_t nx, int32_t ny, int32_t nz, const double lo[3], const double d[3]) {
    if (!out) return fail(BT_ERR_INVALID, "bt_grid_create: out is NULL");
    *out = nullptr;
    if (!lo || !d) return fail(BT_ERR_INVALID, "bt_grid_create: NULL argument");
    if (nx < 2 || ny < 2 || nz < 2) return fail(BT_ERR_INVALID, "bt_grid_create: need >= 2 nodes per axis");
    const int64_t nn = (int64_t)nx * ny * nz;
    if (nn > ((int64_t)1 << 31) - 1) return fail(BT_ERR_INVALID, "bt_grid_create: nx*ny*nz overflows int32");
    for (int a = 0; a < 3; ++a)
        if (!(d[a] > 0.0) || !isfinite(d[a]) || !isfinite(lo[a])) return fail(BT_ERR_INVALID, "bt_grid_create: d <= 0 or not finite");
    bt_grid *h = new (std::nothrow) bt_grid();
    if (!h) return fail(BT_ERR_OOM, "bt_grid_create: host allocation failed");
    Grid &g = h->g;
    g.nx = nx;
    g.ny = ny;
    g.nz = nz;
    g.nn = nn;
    for (int a = 0; a < 3; ++a) {
        g.lo[a] = lo[a];
        g.d[a] = d[a];
        g.inv_d[a] = 1.0 / d[a];  // R11: computed once on the host
    }
    cudaError_t e = cudaMalloc(&g.rho, (size_t)nn * sizeof(double));
    if (e == cudaSuccess) e = cudaMemset(g.rho, 0, (size_t)nn * sizeof(double));
    if (e != cudaSuccess) {
        if (g.rho) cudaFree(g.rho);
        delete h;
        return fail(e == cudaErrorMemoryAllocation ? BT_ERR_OOM : BT_ERR_CUDA, std::string("bt_grid_create: ") + cudaGetErrorString(e));
    }
    *out = h;
    return BT_OK;
}

void bt_grid_destroy(bt_grid *grid) {
    if (!grid) return;
    cudaDeviceSynchronize();
    poisson_free(&grid->g);
    if (grid->g.rho) cudaFree(grid->g.rho);
    if (grid->g.field) cudaFree(grid->g.field);
    if (grid->g.phi) cudaFree(grid->g.phi);
    if (grid->g.done) cudaEventDestroy(grid->g.done);
    delete grid;
}

int bt_grid_set_field(bt_grid *grid, const double *Ex, const double *Ey, const double *Ez, int on_device) {
    if (!grid || !Ex || !Ey || !Ez) return fail(BT_ERR_INVALID, "bt_grid_set_field: NULL argument");
    Grid &g = grid->g;
    const size_t bytes = (size_t)g.nn * sizeof(double);
    if (!g.field) BT_CUDA_TRY(cudaMalloc(&g.field, bytes * 4));
    cudaStream_t s = g.last_stream;  // ordered after whatever used the grid last; the caller's Ex/Ey/Ez must be ready on it
    if (on_device) {
        const int rc = launch_field_pack(&g, Ex, Ey, Ez, s);
        return rc != BT_OK ? rc : grid_release(&g, s);
    }
    double *tmp = nullptr;
    BT_CUDA_TRY(cudaMalloc(&tmp, bytes * 3));
    cudaError_t e = cudaMemcpyAsync(tmp, Ex, bytes, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(tmp + g.nn, Ey, bytes, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(tmp + 2 * g.nn, Ez, bytes, cudaMemcpyHostToDevice, s);
    int rc = BT_OK;
    if (e != cudaSuccess)
        rc = fail(BT_ERR_CUDA, std::string("bt_grid_set_field: ") + cudaGetErrorString(e));
    else
        rc = launch_field_pack(&g, tmp, tmp + g.nn, tmp + 2 * g.nn, s);
    cudaStreamSynchronize(s);
    cudaFree(tmp);
    return rc != BT_OK ? rc : grid_release(&g, s);
}

int bt_grid_rho(bt_grid *grid, double **dev_rho_out) {
    if (!grid || !dev_rho_out) return fail(BT_ERR_INVALID, "bt_grid_rho: NULL argument");
    *dev_rho_out = grid->g.rho;
    return BT_OK;
}

int bt_grid_download_rho(bt_grid *grid, double *host_rho) {
    if (!grid || !host_rho) return fail(BT_ERR_INVALID, "bt_grid_download_rho: NULL argument");
    Grid &g = grid->g;
    BT_CUDA_TRY(cudaMemcpyAsync(host_rho, g.rho, (size_t)g.nn * sizeof(double), cudaMemcpyDeviceToHost, g.last_stream));
    BT_CUDA_TRY(cudaStreamSynchronize(g.last_stream));
    return BT_OK;
}

int bt_grid_solve_poisson(bt_grid *grid, double gz, void *cuda_stream) {
    if (!grid) return fail(BT_ERR_INVALID, "bt_grid_solve_poisson: grid is NULL");
    if (!(gz > 0.0) || !isfinite(gz)) return fail(BT_ERR_INVALID, "bt_grid_solve_poisson: gz must be positive and finite");
    Grid &g = grid->g;
    if ((int64_t)8 * g.nn > ((int64_t)1 << 31) - 1) return fail(BT_ERR_UNSUPPORTED, "bt_grid_solve_poisson: padded grid exceeds 2^31 nodes");
    int rc = grid_acquire(&g, (cudaStream_t)cuda_stream);  // rho may still be in flight on a beam's stream
    if (rc == BT_OK) rc = poisson_solve(&g, gz, (cudaStream_t)cuda_stream);
    return rc != BT_OK ? rc : grid_release(&g, (cudaStream_t)cuda_stream);
}

int bt_grid_download_phi(bt_grid *grid, double *host_phi) {
    if (!grid || !host_phi) return fail(BT_ERR_INVALID, "bt_grid_download_phi: NULL argument");
    Grid &g = grid->g;
    if (!g.phi) return fail(BT_ERR_STATE, "bt_grid_download_phi: bt_grid_solve_poisson not called");
    BT_CUDA_TRY(cudaMemcpyAsync(host_phi, g.phi, (size_t)g.nn * sizeof(double), cudaMemcpyDeviceToHost, g.last_stream));
    BT_CUDA_TRY(cudaStreamSynchronize(g.last_stream));
    return BT_OK;
}

int bt_grid_download_field(bt_grid *grid, double *host_Ex, double *host_Ey, double *host_Ez) {
    if (!grid || !host_Ex || !host_Ey || !host_Ez) return fail(BT_ERR_INVALID, "bt_grid_download_field: NULL argument");
    Grid &g = grid->g;
    if (!g.field) return fail(BT_ERR_STATE, "bt_grid_download_field: no field (bt_grid_set_field / bt_grid_solve_poisson not called)");
    double *tmp = nullptr;
    BT_CUDA_TRY(cudaMalloc(&tmp, (size_t)g.nn * 3 * sizeof(double)));
    int rc = field_unpack(&g, tmp, tmp + g.nn, tmp + 2 * g.nn, g.last_stream);
    double *host[3] = {host_Ex, host_Ey, host_Ez};
    for (int c = 0; c < 3 && rc == BT_OK; ++c)
        if (cudaMemcpyAsync(host[c], tmp + c * g.nn, (size_t)g.nn * sizeof(double), cudaMemcpyDeviceToHost, g.last_stream) != cudaSuccess)
            rc = fail(BT_ERR_CUDA, "bt_grid_download_field: copy failed");
    cudaStreamSynchronize(g.last_stream);
    cudaFree(tmp);
    return rc;
}

int bt_grid_set_particle_shape(bt_grid *grid, int32_t order) {
    if (!grid) return fail(BT_ERR_INVALID, "bt_grid_set_particle_shape: grid is NULL");
    if (order != 1 && order != 2) return fail(BT_ERR_UNSUPPORTED, "bt_grid_set_particle_shape: order must be 1 (CIC) or 2 (quadratic B-spline)");
    Grid &g = grid->g;
    if (order == 2 && (g.nx < 3 || g.ny < 3 || g.nz < 3)) return fail(BT_ERR_INVALID, "bt_grid_set_particle_shape: order 2 needs >= 3 nodes per axis");
    g.order = order;
    return BT_OK;
}

int bt_deposit_cic(bt_beam *beam, bt_grid *grid, double q_weight, double zscale, int zero_first) {
    if (!beam || !grid) return fail(BT_ERR_INVALID, "bt_deposit_cic: NULL argument");
    if (!isfinite(q_weight) || !isfinite(zscale)) return fail(BT_ERR_INVALID, "bt_deposit_cic: q_weight or zscale not finite");
    Beam &b = beam->b;
    Grid &g = grid->g;
    int arc = grid_acquire(&g, b.stream);
    if (arc != BT_OK) return arc;
    if (b.resort_interval > 0) {  // S4 cadence: re-bin the storage every resort_interval deposits (the first one included)
        if (b.deposits_since_sort % b.resort_interval == 0) {
            const int rc = sort_by_cell(&b, &g, zscale);
            if (rc != BT_OK) return rc;
            b.deposits_since_sort = 0;
        }
        b.deposits_since_sort += 1;
    }
    if (zero_first) BT_CUDA_TRY(cudaMemsetAsync(g.rho, 0, (size_t)g.nn * sizeof(double), b.stream));
    arc = launch_deposit(&b, &g, q_weight, zscale);
    return arc != BT_OK ? arc : grid_release(&g, b.stream);
}

int bt_beam_set_resort_interval(bt_beam *beam, int32_t every_n_deposits) {
    if (!beam) return fail(BT_ERR_INVALID, "bt_beam_set_resort_interval: beam is NULL");
    if (every_n_deposits < 0) return fail(BT_ERR_INVALID, "bt_beam_set_resort_interval: negative interval");
    beam->b.resort_interval = every_n_deposits;
    beam->b.deposits_since_sort = 0;
    return BT_OK;
}

int bt_beam_moments(bt_beam *beam, double host_mean[6], double host_cov[36]) {
    if (!beam || !host_mean || !host_cov) return fail(BT_ERR_INVALID, "bt_beam_moments: NULL argument");
    return launch_moments(&beam->b, host_mean, host_cov);
}

int bt_beam_moments_device(bt_beam *beam, double *dev_out) {
    if (!beam || !dev_out) return fail(BT_ERR_INVALID, "bt_beam_moments_device: NULL argument");
    return launch_moments_async(&beam->b, dev_out);
}

int bt_gather_kick(bt_beam *beam, const bt_grid *grid, const double coef[3], double zscale, double half_drift_before,
                   double half_drift_after) {
    if (!beam || !grid || !coef) return fail(BT_ERR_INVALID, "bt_gather_kick: NULL argument");
    if (!isfinite(zscale) || !isfinite(coef[0]) || !isfinite(coef[1]) || !isfinite(coef[2]))
        return fail(BT_ERR_INVALID, "bt_gather_kick: coef or zscale not finite");
    if (!(half_drift_before >= 0.0) || !(half_drift_after >= 0.0) || !isfinite(half_drift_before) || !isfinite(half_drift_after))
        return fail(BT_ERR_INVALID, "bt_gather_kick: negative or non-finite drift length");
    Beam &b = beam->b;
    Grid &g = const_cast<Grid &>(grid->g);  // const for the caller: the field is only read; the ordering event is bookkeeping
    if (!g.field) return fail(BT_ERR_STATE, "bt_gather_kick: bt_grid_set_field not called");
    if (!b.has_ref) return fail(BT_ERR_STATE, "bt_gather_kick: bt_beam_set_ref not called");
    int rc = grid_acquire(&g, b.stream);  // the field may still be in flight on the stream of bt_grid_solve_poisson
    if (rc != BT_OK) return rc;
    const double bg2 = b.gamma * b.gamma - 1.0;
    const double bg = sqrt(bg2);
    const double tcb = half_drift_before / (bg * bg), tca = half_drift_after / (bg * bg);  // R4
    rc = launch_gather_kick(&b, &g, coef, zscale, half_drift_before, tcb, half_drift_after, tca);
    if (rc == BT_OK) rc = grid_release(&g, b.stream);
    if (rc != BT_OK) return rc;
    b.s += half_drift_before + half_drift_after;
    return BT_OK;
}

}  // extern "C"
