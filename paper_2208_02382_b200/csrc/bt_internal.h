// Internal declarations of libbt.so (not part of the ABI).  Product code: shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <string>
#include <vector>

#include "../../include/bt.h"

namespace bt {

// ---- error plumbing ---------------------------------------------------------------------------
void set_error(const std::string &msg);
int fail(int code, const std::string &msg);
extern std::atomic<int64_t> g_launch_count;

// Debug knobs (bt_debug_knob): A/B measurements and the tests that exercise every kernel variant.  -1 = measured default.
enum Knob { KNOB_TRACK_PPT = 0, KNOB_TRACK_BLOCK, KNOB_TRACK_FUSE, KNOB_DEPOSIT_MODE, KNOB_GATHER_MODE, KNOB_PLAN_WINDOW, KNOB_COUNT };
extern std::atomic<int32_t> g_knob[KNOB_COUNT];
static inline int knob(Knob k, int dflt) {
    const int v = g_knob[k].load(std::memory_order_relaxed);
    return v < 0 ? dflt : v;
}

#define BT_CUDA_TRY(expr)                                                                        \
    do {                                                                                         \
        cudaError_t _e = (expr);                                                                 \
        if (_e != cudaSuccess)                                                                   \
            return ::bt::fail(_e == cudaErrorMemoryAllocation ? BT_ERR_OOM : BT_ERR_CUDA,        \
                              std::string(#expr) + ": " + cudaGetErrorString(_e));               \
    } while (0)

// ---- device op records (S1): 64-byte records in the constant bank ------------------------------------
// The host turns each bt_element into the coefficients of ONE slice map of length h = ds/nslice.  Opcodes are
// one-hot so the kernel can dispatch with a short tree of uniform bit tests (track.cu).
enum Op : int32_t {
    OP_DRIFT1 = 1 << 0,   // one slice;  c0 = h, c1 = h/(b0 g0)^2
    OP_DRIFT = 1 << 1,    // count slices, same coefficients
    OP_QUAD1 = 1 << 2,    // one slice;  x' = c0 x + c1 px, px' = c2 x + c0 px ; y' = c3 y + c4 py, py' = c5 y + c3 py ; t += c6 pt
    OP_QUAD = 1 << 3,     // count slices, same coefficients
    OP_QUAD5 = 1 << 4,    // count groups of FIVE slices: a thick quad of nslice = 5a + b slices becomes {QUAD5, a} then
                          // {QUAD, b} / {QUAD1}, so the unrolled loop needs no remainder logic
    OP_SBEND = 1 << 5,    // count slices; c0 = C, c1 = rho S, c2 = -S/rho, c3 = r16, c4 = r26, c5 = r56, c6 = h (r51 = -r26, r52 = -r16)
    OP_EDGE = 1 << 6,     // px += c0 x ; py += c1 y
    OP_SEXT = 1 << 7,     // normal sextupole: px -= c0 (x^2 - y^2) ; py += c1 x y      (c0 = Kn/2, c1 = Kn)
    OP_OCT = 1 << 8,      // normal octupole:  px -= c2 x (x^2 - 3y^2) ; py += c2 y (3x^2 - y^2)   (c2 = Kn/6)
    OP_SEXTOCT = 1 << 9,  // OP_SEXT then OP_OCT (adjacent elements) in one dispatch; same arithmetic, same order
    OP_MULT = 1 << 10,    // general thin multipole: count = m, c0 = Kn/(m-1)!, c1 = Ks/(m-1)!
    OP_RF = 1 << 11,      // px *= c0 ; py *= c0 ; pt = c0 pt + c1 t
    OP_DRIFTX = 1 << 13,  // exact drift (R17), count slices: c0 = h, c1 = 1/beta0
    OP_QUADCHR = 1 << 15, // chromatic quad (R20), count slices: c0 = h, c1 = 1/beta0, c2 = |k|, c3 = +1 (k > 0: x focusing) / -1 / 0 (k = 0)
    OP_RFSIN = 1 << 14,   // sinusoidal short RF (R18): px *= c0; py *= c0; pt = c0 pt + c1 (cos(c2 t + c3) - c4)
    OP_TAILDRIFT = 1 << 12,  // modifier of SEXT/OCT/SEXTOCT: the single-slice drift that follows the kick rides in the
                             // same record (c3 = h, c4 = h/(b0 g0)^2); same arithmetic, same order, one dispatch less
    OP_MARK = 1 << 17,      // diagnostics tables only: an element ends with this record (a statistics row follows its last slice)
    OP_HALFCELL = 1 << 16   // head of a run of `count` half cells [QUAD1][SEXTOCT|TAILDRIFT]: this record holds the first quad's
                            // coefficients (c0..c6 as QUAD1), the next one the kicks' and the drift's (as SEXTOCT|TAILDRIFT), and so
                            // on for 2*count records, which the walk consumes in one dispatch
};

struct alignas(16) DevOp {
    int32_t op;
    int32_t count;  // slices (DRIFT, QUAD, SBEND), groups of five slices (QUAD5), order m (MULT), else 1
    double c[7];
};
static_assert(sizeof(DevOp) == 64, "DevOp must be 64 bytes");

// The record table of a launch travels in the kernel's parameter space (32 764 bytes on sm_70+; constant bank 0).
constexpr int kTableRecords = 510;      // 80-byte launch header + 510 x 64 B = 32 720 B
constexpr int kTableRecordsSmall = 30;  // short lattices: 2 000 B of parameters
constexpr int kMaxDevices = 64;

struct TrackLaunchInfo {
    int32_t grid = 0, block = 0, ppt = 0, smem = 0;
    int64_t launches = 0;  // fused-walk kernels launched by this beam so far
};

// A sub-range of the beam walked on its own stream (bt_track_host): launch_track then works on [off, off + n) of the
// arrays; the launch geometry is chosen for geom_n particles (the whole bunch), not for the chunk.
struct TrackRange {
    long long off = 0, n = 0, geom_n = 0;
    cudaStream_t stream = nullptr;
};

struct Beam {
    int64_t n = 0;
    double *q[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};     // where the particles are now (home or alt)
    double *home[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};  // the caller's arrays (borrowed) or the library's
    double *alt[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // library-owned partner set (bt_beam_sort_by_cell ping-pong)
    bool in_alt = false;
    bool pingpong = false;       // a sort may leave the bunch in alt (set at creation: library-owned storage yes, lent arrays no)
    int64_t storage_epoch = 0;   // bumped whenever the bunch changes arrays or storage order (bt_beam_storage)
    double *dl_tmp = nullptr;    // n doubles: bt_beam_download's un-permute scratch when the idle set is the caller's (lent) arrays
    bool owns = false;
    bool aligned16 = false;
    bool aligned32 = false;  // all six arrays 32-byte aligned: 256-bit lane-run access in the grid kernels
    int device = 0;
    int num_sms = 0;
    int max_smem_optin = 0;
    cudaStream_t stream = nullptr;
    // reference particle (R2)
    bool has_ref = false;
    double gamma = 0.0, mass_MeV = 0.0, charge_qe = 0.0, s = 0.0;
    int64_t turn = 0;
    // lattice
    std::vector<bt_element> lattice;
    bool energy_changes = false;  // some SHORTRF with Vhat*cos(phi) != 0
    double lattice_length = 0.0;
    std::vector<DevOp> h_table;  // single-turn record table for the current lattice and gamma (static lattices)
    bool table_valid = false;    // h_table is up to date
    int table_fuse = 1;          // value of the track_fuse knob h_table was built under
    double table_slots = 0.0;    // FP64 slots per particle per turn of that table
    TrackLaunchInfo last_launch;
    // S4 cell binning: storage order != original order once sorted; ids[j] = original index of slot j
    bool permuted = false;
    int32_t resort_interval = 0;      // bt_beam_set_resort_interval: re-sort every n-th bt_deposit_cic (0 = never)
    int32_t deposits_since_sort = 0;
    int *ids = nullptr, *ids_tmp = nullptr;
    int *sort_count = nullptr, *sort_block_sum = nullptr;
    long long sort_count_cap = 0;
    const TrackRange *range = nullptr;  // non-NULL only inside bt_track_host
    cudaStream_t pipe_stream[3] = {nullptr, nullptr, nullptr};  // bt_track_host: chunk streams, created on first use
    cudaEvent_t pipe_event[3] = {nullptr, nullptr, nullptr};
    double *mom_buf = nullptr;  // beam statistics: out[42], pad, per-block partials, ticket (moments.cu)
    double *mom_host = nullptr; // 42 doubles of mapped pinned host memory: bt_beam_moments' result lands there without a copy
    double *mom_host_dev = nullptr;  // device address of mom_host
    int mom_blocks = 0;         // resident blocks of moments_kernel on this device (occupancy query, once)
    double *diag_rows = nullptr;  // bt_track_diagnostics: per-(boundary, warp) rows of partial sums, kept between calls
    size_t diag_rows_bytes = 0;
    double *diag_out = nullptr;   // bt_track_diagnostics: records (42 doubles per boundary) + the provisional centre, kept between calls
    size_t diag_out_bytes = 0;
};

struct Grid {
    int32_t nx = 0, ny = 0, nz = 0;
    int32_t order = 1;  // particle shape: 1 = CIC (R11), 2 = quadratic B-spline (R16)
    double lo[3] = {0, 0, 0}, d[3] = {0, 0, 0}, inv_d[3] = {0, 0, 0};
    int64_t nn = 0;
    double *rho = nullptr;
    double *field = nullptr;  // interleaved (Ex,Ey,Ez,pad) per node: 4*nn doubles, or nullptr
    double *phi = nullptr;    // potential at the nodes (bt_grid_solve_poisson), or nullptr
    void *poisson = nullptr;  // solver state (plans, padded buffers, cached Green transform), poisson.cu
    // cross-stream ordering: every operation on the grid's arrays waits for `done` of the previous one when it runs on
    // another stream (deposit on the beam's stream, solve on the caller's, gather on the beam's again, ...)
    cudaStream_t last_stream = nullptr;
    cudaEvent_t done = nullptr;
    bool done_valid = false;
};

// ---- host precompute (S1/S3), in bt_api.cu ------------------------------------------------------
// Appends the records of one pass over the lattice starting at reference gamma; returns gamma after.
// The number of records appended depends on the lattice only (not on gamma).  *slots (may be NULL) receives the
// FP64 instruction slots one particle spends in this pass (minimal DFMA/DMUL sequences).
double build_turn_table(const std::vector<bt_element> &lat, double gamma, std::vector<DevOp> &out, double *slots, int diag = 0);

int grid_acquire(Grid *g, cudaStream_t s);  // make `s` wait for the last operation enqueued on the grid (no-op on the same stream)
int grid_release(Grid *g, cudaStream_t s);  // record that the grid's latest operation was enqueued on `s`

// ---- launchers --------------------------------------------------------------------------------
// One fused-walk launch: n_ops (<= kTableRecords) host records travel as kernel parameters and are walked nturns times.
// slots_per_record (FP64 slots per particle per record, averaged) steers the particles-per-thread choice.
int launch_track(Beam *b, const DevOp *h_table, int32_t n_ops, int32_t nturns, double slots_per_record);
// Diagnostics walk (un-fused records, OP_MARK at element ends): one walk launch writing `nb` boundaries' rows + their combination
// into out[nb][42].  diag_warps = rows per boundary for this beam (sizes the row buffer).
int launch_track_diag(Beam *b, const DevOp *h_table, int32_t n_ops, int slice_gran, int nb, const double *centre, double *rows, double *out);
int diag_warps(const Beam *b, int *particles_per_thread, int *block);
int launch_moments_centre(Beam *b, double *dev_centre);  // provisional centre k[6] of the current bunch (moments.cu)
int launch_deposit(Beam *b, Grid *g, double q_weight, double zscale);
int launch_gather_kick(Beam *b, const Grid *g, const double coef[3], double zscale, double h_before,
                       double tc_before, double h_after, double tc_after);
int sort_by_cell(Beam *b, const Grid *g, double zscale);
int unpermute_to(Beam *b, int c, double *out);  // out[ids[j]] = q[c][j] on the beam's stream
int ensure_alt_storage(Beam *b);                 // allocates the partner arrays and the id arrays on first use
void set_current_storage(Beam *b, bool use_alt); // q = alt or home; refreshes the alignment flags
int rehome(Beam *b);                             // bunch in alt -> device copy back into home (storage order kept); no-op in home
int launch_moments(Beam *b, double host_mean[6], double host_cov[36]);  // synchronises the beam's stream
int launch_moments_async(Beam *b, double *dev_out);                      // 42 doubles to device memory, no synchronisation
int poisson_solve(Grid *g, double gz, cudaStream_t stream);  // rho -> phi -> field records
void poisson_free(Grid *g);
int field_unpack(Grid *g, double *ex, double *ey, double *ez, cudaStream_t stream);  // device outputs
int launch_field_pack(Grid *g, const double *ex, const double *ey, const double *ez, cudaStream_t s);

}  // namespace bt

struct bt_beam {
    bt::Beam b;
};
struct bt_grid {
    bt::Grid g;
};
