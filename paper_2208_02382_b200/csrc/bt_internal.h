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

#define BT_CUDA_TRY(expr)                                                                        \
    do {                                                                                         \
        cudaError_t _e = (expr);                                                                 \
        if (_e != cudaSuccess)                                                                   \
            return ::bt::fail(_e == cudaErrorMemoryAllocation ? BT_ERR_OOM : BT_ERR_CUDA,        \
                              std::string(#expr) + ": " + cudaGetErrorString(_e));               \
    } while (0)

// ---- device op records (S1): one 64-byte record per lattice element ----------------------------
// The host turns each bt_element into the coefficients of ONE slice map of length h = ds/nslice.
enum Op : int32_t {
    OP_DRIFT = 0,  // c0 = h, c1 = h/(b0 g0)^2
    OP_QUAD = 1,   // x' = c0 x + c1 px, px' = c2 x + c0 px ; y' = c3 y + c4 py, py' = c5 y + c3 py ; t += c6 pt
    OP_SBEND = 2,  // c0 = C, c1 = rho S, c2 = -S/rho, c3 = r16, c4 = r26, c5 = r56, c6 = h   (r51 = -r26, r52 = -r16)
    OP_EDGE = 3,   // px += c0 x ; py += c1 y
    OP_SEXT = 4,   // normal sextupole: px -= c0 (x^2 - y^2) ; py += c1 x y      (c0 = Kn/2, c1 = Kn)
    OP_OCT = 5,    // normal octupole:  px -= c0 x (x^2 - 3y^2) ; py += c0 y (3x^2 - y^2)   (c0 = Kn/6)
    OP_MULT = 6,   // general thin multipole: c0 = m, c1 = Kn/(m-1)!, c2 = Ks/(m-1)!
    OP_RF = 7,     // px *= c0 ; py *= c0 ; pt = c0 pt + c1 t
    OP_COUNT
};

struct alignas(16) DevOp {
    int32_t op;
    int32_t nslice;
    double c[7];
};
static_assert(sizeof(DevOp) == 64, "DevOp must be 64 bytes");

struct TrackLaunchInfo {
    int32_t grid = 0, block = 0, ppt = 0, smem = 0;
};

struct Beam {
    int64_t n = 0;
    double *q[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    bool owns = false;
    bool aligned16 = false;
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
    DevOp *d_table = nullptr;  // device table(s)
    size_t d_table_cap = 0;    // in DevOps
    bool table_valid = false;  // d_table holds the single-turn table for the current lattice and gamma
    TrackLaunchInfo last_launch;
    // S4 cell binning: storage order != original order once sorted; ids[j] = original index of slot j
    bool permuted = false;
    int *ids = nullptr, *ids_tmp = nullptr;
    int *sort_key = nullptr, *sort_dest = nullptr, *sort_count = nullptr, *sort_block_sum = nullptr;
    long long sort_count_cap = 0;
    double *scratch = nullptr;  // one array of n doubles
};

struct Grid {
    int32_t nx = 0, ny = 0, nz = 0;
    double lo[3] = {0, 0, 0}, d[3] = {0, 0, 0}, inv_d[3] = {0, 0, 0};
    int64_t nn = 0;
    double *rho = nullptr;
    double *field = nullptr;  // interleaved (Ex,Ey,Ez,pad) per node: 4*nn doubles, or nullptr
    cudaStream_t last_stream = nullptr;
};

// ---- host precompute (S1/S3), bt_lattice.cpp part of bt_api.cu ---------------------------------
// Fills ops[0..n) for one pass over the lattice starting at reference gamma; returns gamma after.
double build_turn_table(const std::vector<bt_element> &lat, double gamma, DevOp *ops);

// ---- launchers --------------------------------------------------------------------------------
int launch_track(Beam *b, const DevOp *d_table, int32_t n_ops, int32_t nturns, int32_t turn_stride);
int launch_deposit(Beam *b, Grid *g, double q_weight, double zscale);
int launch_gather_kick(Beam *b, const Grid *g, const double coef[3], double zscale, double h_before,
                       double tc_before, double h_after, double tc_after);
int sort_by_cell(Beam *b, const Grid *g, double zscale);
int unpermute_to(Beam *b, int c, double *out);  // out[ids[j]] = q[c][j] on the beam's stream
int launch_field_pack(Grid *g, const double *ex, const double *ey, const double *ez, cudaStream_t s);

}  // namespace bt

struct bt_beam {
    bt::Beam b;
};
struct bt_grid {
    bt::Grid g;
};
