/*
 * bt.h -- C-ABI of libbt.so: the data-parallel hot path of the s-based beam-dynamics PIC method of
 * arxiv 2208.02382 (Huebl et al., "Next generation computational tools for the modeling and design
 * of particle accelerators at exascale"), built for NVIDIA B200 (sm_100a).
 *
 * Citation convention: "P:l.N" = line N of the paper text; "R<n>" = reading n of the
 * paper stated in DESIGN.md section 3 (the paper prints no formulas; P:l.47 states the method:
 * "Tracking through lattice elements is performed by pushing particles in s using a symplectic
 * map ... accurate through linear order").
 *
 * General rules
 *  - Every function returns int: BT_OK (0) or a negative bt_status.  No exception crosses the ABI.
 *    bt_last_error() returns a thread-local, human-readable description of the last failure.
 *  - "host" pointers are ordinary CPU memory (pinned memory makes uploads/downloads asynchronous
 *    to the host until the next synchronising call); "device" pointers are CUDA global memory of
 *    the device that was current when bt_beam_create was called.
 *  - All floating point data is IEEE fp64.  Coordinates (R1): x [m], px = Px/p0, y [m], py = Py/p0,
 *    t = c*(arrival time - reference arrival time) [m], pt = -(E - E0)/(p0 c); array order is always
 *    x, px, y, py, t, pt; each is a separate contiguous array of n doubles (SoA).
 *  - Asynchrony: calls enqueue work on the beam's CUDA stream and return.  bt_beam_download,
 *    bt_grid_download_rho and bt_sync synchronise that stream.  A bt_grid used with a beam is
 *    accessed on that beam's stream.
 *  - Arguments are validated before anything is launched; an invalid call changes no state.
 *  - There is no CPU fallback: without a CUDA device every entry point that touches the device
 *    fails with BT_ERR_CUDA.
 *  - Particle order seen through bt_beam_upload / bt_beam_download never changes.  bt_beam_ptrs exposes the
 *    STORAGE order, which equals the caller's order unless the caller has asked for bt_beam_sort_by_cell
 *    (then bt_beam_ids maps storage slots to original indices).  Arrays lent to bt_beam_create hold the bunch at all
 *    times unless the caller opts in to bt_beam_set_sort_pingpong.
 *  - NaN/Inf coordinates are not checked on the hot path; in deposit/gather they count as
 *    "outside the grid" (R13).
 */
#ifndef BT_H_
#define BT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BT_VERSION 100 /* 0.1.0 */

typedef struct bt_beam bt_beam; /* opaque: 6 device arrays (owned or borrowed), reference particle, lattice tables */
typedef struct bt_grid bt_grid; /* opaque: rho (nx*ny*nz doubles) and optionally a 3-component node field     */

typedef enum {
    BT_OK = 0,
    BT_ERR_INVALID = -1,     /* bad argument (null, n <= 0, nslice < 1, ds < 0, rc == 0, cos(psi) == 0, ...) */
    BT_ERR_CUDA = -2,        /* a CUDA runtime call failed; text in bt_last_error()                          */
    BT_ERR_OOM = -3,         /* host or device allocation failed                                             */
    BT_ERR_STATE = -4,       /* call order: bt_track before bt_lattice_set / bt_beam_set_ref, no field set..  */
    BT_ERR_UNSUPPORTED = -5  /* valid request this build does not implement                                  */
} bt_status;

/* Element kinds (P:l.86-91 Drift, Quad; P:l.108, l.124 name the others). */
typedef enum {
    BT_DRIFT = 0,     /* R4 */
    BT_QUAD = 1,      /* R5 thick quadrupole, k > 0 focuses x */
    BT_SBEND = 2,     /* R6 sector bend, no field index */
    BT_DIPEDGE = 3,   /* R7 thin pole-face rotation with fringe correction */
    BT_MULTIPOLE = 4, /* R8 thin multipole kick */
    BT_SHORTRF = 5,   /* R9 short RF cavity, linearised, energy kick only, updates the reference energy */
    /* non-linearised maps (P:l.168 "non-linear elements, RF-modeling"): */
    BT_DRIFT_EXACT = 6, /* R17: ps = sqrt(1 - 2pt/beta0 + pt^2 - px^2 - py^2); x += h px/ps; y += h py/ps;
                           t += h ((1/beta0 - pt)/ps - 1/beta0)  -- straight line with the exact time of flight */
    BT_QUAD_CHROMATIC = 8, /* R20: thick quad with focusing k/(1+delta) per particle and the second-order path length;
                              closed-form flow of H = -(1+d) + (px^2+py^2)/(2(1+d)) + k(x^2-y^2)/2 - pt/beta0; p0 = k */
    BT_SHORTRF_SIN = 7  /* R18: R9 without the expansion in t: pt = r pt - (Vhat/(bg)_f)(cos(k_rf t + phi) - cos(phi)),
                           px *= r, py *= r; same reference-energy update as R9 */
} bt_element_type;

/*
 * One lattice element: 64 bytes of plain data, caller-owned, copied by bt_lattice_set.
 * Mirrors the user-facing element vocabulary of the paper's Listing 1, e.g.
 * elements.Quad(ds=1.0, k=1.0, nslice=ns) (P:l.88).
 *   type    bt_element_type
 *   nslice  >= 1; the element is applied as nslice maps of length ds/nslice (R3; P:l.47, l.87).
 *           Thin elements (DIPEDGE, MULTIPOLE, SHORTRF, SHORTRF_SIN) must have nslice == 1.
 *   ds      length [m], >= 0; ignored for the map of thin elements but still added to s.
 *   p[6]    QUAD, QUAD_CHROMATIC: p0 = k [m^-2]
 *           SBEND:     p0 = rc [m], signed bending radius, != 0
 *           DIPEDGE:   p0 = psi [rad], p1 = rc [m] (!= 0), p2 = g [m] full gap, p3 = K fringe integral
 *           MULTIPOLE: p0 = m (integer 1..10; 1 dipole, 2 quad, 3 sext, 4 oct), p1 = Kn, p2 = Ks
 *                      (integrated strengths [m^-(m-1)], MAD-X sign: Kn > 0 at m = 2 focuses x)
 *           SHORTRF, SHORTRF_SIN: p0 = Vhat = qV/(mc^2), p1 = frequency [Hz], p2 = phase [deg] (cosine convention)
 *           DRIFT_EXACT: none
 *           unused entries are ignored.
 */
typedef struct {
    int32_t type;
    int32_t nslice;
    double ds;
    double p[6];
} bt_element;

/* ---- beam (particle container, S0) ---------------------------------------------------------- */

/*
 * Create a beam of n particles (n >= 1) on the current CUDA device.
 *   dev_ptrs   NULL: the library allocates 6 arrays of n doubles (256-byte aligned, uninitialised).
 *              else: 6 device pointers, BORROWED -- the caller (e.g. torch.empty(n, dtype=float64,
 *              device="cuda")) keeps them alive until bt_beam_destroy and frees them; each must be
 *              8-byte aligned (16-byte alignment enables the vectorised path).
 *   cuda_stream  a cudaStream_t cast to void* (0 = legacy default stream); all work of this beam is
 *              enqueued there.
 * Mirrors ImpactX() + add_particles(..., npart) (P:l.58, l.81).
 */
int bt_beam_create(bt_beam **out, int64_t n, double *const dev_ptrs[6], void *cuda_stream);
void bt_beam_destroy(bt_beam *beam);

/*
 * Reference particle (R2): kinetic energy [MeV] (> 0), rest mass [MeV] (> 0), charge [e] (informational).
 * gamma0 = 1 + E_kin/mc^2.  Resets s = 0 and turn = 0 and invalidates the coefficient tables (they are
 * rebuilt by the next bt_track).  Mirrors ref_particle().set_energy_MeV(energy_MeV, mass_MeV) (P:l.82-83).
 */
int bt_beam_set_ref(bt_beam *beam, double kin_energy_MeV, double mass_MeV, double charge_qe);
int bt_beam_get_ref(const bt_beam *beam, double *gamma, double *s, int64_t *turn); /* any out may be NULL */

/* Copy 6 host arrays of n doubles to / from the device arrays (order x,px,y,py,t,pt). upload is
 * enqueued (the host arrays must stay valid until the next synchronising call unless they are pageable
 * memory); download returns after the data has arrived. */
int bt_beam_upload(bt_beam *beam, const double *const host[6]);
int bt_beam_download(const bt_beam *beam, double *const host[6]);
/* Zero-copy view of the 6 device arrays the particles live in (P:l.102 "zero-copy access"), in STORAGE order.
 * Arrays LENT to bt_beam_create always hold the bunch: these are the caller's own pointers, whatever was called in between,
 * and the library never writes them except to update the bunch (external code holding the same pointers -- torch, cupy,
 * numba -- keeps seeing the particles).  A sort works out of place, into a library-owned partner set, and copies the result
 * back (one device copy, 96 bytes of traffic per particle and sort).
 * Ping-pong mode skips that copy: a sort leaves the bunch in the partner set and the next one moves it back (a particle's
 * data crosses memory once per sort).  It is the default for arrays the LIBRARY allocated (dev_ptrs == NULL) and opt-in for
 * lent arrays (bt_beam_set_sort_pingpong): then the lent arrays are stale after every other sort -- including the sorts
 * bt_deposit_cic triggers under bt_beam_set_resort_interval -- so ask bt_beam_ptrs again after anything that may sort, or
 * compare bt_beam_storage's epoch, or call bt_beam_rehome before handing the arrays to other code.
 * bt_beam_upload and bt_track_host always return the bunch to the original arrays. */
int bt_beam_ptrs(bt_beam *beam, double *dev_ptrs_out[6]);
/* enable != 0: sorts may leave the bunch in the partner arrays (see bt_beam_ptrs); 0: every sort ends in the arrays of
 * bt_beam_create, and a bunch that is in the partner set now is copied back. */
int bt_beam_set_sort_pingpong(bt_beam *beam, int enable);
/* Bring the bunch back into the arrays of bt_beam_create if a ping-pong sort left it elsewhere (device copy on the beam's
 * stream, storage order and bt_beam_ids unchanged); no-op otherwise. */
int bt_beam_rehome(bt_beam *beam);
/* Where the bunch is: *in_home = 1 iff bt_beam_ptrs currently returns the arrays of bt_beam_create; *epoch counts the
 * events that changed the arrays or the storage order (sort, re-home, upload, bt_track_host) since creation -- a caller
 * caching pointers or ids re-reads them when it moves.  Either out may be NULL. */
int bt_beam_storage(const bt_beam *beam, int32_t *in_home, int64_t *epoch);
int64_t bt_beam_size(const bt_beam *beam);

/*
 * Cell binning (S4; B:north_star "bins particles by cell").  Physically reorders the beam's six arrays by
 * the linear index (k*ny + j)*nx + i of the lowest node of each particle's stencil on `grid` for the grid's particle shape
 * (order 1: the cell's lower-corner node, R11 canonical index; order 2: nearest node - 1, R16; third axis zscale*t;
 * particles outside the grid go last), by a counting sort on the beam's stream.
 * Opt-in and purely a performance hint: it makes every chunk of consecutive particles spatially compact, which is
 * what bt_deposit_cic needs to bin a chunk by cell in shared memory and sum same-cell particles in registers before
 * touching rho, and what lets bt_gather_kick find its nodes in L1; both remain correct for any order and stay fast
 * while particles wander a few cells from where the sort left them, so one sort serves many steps.
 * bt_beam_download still returns the original order; bt_beam_upload resets storage to the caller's order.
 * The order of particles within one cell is not deterministic.  Needs n < 2^31; allocates 56 bytes per
 * particle on first use (the partner set of six arrays the sort writes into -- see bt_beam_ptrs -- and two id arrays).
 */
int bt_beam_sort_by_cell(bt_beam *beam, const bt_grid *grid, double zscale);
/*
 * Cadence of the cell binning: with every_n_deposits = n > 0, bt_deposit_cic calls bt_beam_sort_by_cell(beam, grid, zscale)
 * itself before its 1st, (n+1)th, (2n+1)th ... call since the last bt_beam_upload; 0 (default) = never, the caller sorts.
 * Particles wander away from where a sort left them and chunk membership is fixed, so deposit and gather slow down from
 * one sort to the next (measured on configs[4]: deposit 101 -> 116 us over 5 steps, gather 141 -> 188 us; one re-sort of a
 * nearly sorted beam 0.27 ms): n = 5..6 is the measured optimum there.  Results never depend on it.
 */
int bt_beam_set_resort_interval(bt_beam *beam, int32_t every_n_deposits);
/* Device array of n int32: ids[j] = original index of storage slot j; NULL while storage order == original order. */
int bt_beam_ids(bt_beam *beam, int32_t **dev_ids_out);

/* ---- lattice (S1) and fused walk (S2, S3) --------------------------------------------------- */

/*
 * Validate and copy the element list (n_elems >= 1).  Mirrors sim.lattice.extend([...]) (P:l.93).
 * The per-slice map coefficients are computed on the host from (type, params, beta0, beta0*gamma0)
 * when bt_track needs them and packed into 64-byte records; a launch of the walk carries its records as kernel
 * parameters (<= 510 records; constant bank 0), so nothing on the device is shared between beams or streams:
 * beams may be used concurrently from different host threads / streams (one thread per beam at a time).
 * A bt_grid carries unsynchronised bookkeeping of which stream touched it last (bt_deposit_cic, bt_gather_kick -- through
 * its const pointer too -- and bt_grid_solve_poisson update it): a grid and every beam used with it must be driven from ONE
 * host thread at a time.  bt_debug_knob is process-wide and meant to be set while no other thread is inside the library.
 */
int bt_lattice_set(bt_beam *beam, const bt_element *elems, int32_t n_elems);

/*
 * Fused lattice walk (R3): for turn in 1..nturns, for each element in list order, for each slice:
 * apply the element's map of length ds/nslice to every particle.  ONE kernel: each particle is
 * loaded once, every element map and slice is applied in registers, and it is stored once per launch
 * (96 bytes of HBM traffic per particle per launch).  Lattices whose RF cavities change the reference
 * energy are processed in chunks of whole turns (one launch per <= 510 records, per-turn coefficient tables),
 * lattices with more than 510 records per turn in several launches per turn.
 * Updates the reference gamma, s and turn.  Bit-reproducible run to run.  nturns >= 0.
 * Mirrors sim.evolve() (P:l.95) without space charge.
 */
int bt_track(bt_beam *beam, int32_t nturns);

/*
 * The same walk with HOST buffers on both sides: upload, bt_track(nturns), download -- what a caller whose bunch
 * lives in host memory does per call (sim.evolve() on a host-resident container, P:l.95).  The bunch is cut into
 * `nchunks` contiguous chunks that ride three internal streams, so the host->device copy of chunk k+1, the walk of
 * chunk k and the device->host copy of chunk k-1 overlap; particles never interact in the walk (S:8e), so the result
 * is bit-identical to bt_beam_upload + bt_track + bt_beam_download for any nchunks.  host_in / host_out: 6 host arrays
 * of n doubles each (order x, px, y, py, t, pt; pinned memory for the copies to be asynchronous; host_out may alias
 * host_in).  Synchronous: returns when host_out is complete.  The beam's device arrays hold the result too; storage
 * order is reset as by bt_beam_upload.  nchunks in [1, 256].  Any lattice is pipelined, including those whose RF changes
 * the reference energy (P:l.82-83 reference particle; S3): every chunk runs the same sequence of launches, each launch
 * carrying its own coefficient table.
 */
int bt_track_host(bt_beam *beam, const double *const host_in[6], double *const host_out[6], int32_t nturns, int32_t nchunks);

/* ---- grid, CIC deposit (S4, S5) and gather + kick (S6, S7) ---------------------------------- */

/*
 * Node-centred grid (R10): nx,ny,nz >= 2 nodes per axis, node (i,j,k) at lo + (i,j,k)*d, d > 0,
 * linear index (k*ny + j)*nx + i (x fastest).  Third axis coordinate zeta = zscale * t.
 * Allocates rho (zeroed).  Mirrors init_grids() (P:l.64).
 */
int bt_grid_create(bt_grid **out, int32_t nx, int32_t ny, int32_t nz, const double lo[3], const double d[3]);
void bt_grid_destroy(bt_grid *grid);
/* Field at the nodes, 3 arrays of nx*ny*nz doubles, x fastest; on_device != 0: device pointers (copied
 * device-to-device), else host pointers.  The library keeps its own (internally re-laid-out) copy. */
int bt_grid_set_field(bt_grid *grid, const double *Ex, const double *Ey, const double *Ez, int on_device);
/*
 * Particle shape used by bt_deposit_cic and bt_gather_kick on this grid; mirrors sim.set_particle_shape(order)
 * (P:l.60).  order = 1 (default): CIC / trilinear, 8 nodes (R11).  order = 2: quadratic B-spline,
 * 27 nodes (reading R16): v = u + 0.5, j = floor(v) the nearest node, delta = u - j, weights on nodes j-1, j, j+1
 *   (1/2)(1/2 - delta)^2,  3/4 - delta^2,  (1/2)(1/2 + delta)^2     (each operation rounded once, in this order),
 * node weight (wx*wy)*wz; inside iff 1 <= j <= n-2 on all axes (tested as v >= 1 && v < n-1), else skipped / zero
 * field.  Needs >= 3 nodes per axis.  Other orders: BT_ERR_UNSUPPORTED.  bt_beam_sort_by_cell keeps ordering by the
 * order-1 cell; both kernels are correct for any order of the particles.
 */
int bt_grid_set_particle_shape(bt_grid *grid, int32_t order);
int bt_grid_rho(bt_grid *grid, double **dev_rho_out);    /* zero-copy device view of rho */

/*
 * Space-charge field from the deposited charge (P:l.49 "the Poisson equation is solved in the bunch
 * rest frame"), reading R19: open boundaries, rho = charge per node [C],
 *   phi_a = (1/(4 pi eps0)) sum_b q_b G(r_a - r_b),  G(r) = 1/|r| for a != b,  G(0) = (1/V) int_cell 1/|r| dV,
 * with the third-axis spacing stretched to gz*dz (gz = gamma0 turns zeta = beta0 c dt into the rest-frame length), then
 *   E = -grad phi  (rest frame; centred differences, one-sided first-order at the faces; third axis with gz*dz).
 * The sum is evaluated as a zero-padded FFT convolution (Hockney) on `cuda_stream` (cudaStream_t, may be 0): rho -> phi [V]
 * -> the grid's field (replacing any field given to bt_grid_set_field), ready for bt_gather_kick, whose coef[] carries the
 * rest-frame -> kick factors.  Allocates ~35 x nx*ny*nz x 8 bytes on first use; the transformed Green table is cached per gz.
 * Asynchronous.  Grids up to 2^28 nodes.
 */
int bt_grid_solve_poisson(bt_grid *grid, double gz, void *cuda_stream);
int bt_grid_download_phi(bt_grid *grid, double *host_phi);   /* nx*ny*nz doubles, x fastest; synchronises */
/* The grid's current field (from bt_grid_set_field or bt_grid_solve_poisson), 3 host arrays of nx*ny*nz doubles; synchronises. */
int bt_grid_download_field(bt_grid *grid, double *host_Ex, double *host_Ey, double *host_Ez);
int bt_grid_download_rho(bt_grid *grid, double *host_rho); /* synchronises the last beam stream used */

/*
 * CIC (order-1) charge deposition (R11, R13; P:l.43 "charge deposition", P:l.60 particle shape):
 *   rho[node] += q_weight * (wx*wy)*wz for the 8 nodes around each particle, with per axis
 *   u = (q - lo)*(1/d), i = floor(u), w1 = u - i, w0 = 1 - w1, third axis q = zscale*t.
 * rho is charge per node.  Particles with i outside [0, n-2] on any axis (or NaN) are skipped.
 * zero_first != 0 clears rho first (on the beam's stream).  The summation order is not deterministic;
 * results are reproducible to fp64 rounding of the per-node sums only.
 */
int bt_deposit_cic(bt_beam *beam, bt_grid *grid, double q_weight, double zscale, int zero_first);

/*
 * Split-operator space-charge push (R12; P:l.49 "map-based split-operator approach"):
 *   [drift(half_drift_before)]  ->  E = trilinear(field) at (x, y, zscale*t), outside => 0
 *   px += coef[0]*Ex; py += coef[1]*Ey; pt += coef[2]*Ez   ->  [drift(half_drift_after)]
 * in one pass over the particles (96 bytes per particle).  The drifts are R4 with the beam's current
 * reference energy and advance s; 0, 0 => kick only.  Requires bt_grid_set_field and bt_beam_set_ref.
 */
int bt_gather_kick(bt_beam *beam, const bt_grid *grid, const double coef[3], double zscale,
                   double half_drift_before, double half_drift_after);

/* ---- beam statistics ---------------------------------------------------- */

/*
 * Means and second moments of the six coordinates (P:l.43 "beam statistics"; P:l.112 "beam second moments ...
 * emittances"; the quantity every benchmark of the paper is judged on, and what slice-step diagnostics (P:l.61)
 * print), order x, px, y, py, t, pt:
 *   host_mean[i]    = (1/n) sum_p q_i[p]
 *   host_cov[6*i+j] = (1/n) sum_p (q_i[p] - mean_i)(q_j[p] - mean_j)       (population moments, full symmetric 6x6)
 * Both outputs are HOST arrays owned by the caller.  One pass over the particles (48 bytes each) on the beam's
 * stream, sums taken about a provisional centre so that an offset bunch loses no digits; the call synchronises the
 * stream.  Deterministic (fixed reduction order), independent of the storage order up to fp64 rounding.  The
 * unnormalised rms emittance of a plane is sqrt(cov_qq*cov_pp - cov_qp^2).  NaN/Inf coordinates propagate.
 */
int bt_beam_moments(bt_beam *beam, double host_mean[6], double host_cov[36]);
/*
 * The same statistics (P:l.43, l.61), left on the DEVICE: dev_out receives 42 doubles (mean[6], then cov[36] row-major) in
 * device memory owned by the caller, written by the beam's stream; the call only enqueues the kernel and returns -- no
 * synchronisation, no copy -- so a step loop can take the statistics every step and read them back whenever it likes.
 * Bit-identical to bt_beam_moments.
 */
int bt_beam_moments_device(bt_beam *beam, double *dev_out);

/*
 * The same statistics (P:l.43 "beam statistics", P:l.112 second moments) for a caller that is not allowed to allocate
 * device memory: no bt_beam is needed and the call makes no cudaMalloc / cudaFree / cudaHostAlloc or any other
 * allocating call, now or later.
 *
 * Who that is: a host application whose own memory arena took (almost) all of HBM at start-up, as the mesh frameworks
 * underneath the paper's code do, so that an allocation made behind its back fails or eats into what the arena counts
 * on; a step loop with several busy streams, which a cudaMalloc would stall because it synchronises the whole device;
 * a process run under an allocation checker that treats any device allocation by a library as an error.  Every other
 * statistics call of this library allocates on first use (bt_beam_create, the partial-sum buffer of bt_beam_moments).
 *
 *   dev_q       six DEVICE arrays of n doubles, order x, px, y, py, t, pt, owned by the caller, read only; 8-byte
 *               aligned (all six 16-byte aligned: the vectorised kernel).  They must belong to the CURRENT device.
 *   n           1 <= n <= BT_MOMENTS_STATIC_MAX_PARTICLES.  Anything larger returns BT_ERR_INVALID and launches
 *               nothing: the partial sums go into a fixed array inside the library (one 216-byte row per 32 768
 *               particles, 2 048 rows), and that array cannot grow.
 *   dev_out     DEVICE array of 42 doubles owned by the caller: mean[6], then cov[36] row-major, as bt_beam_moments_device.
 *   cuda_stream cudaStream_t cast to void* (0 = legacy default stream).  The call enqueues one 4-byte memset and one
 *               kernel there and returns; nothing is synchronised.
 *
 * Same definition and same kernel as bt_beam_moments; the grid depends on n only (not on the GPU model), so the fp64
 * sums are associated differently and the results agree with bt_beam_moments to rounding (|d cov_ij| <= 1e-12
 * sqrt(cov_ii cov_jj)), not bit for bit.  Deterministic run to run.
 *
 * What the fixed array costs -- read before use:
 *  - 432.25 KiB of device memory on EVERY GPU that loads libbt.so, from load until the process exits, used or not.
 *  - One array per GPU, shared by all calls from all threads.  Two calls whose kernels can run at the same time on one GPU
 *    (different streams without an event between them, different host threads) corrupt each other's sums.  Issue them
 *    on one stream, or order the streams yourself.
 *  - The array still holds the previous call's rows.  Nothing depends on that (rows are written before they are read;
 *    the completion counter is cleared on cuda_stream before every launch), so a failed earlier call does no harm.
 *  - The first call on each GPU looks up the array's device address (cudaGetSymbolAddress, with that GPU current) and
 *    caches it.  Make that first call during set-up, outside any stream capture.
 */
#define BT_MOMENTS_STATIC_MAX_PARTICLES 67108864LL /* 2048 rows x 32768 particles */
int bt_moments_static(const double *const dev_q[6], int64_t n, double *dev_out, void *cuda_stream);

/*
 * Slice-step diagnostics (mirrors sim.set_slice_step_diagnostics(True), P:l.61; the statistics are P:l.43 "beam statistics"):
 * the same walk as bt_track(nturns) -- bit-identical final coordinates, reference energy, s and turn -- with the beam
 * statistics of bt_beam_moments taken INSIDE the walk, after every element (BT_DIAG_ELEMENT) or after every slice of every
 * element (BT_DIAG_SLICE).  host_moments receives nturns * B records of 42 doubles (mean[6], then cov[36] row-major) in walk
 * order, B = number of elements (resp. the sum of their nslice): record (turn * B + b) is the beam right after boundary b
 * of that turn.  No extra pass over the particles (96 bytes per particle per launch, as bt_track): each warp writes one
 * 216-byte row of partial sums per boundary and a second kernel combines them in a fixed order (bit-reproducible); O(1)
 * launches per record table (<= 510 records) / per GiB of rows.  The sums are taken about the centre of the bunch as it
 * is when the call starts, so a record loses about 2 log10(|mean - centre| / sigma) digits if the centroid runs away from
 * there during the walk (none on any configuration whose centroid stays within a few sigma).  Synchronous.
 */
enum { BT_DIAG_ELEMENT = 0, BT_DIAG_SLICE = 1 };
int bt_track_diagnostics(bt_beam *beam, int32_t nturns, int32_t granularity, double *host_moments);
/* How many 42-double records bt_track_diagnostics(beam, nturns, granularity, ...) writes for the beam's current lattice
 * (nturns x number of elements, resp. x the sum of their nslice): size host_moments from this. */
int bt_track_diagnostics_records(const bt_beam *beam, int32_t nturns, int32_t granularity, int64_t *n_records);
/* bt_track_diagnostics with the capacity of host_moments stated (in records of 42 doubles): BT_ERR_INVALID, and nothing
 * launched, when the call would write more.  Prefer this one from any language where the buffer's size is a separate fact. */
int bt_track_diagnostics_n(bt_beam *beam, int32_t nturns, int32_t granularity, double *host_moments, int64_t capacity_records);
/* Frees what the beam keeps between calls for the diagnostics walk (the row buffer, up to 1 GiB, and the record buffer) and
 * bt_beam_download's un-permute scratch; they are re-allocated on demand.  Synchronises the beam's stream. */
int bt_beam_release_scratch(bt_beam *beam);
/* Failure part-way: if a launch fails inside bt_track, bt_track_host or bt_track_diagnostics (BT_ERR_CUDA), the particles
 * have been advanced through part of the lattice while the reference energy, s and turn are left as they were.  The
 * beam's state is then undefined: upload the bunch and set the reference again. */

/* ---- utilities ------------------------------------------------------------------------------ */
int bt_sync(bt_beam *beam); /* cudaStreamSynchronize on the beam's stream */
const char *bt_last_error(void);
int bt_version(void);

/* ==== diagnostics and measurement helpers: NOT part of the method, no passage of the paper behind them ================
 * They exist for bench.py (launch counts, roofline denominators measured on the box) and for the tests (forcing every
 * kernel variant).  A caller of the method never needs them. */
/* Number of CUDA kernels this library has launched in this process (all beams/grids). */
int64_t bt_launch_count(void);
/* Name and launch geometry of the last fused-walk launch (any out may be NULL). */
int bt_track_last_launch(const bt_beam *beam, int32_t *grid_dim, int32_t *block_dim,
                         int32_t *particles_per_thread, int32_t *smem_bytes);
/*
 * Force a kernel variant, process-wide (typed replacement of round 1's BT_* environment variables; nothing in the library
 * reads the environment).  value < 0 restores the measured default.  Results never depend on a knob; speed does.
 *   "track_ppt"     particles per thread of the fused walk: 1, 2, 4
 *   "track_block"   threads per block of the fused walk: 32, 64, 96, 128
 *   "track_fuse"    0: one record per lattice element (no peephole fusion of records)
 *   "deposit_mode"  0: one particle per thread, plain reductions; 1: default; 2: 4 particles per thread
 *   "gather_mode"   0: registers; 1: default; 2 / 3: 512- / 128-particle chunks; 4: field tile in shared memory
 *   "plan_window"   records of per-turn coefficient tables the host builds ahead of the launches (default 65 280 = 4 MiB;
 *                   whole turns, at least one): bt_track / bt_track_host of many turns through a lattice whose RF changes
 *                   the reference energy build and enqueue one such window at a time
 */
int bt_debug_knob(const char *name, int32_t value);

/*
 * Measurement utilities (roofline denominators measured on the box):
 *  bt_calib_fp64: runs a register-only kernel of independent DFMA chains on all SMs for about
 *     `min_ms` milliseconds and returns the achieved FP64 pipe instruction slots per second
 *     (thread-level DFMA count / elapsed; one slot = one DFMA/DMUL/DADD of one thread).
 *  bt_calib_rw6: streams 6 arrays of n doubles in and 6 out (the access pattern of bt_track)
 *     and returns GB/s (96*n bytes / elapsed).  Allocates and frees its own buffers.
 */
int bt_calib_fp64(void *cuda_stream, double min_ms, double *slots_per_s);
int bt_calib_rw6(void *cuda_stream, int64_t n, int32_t reps, double *gbytes_per_s);

#ifdef __cplusplus
}
#endif
#endif /* BT_H_ */
