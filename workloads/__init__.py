"""Seeded synthetic inputs for the five BASELINE.json configs -- shared by the oracle side and the
CUDA side, and holding NONE of the method's arithmetic (no maps, no weights, no reference-particle
kinematics): only input data -- particle coordinates, element lists, grid geometry, a prescribed
field, physical constants -- and the recipe that draws them.

Stand-in statement: the paper's own inputs (IOTA v8.4 lattice, Berlin-Zeuthen chicane parameters,
Zenodo artefacts) are not available; these configs take their *shape*
(element kinds, slicing, bunch sizes, Gaussian / matched phase space) from PAPER.md l.56-95
(Listing 1), l.108-148, as fixed by BASELINE.json `configs` and SURVEY.md 8(d).

Generator (SURVEY 8d "Inputs, concretely"): numpy.random.Generator(PCG64(seed)),
standard_normal(N) drawn in the order x, px, y, py, t, pt (unit variates first, then transformed);
seed = config index (0,1,2,3,4) and 5 for the adversarial variant 4B.

Lattice format: list of tuples (kind, ds, nslice, *params) with kind in
{"drift","quad","sbend","dipedge","multipole","shortrf"}; params as in include/bt.h:
quad: k | sbend: rc | dipedge: psi, rc, g, K | multipole: m, Kn, Ks | shortrf: Vhat, freq_Hz, phase_deg.
"""
from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

MASS_ELECTRON_MEV = 0.510998950
MASS_PROTON_MEV = 938.27208816         # CODATA-2018 (not in the paper)
C_LIGHT = 299792458.0
EPS0 = 8.8541878128e-12

COORD_NAMES = ("x", "px", "y", "py", "t", "pt")


# --------------------------------------------------------------------------------------------
# lattices (input data only)
# --------------------------------------------------------------------------------------------
def fodo_cell(nslice_quad: int) -> List[tuple]:
    """The cell of PAPER.md Listing 1 (l.86-91): D .25 / Q L=1 k=+1 / D .5 / Q L=1 k=-1 / D .25."""
    return [
        ("drift", 0.25, 1),
        ("quad", 1.0, nslice_quad, 1.0),
        ("drift", 0.5, 1),
        ("quad", 1.0, nslice_quad, -1.0),
        ("drift", 0.25, 1),
    ]


def chicane() -> List[tuple]:
    """BASELINE configs[2] with reading R7: rectangular magnets, one non-trivial face per bend."""
    L, th, rc, g, K = 0.5, 0.05, 10.0, 0.02, 0.5
    return [
        ("sbend", L, 1, +rc), ("dipedge", 0.0, 1, +th, +rc, g, K),
        ("drift", 5.0, 1),
        ("dipedge", 0.0, 1, -th, -rc, g, K), ("sbend", L, 1, -rc),
        ("drift", 1.0, 1),
        ("sbend", L, 1, -rc), ("dipedge", 0.0, 1, -th, -rc, g, K),
        ("drift", 5.0, 1),
        ("dipedge", 0.0, 1, +th, +rc, g, K), ("sbend", L, 1, +rc),
    ]


RING_CELLS = 25
RING_LENGTH_M = 75.0
RING_RF_VHAT = 1.0 / MASS_PROTON_MEV            # 1 MV on a proton: qV/(mc^2)
RING_RF_FREQ_HZ = 3.4976811924685272e6          # h=1: beta0*c/C at injection, held fixed
RING_RF_PHASE_DEG = -30.0


def ring_cell(sext: float = 5.0, octu: float = 50.0) -> List[tuple]:
    cell = [("quad", 1.0, 1, +1.0)]
    if sext != 0.0:
        cell.append(("multipole", 0.0, 1, 3, +sext, 0.0))
    if octu != 0.0:
        cell.append(("multipole", 0.0, 1, 4, octu, 0.0))
    cell.append(("drift", 0.5, 1))
    cell.append(("quad", 1.0, 1, -1.0))
    if sext != 0.0:
        cell.append(("multipole", 0.0, 1, 3, -sext, 0.0))
    if octu != 0.0:
        cell.append(("multipole", 0.0, 1, 4, octu, 0.0))
    cell.append(("drift", 0.5, 1))
    return cell


def nonlinear_ring(rf: bool = True, sext: float = 5.0, octu: float = 50.0) -> List[tuple]:
    """BASELINE configs[3]: 25 x 8-element cells (= 200 elements) + one short RF (element 201)."""
    lat = ring_cell(sext, octu) * RING_CELLS
    if rf:
        lat.append(("shortrf", 0.0, 1, RING_RF_VHAT, RING_RF_FREQ_HZ, RING_RF_PHASE_DEG))
    return lat


# --------------------------------------------------------------------------------------------
# config descriptors
# --------------------------------------------------------------------------------------------
@dataclass
class TrackConfig:
    name: str
    index: int
    n: int
    seed: int
    kin_energy_MeV: float
    mass_MeV: float
    charge_qe: float
    lattice: List[tuple]
    nturns: int
    # distribution recipe
    twiss_x: Optional[Tuple[float, float, float]] = None   # (beta, alpha, emittance)
    twiss_y: Optional[Tuple[float, float, float]] = None
    sigma_xy: float = 1e-3
    sigma_pxy: float = 1e-3
    sigma_t: float = 1e-3
    sigma_pt: float = 1e-3
    chirp: float = 0.0             # pt = chirp * t + sigma_pt * u

    @property
    def n_elements(self) -> int:
        return len(self.lattice)

    @property
    def slice_maps_per_turn(self) -> int:
        return sum(el[2] for el in self.lattice)


# Periodic Twiss at the cell start, as printed in SURVEY 8(d) (and re-derived from the oracle's
# cell matrix in tests/test_oracle_pins.py::test_workload_twiss_values).
FODO_BETA = 2.821619407971768
FODO_ALPHA_X = -1.5905003549009842
RING_TWISS_X = (3.695053663175798, -1.90323666591514)
RING_TWISS_Y = (2.1045533082748147, 1.2777640438868274)


def config(index: int, n: Optional[int] = None) -> TrackConfig:
    """Tracking configs 0-3 of BASELINE.json; `n` overrides the particle count (reduced parity cases)."""
    if index == 0:
        c = TrackConfig("tiny_fodo", 0, 10_000, 0, 2000.0, MASS_PROTON_MEV, +1.0, fodo_cell(10), 10)
    elif index == 1:
        c = TrackConfig("fodo_channel", 1, 1_000_000, 1, 2000.0, MASS_ELECTRON_MEV, -1.0,
                        fodo_cell(25) * 100, 1,
                        twiss_x=(FODO_BETA, FODO_ALPHA_X, 1e-6), twiss_y=(FODO_BETA, -FODO_ALPHA_X, 1e-6))
    elif index == 2:
        c = TrackConfig("chicane", 2, 16_000_000, 2, 5000.0, MASS_ELECTRON_MEV, -1.0, chicane(), 1,
                        sigma_pt=1e-4, chirp=-20.0)
    elif index == 3:
        c = TrackConfig("nonlinear_ring", 3, 64_000_000, 3, 1000.0, MASS_PROTON_MEV, +1.0,
                        nonlinear_ring(), 100,
                        twiss_x=RING_TWISS_X + (1e-6,), twiss_y=RING_TWISS_Y + (1e-6,))
    else:
        raise ValueError("tracking configs are 0..3; see spacecharge_config for 4A/4B")
    if n is not None:
        c.n = int(n)
    return c


def rank_seed(seed: int, rank: int) -> int:
    """Weak scaling (bench.py --gpus N): every rank tracks its own bunch of the config's size, drawn from its own stream.
    Lives here, not in the package, so that the oracle arm of bench.py never loads the product library."""
    return int(seed) + 1000 * int(rank)


def _plane(u1, u2, twiss, sigma_q, sigma_p):
    if twiss is None:
        return sigma_q * u1, sigma_p * u2
    beta, alpha, eps = twiss
    q = np.sqrt(eps * beta) * u1
    p = np.sqrt(eps / beta) * (u2 - alpha * u1)
    return q, p


def make_bunch(cfg: TrackConfig, n: Optional[int] = None, stride: int = 1) -> List[np.ndarray]:
    """[x, px, y, py, t, pt] float64.  `stride` > 1 returns particles i with i % stride == 0 of the
    FULL n-particle draw (so a subset is bit-identical to the same particles of the full bunch)."""
    n = cfg.n if n is None else int(n)
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    u = [rng.standard_normal(n)[::stride].copy() for _ in range(6)]
    x, px = _plane(u[0], u[1], cfg.twiss_x, cfg.sigma_xy, cfg.sigma_pxy)
    y, py = _plane(u[2], u[3], cfg.twiss_y, cfg.sigma_xy, cfg.sigma_pxy)
    t = cfg.sigma_t * u[4]
    pt = cfg.chirp * t + cfg.sigma_pt * u[5]
    return [np.ascontiguousarray(a, dtype=np.float64) for a in (x, px, y, py, t, pt)]


# --------------------------------------------------------------------------------------------
# config 4: space-charge step
# --------------------------------------------------------------------------------------------
@dataclass
class SpaceChargeConfig:
    name: str
    variant: str                     # "A" Gaussian, "B" adversarial cold core
    n: int
    seed: int
    kin_energy_MeV: float = 1000.0
    mass_MeV: float = MASS_PROTON_MEV
    charge_qe: float = +1.0
    bunch_charge_C: float = 1.0e-9
    sigma: float = 1e-3
    shape: Tuple[int, int, int] = (128, 128, 128)   # nodes per axis (R10)
    nsteps: int = 10
    ds: float = 0.01
    zscale: float = 1.0
    # caller-supplied kick coefficients [m/V] (SURVEY R12, 1 GeV proton, ds = 0.01 m, zscale = +1):
    # (q/mc^2) ds/(b0 g0)^2 transverse, +(q/mc^2) ds/(b0 g0) longitudinal.  Input data for the kernels;
    # re-derived from the oracle's reference kinematics in tests/test_oracle_pins.py.
    kick_coef: Tuple[float, float, float] = (3.2618031590960778e-12, 3.2618031590960778e-12,
                                             5.896095048256809e-12)
    lo: Tuple[float, float, float] = field(init=False)
    d: Tuple[float, float, float] = field(init=False)

    def __post_init__(self):
        self.lo = tuple(-6.0 * self.sigma for _ in range(3))
        self.d = tuple(12.0 * self.sigma / (s - 1) for s in self.shape)

    @property
    def q_weight(self) -> float:
        return self.bunch_charge_C / self.n


def spacecharge_config(variant: str = "A", n: Optional[int] = None,
                       shape: Optional[Tuple[int, int, int]] = None) -> SpaceChargeConfig:
    variant = variant.upper()
    seed = {"A": 4, "B": 5}[variant]
    kw = {}
    if shape is not None:
        kw["shape"] = tuple(shape)
    return SpaceChargeConfig("spacecharge_" + variant, variant, 8_000_000 if n is None else int(n), seed, **kw)


def make_spacecharge_bunch(cfg: SpaceChargeConfig) -> List[np.ndarray]:
    n = cfg.n
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    u = [rng.standard_normal(n) for _ in range(6)]
    s = cfg.sigma
    x, px, y, py, t, pt = s * u[0], 1e-3 * u[1], s * u[2], 1e-3 * u[3], s * u[4], 1e-3 * u[5]
    if cfg.variant == "B":
        # 90% of the particles (i % 10 != 0) uniform in the 2-cell-wide cube around the centre
        # [node c-1, node c+1)^3 with c = shape//2 (nodes 63..65 for 128), cold.
        v = [rng.random(n) for _ in range(3)]
        core = (np.arange(n) % 10) != 0
        for q, vv, ax in ((x, v[0], 0), (y, v[1], 1), (t, v[2], 2)):
            c = cfg.shape[ax] // 2
            lo_core = cfg.lo[ax] + (c - 1) * cfg.d[ax]
            q[core] = lo_core + 2.0 * cfg.d[ax] * vv[core]
        for p in (px, py, pt):
            p[core] = 0.0
        if cfg.zscale != 1.0:
            t[core] = t[core] / cfg.zscale
    return [np.ascontiguousarray(a, dtype=np.float64) for a in (x, px, y, py, t, pt)]


def gaussian_bunch_field(cfg: SpaceChargeConfig) -> List[np.ndarray]:
    """Prescribed field: field of a spherical Gaussian charge Q, rms sigma, at the origin,
    E(r) = Q/(4 pi eps0) [erf(r/(sqrt2 s)) - sqrt(2/pi) (r/s) exp(-r^2/2s^2)] / r^2  r_hat,
    sampled at the nodes (x fastest); series Q r sqrt(2/pi)/(4 pi eps0 3 s^3) (1 - 3r^2/(10 s^2))
    for r < 0.01 s.  Input data handed to both sides; erf never enters parity."""
    from scipy.special import erf
    nx, ny, nz = cfg.shape
    ax = [cfg.lo[a] + cfg.d[a] * np.arange(n) for a, n in enumerate((nx, ny, nz))]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")      # arrays [nz, ny, nx]
    r = np.sqrt(X * X + Y * Y + Z * Z)
    s = cfg.sigma
    kq = cfg.bunch_charge_C / (4.0 * np.pi * EPS0)
    rs = np.where(r > 0, r, 1.0)
    closed = kq * (erf(rs / (np.sqrt(2.0) * s)) - np.sqrt(2.0 / np.pi) * (rs / s) * np.exp(-rs * rs / (2 * s * s))) / rs**3
    series = kq * np.sqrt(2.0 / np.pi) / (3.0 * s**3) * (1.0 - 3.0 * r * r / (10.0 * s * s))
    e_over_r = np.where(r < 0.01 * s, series, closed)
    return [np.ascontiguousarray(e_over_r * q) for q in (X, Y, Z)]
