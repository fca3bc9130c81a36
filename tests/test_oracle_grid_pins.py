"""Pins for the oracle's CIC deposit (R10, R11, R13, R15) and trilinear gather + kick (R12).

Independent of the oracle's own code: hand-computed weights, a pure-Python brute force of the
definition on tiny grids, partition of unity / exact total charge, multilinear exactness of the
interpolation, the deposit<->gather adjoint identity, and the thin-quadrupole equivalence.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

import oracle as O
import workloads as W

GAMMA_P1GEV = O.ref_from_kinetic(1000.0, W.MASS_PROTON_MEV)[0]


def brute_deposit(x, y, t, shape, lo, d, qw, zscale=1.0):
    """The definition, particle by particle, in exact rational arithmetic on the fp64 inputs
    (u is formed with fp64 ops as R11 prescribes; the weights' products and sums are exact)."""
    nx, ny, nz = shape
    rho = [[[Fraction(0) for _ in range(nx)] for _ in range(ny)] for _ in range(nz)]
    inside = 0
    inv = [1.0 / d[a] for a in range(3)]
    for p in range(len(x)):
        q = (x[p], y[p], zscale * t[p])
        idx, w = [], []
        ok = True
        for a, n in enumerate((nx, ny, nz)):
            u = (q[a] - lo[a]) * inv[a]
            if not (u >= 0.0 and u < n - 1):
                ok = False
                break
            i = math.floor(u)
            w1 = u - i
            w0 = 1.0 - w1
            idx.append(i)
            w.append((w0, w1))
        if not ok:
            continue
        inside += 1
        for dz in range(2):
            for dy in range(2):
                for dx in range(2):
                    ww = (w[0][dx] * w[1][dy]) * w[2][dz]           # fp64, R11 association
                    rho[idx[2] + dz][idx[1] + dy][idx[0] + dx] += Fraction(qw * ww)
    return np.array([[[float(v) for v in row] for row in plane] for plane in rho]), inside


def test_hand_weights_node_and_cell_centre():
    shape, lo, d = (4, 4, 4), (0.0, 0.0, 0.0), (1.0, 1.0, 1.0)
    # particle exactly on node (1,2,1): weight 1 there
    rho, n_in = O.deposit_cic(np.array([1.0]), np.array([2.0]), np.array([1.0]), shape, lo, d, 3.0)
    assert n_in == 1 and rho[1, 2, 1] == 3.0 and rho.sum() == 3.0 and np.count_nonzero(rho) == 1
    # particle at a cell centre: 8 x 0.125
    rho, n_in = O.deposit_cic(np.array([0.5]), np.array([1.5]), np.array([2.5]), shape, lo, d, 1.0)
    assert n_in == 1 and np.count_nonzero(rho) == 8
    assert np.all(rho[2:4, 1:3, 0:2] == 0.125)
    # asymmetric: x fastest, t (third axis) slowest: weights (.75,.25) x (1,0) x (.5,.5)
    rho, _ = O.deposit_cic(np.array([0.25]), np.array([1.0]), np.array([0.5]), shape, lo, d, 1.0)
    assert rho[0, 1, 0] == 0.375 and rho[0, 1, 1] == 0.125 and rho[1, 1, 0] == 0.375 and rho[1, 1, 1] == 0.125
    assert rho.sum() == 1.0


@pytest.mark.parametrize("zscale", [1.0, -1.8, 0.37])
def test_brute_force_tiny_grid(zscale):
    rng = np.random.default_rng(123)
    shape, lo, d = (4, 5, 3), (-1.0, -2.0, -0.5), (0.7, 1.1, 0.6)
    n = 10
    x = rng.uniform(-1.2, 1.2, n)
    y = rng.uniform(-2.2, 2.5, n)
    t = rng.uniform(-0.6, 0.8, n) / zscale
    ref, n_ref = brute_deposit(x, y, t, shape, lo, d, 1e-10, zscale)
    rho, n_in = O.deposit_cic(x, y, t, shape, lo, d, 1e-10, zscale)
    assert n_in == n_ref and 0 < n_in < n
    assert rho.shape == (3, 5, 4)
    assert np.array_equal(rho, ref)          # long-double accumulation of <= 10 terms rounds like the exact sum


def test_boundary_rules_R13():
    shape, lo, d = (5, 5, 5), (-2.0, -2.0, -2.0), (1.0, 1.0, 1.0)
    mid = 0.3
    cases = [
        (-2.0, mid, mid, True),      # exactly on lo: inside, i = 0, w1 = 0
        (2.0, mid, mid, False),      # exactly on the last node: i = n-1 -> outside
        (math.nextafter(2.0, 0.0), mid, mid, False),   # (q - lo) rounds to 4.0: the ROUNDED u decides (R11)
        (2.0 - 1e-15, mid, mid, True),
        (math.nextafter(-2.0, -3.0), mid, mid, False),
        (mid, 2.5, mid, False),
        (mid, mid, -2.5, False),
        (float("nan"), mid, mid, False),
        (mid, float("inf"), mid, False),
    ]
    for x, y, t, inside in cases:
        rho, n_in = O.deposit_cic(np.array([x]), np.array([y]), np.array([t]), shape, lo, d, 1.0)
        assert n_in == int(inside), (x, y, t)
        assert (abs(rho.sum() - 1.0) < 1e-15) if inside else (not rho.any())
    rho, _ = O.deposit_cic(np.array([-2.0]), np.array([-2.0]), np.array([-2.0]), shape, lo, d, 1.0)
    assert rho[0, 0, 0] == 1.0


def test_total_charge_exact_and_partition_of_unity():
    sc = W.spacecharge_config("A", n=200_000, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    c[0][:5] = 1.0                         # force a few outside (beyond +6 sigma = 6e-3)
    rho, n_in = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight)
    assert n_in == sc.n - 5
    total = math.fsum(rho.ravel())
    assert abs(total - sc.q_weight * n_in) <= 1e-13 * sc.q_weight * n_in
    assert rho.min() >= 0.0


def test_accumulate_mode_and_linearity():
    rng = np.random.default_rng(5)
    shape, lo, d = (6, 6, 6), (0.0, 0.0, 0.0), (1.0, 1.0, 1.0)
    a = [rng.uniform(0, 5, 50) for _ in range(3)]
    b = [rng.uniform(0, 5, 70) for _ in range(3)]
    ra, _ = O.deposit_cic(*a, shape, lo, d, 2.0)
    rab, _ = O.deposit_cic(*b, shape, lo, d, 2.0, rho=ra.copy())
    both, _ = O.deposit_cic(*[np.concatenate([u, v]) for u, v in zip(a, b)], shape, lo, d, 2.0)
    assert np.max(np.abs(rab - both)) < 1e-14
    r2, _ = O.deposit_cic(*a, shape, lo, d, 4.0)
    assert np.array_equal(r2, 2.0 * ra)


def test_adversarial_bunch_stays_in_core_nodes():
    sc = W.spacecharge_config("B", n=100_000, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    core = (np.arange(sc.n) % 10) != 0
    assert np.all(c[1][core] == 0) and np.all(c[3][core] == 0) and np.all(c[5][core] == 0)
    rho, _ = O.deposit_cic(c[0][core], c[2][core], c[4][core], sc.shape, sc.lo, sc.d, 1.0)
    nz = np.argwhere(rho > 0)
    assert nz.min() >= 15 and nz.max() <= 17 and len(nz) == 27       # 2 cells wide -> 27 nodes (c-1..c+1)
    assert abs(rho.sum() - core.sum()) < 1e-9 * core.sum()


# ------------------------------------------------------------------------------------------------
# gather
# ------------------------------------------------------------------------------------------------
def _nodes(shape, lo, d):
    ax = [lo[a] + d[a] * np.arange(n) for a, n in enumerate(shape)]
    Z, Y, X = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
    return X, Y, Z


def test_trilinear_reproduces_multilinear_functions():
    rng = np.random.default_rng(9)
    shape, lo, d = (7, 6, 5), (-1.0, 0.5, -2.0), (0.4, 0.3, 0.9)
    X, Y, Z = _nodes(shape, lo, d)
    co = rng.uniform(-1, 1, (3, 8))

    def f(c, x, y, z):
        return c[0] + c[1] * x + c[2] * y + c[3] * z + c[4] * x * y + c[5] * y * z + c[6] * x * z + c[7] * x * y * z

    E = [f(co[k], X, Y, Z) for k in range(3)]
    n = 500
    x = rng.uniform(lo[0], lo[0] + d[0] * (shape[0] - 1) * 0.999, n)
    y = rng.uniform(lo[1], lo[1] + d[1] * (shape[1] - 1) * 0.999, n)
    zs = -1.7
    zeta = rng.uniform(lo[2], lo[2] + d[2] * (shape[2] - 1) * 0.999, n)
    t = zeta / zs
    got = O.gather_field(x, y, t, shape, lo, d, E, zscale=zs)
    for k in range(3):
        assert np.max(np.abs(got[k] - f(co[k], x, y, zs * t))) < 2e-14


def test_gather_axis_order_and_component_mapping():
    """Ex = x-coordinate, Ey = 10*y, Ez = 100*zeta at the nodes: pins x-fastest layout and which component
    kicks which momentum (px<-Ex, py<-Ey, pt<-Ez) with the caller's three coefficients."""
    shape, lo, d = (4, 5, 6), (0.0, 0.0, 0.0), (1.0, 1.0, 1.0)
    X, Y, Z = _nodes(shape, lo, d)
    c = [np.array([1.25]), np.array([0.5]), np.array([2.5]), np.array([-0.5]), np.array([3.75]), np.array([0.25])]
    n_in = O.gather_kick(c, shape, lo, d, (X, 10 * Y, 100 * Z), (2.0, 3.0, -1.0))
    assert n_in == 1
    assert c[1][0] == 0.5 + 2.0 * 1.25 and c[3][0] == -0.5 + 3.0 * 25.0 and c[5][0] == 0.25 - 375.0
    assert c[0][0] == 1.25 and c[2][0] == 2.5 and c[4][0] == 3.75


def test_uniform_field_and_outside_zero():
    shape, lo, d = (4, 4, 4), (0.0, 0.0, 0.0), (1.0, 1.0, 1.0)
    E = [np.full((4, 4, 4), v) for v in (2.0, -3.0, 5.0)]
    x = np.array([0.1, 2.9, 3.0, -0.1, 1.5])
    c = [x, np.zeros(5), np.full(5, 1.5), np.zeros(5), np.full(5, 1.5), np.zeros(5)]
    n_in = O.gather_kick(c, shape, lo, d, E, (1.0, 1.0, 1.0))
    assert n_in == 3
    inside = np.array([True, True, False, False, True])
    assert np.allclose(c[1][inside], 2.0, rtol=0, atol=1e-15) and np.all(c[1][~inside] == 0.0)
    assert np.allclose(c[3][inside], -3.0, rtol=0, atol=1e-15) and np.all(c[5][~inside] == 0.0)


def test_quadrupole_field_equals_thin_multipole():
    """E = G (x, -y, 0) sampled on the grid is multilinear -> the kick equals R8 with m=2, Kn = -coef*G."""
    sc = W.spacecharge_config("A", n=5000, shape=(16, 16, 16))
    c = W.make_spacecharge_bunch(sc)
    ref = [a.copy() for a in c]
    X, Y, Z = _nodes(sc.shape, sc.lo, sc.d)
    G, coef = 1e5, 2e-9
    O.gather_kick(c, sc.shape, sc.lo, sc.d, (G * X, -G * Y, 0 * Z), (coef, coef, coef))
    O.track(ref, [("multipole", 0.0, 1, 2, -coef * G, 0.0)], 1, GAMMA_P1GEV)
    for a, b in zip(c, ref):
        assert np.max(np.abs(a - b)) < 1e-18


def test_deposit_gather_adjoint():
    """sum_nodes rho[node] phi[node] == q_w sum_p phi_interp(x_p): deposit is the transpose of gather."""
    sc = W.spacecharge_config("A", n=20_000, shape=(16, 16, 16))
    c = W.make_spacecharge_bunch(sc)
    rng = np.random.default_rng(11)
    phi = rng.standard_normal((16, 16, 16))
    rho, n_in = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, 1.0)
    got = O.gather_field(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, (phi, phi, phi))[0]
    lhs, rhs = math.fsum((rho * phi).ravel()), math.fsum(got)
    assert abs(lhs - rhs) < 1e-10 * max(1.0, abs(rhs))


def test_prescribed_field_gauss_law_and_series():
    """workloads.gaussian_bunch_field: E r^2 4 pi eps0 -> Q outside the bunch; series joins the closed form."""
    sc = W.spacecharge_config("A", n=1, shape=(128, 128, 128))
    Ex, Ey, Ez = W.gaussian_bunch_field(sc)
    X, Y, Z = _nodes(sc.shape, sc.lo, sc.d)
    r = np.sqrt(X**2 + Y**2 + Z**2)
    Er = (Ex * X + Ey * Y + Ez * Z) / r
    far = r > 5.5 * sc.sigma
    q_enc = Er[far] * r[far] ** 2 * 4 * np.pi * W.EPS0
    assert np.max(np.abs(q_enc / sc.bunch_charge_C - 1)) < 1e-5
    emag = np.sqrt(Ex**2 + Ey**2 + Ez**2)
    assert abs(emag.max() - 1.9233e6) < 2e3                    # peak |E| near r = 1.37 sigma
    assert np.max(np.abs(Ex + Ex[:, :, ::-1])) < 1e-9 * emag.max()     # odd symmetry on the symmetric node set
    # series vs closed form at the switch radius
    from scipy.special import erf
    s, kq = sc.sigma, sc.bunch_charge_C / (4 * np.pi * W.EPS0)
    rr = 0.01 * s
    closed = kq * (erf(rr / (np.sqrt(2) * s)) - np.sqrt(2 / np.pi) * (rr / s) * np.exp(-rr * rr / (2 * s * s))) / rr**2
    series = kq * rr * np.sqrt(2 / np.pi) / (3 * s**3) * (1 - 3 * rr * rr / (10 * s * s))
    assert abs(closed / series - 1) < 1e-8


def test_config4_step_runs_and_kick_direction():
    """One split-operator step (R12): a late particle (zeta>0) behind a positive bunch gains pt; the
    transverse kick is outward."""
    sc = W.spacecharge_config("A", n=20_000, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    E = W.gaussian_bunch_field(sc)
    before = [a.copy() for a in c]
    O.gather_kick(c, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale)
    sel = np.abs(before[0]) > 1e-4
    assert np.all(np.sign(c[1] - before[1])[sel] == np.sign(before[0])[sel])
    sel = np.abs(before[4]) > 1e-4
    assert np.all(np.sign(c[5] - before[5])[sel] == np.sign(before[4])[sel])
    assert np.max(np.abs(c[1] - before[1])) < 1e-5
