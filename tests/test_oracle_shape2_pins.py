"""Pins for the oracle's order-2 particle shape (reading R16; PAPER.md l.60 `sim.set_particle_shape(2)`):
quadratic B-spline deposit and gather.  Independent of the oracle's formula: the B-spline's own definition (the CIC
triangle averaged over a node's cell, integrated in exact rational arithmetic), its moment identities, brute force
on tiny grids, polynomial reproduction of the gather, the deposit<->gather adjoint identity and the boundary rule."""
from fractions import Fraction

import numpy as np
import pytest

import oracle as O


def triangle_integral(a, b, u):
    """Exact integral over [a, b] of the CIC triangle Lambda(s - u) = max(0, 1 - |s - u|) (Fractions)."""
    def prim_left(s):   # primitive of 1 + (s - u) on [u-1, u]
        z = s - u
        return z + z * z / 2
    def prim_right(s):  # primitive of 1 - (s - u) on [u, u+1]
        z = s - u
        return z - z * z / 2
    tot = Fraction(0)
    lo, hi = max(a, u - 1), min(b, u)
    if hi > lo:
        tot += prim_left(hi) - prim_left(lo)
    lo, hi = max(a, u), min(b, u + 1)
    if hi > lo:
        tot += prim_right(hi) - prim_right(lo)
    return tot


def node_weights_1d(u, n=12):
    """Oracle weights of a unit charge at grid coordinate u on a 1-D line of n nodes (via the 3-D deposit)."""
    lo, d = (0.0, 0.0, 0.0), (1.0, 1.0, 1.0)
    rho, n_in = O.deposit_cic(np.array([float(u)]), np.array([5.0]), np.array([5.0]), (n, n, n), lo, d, 1.0, order=2)
    assert n_in == 1
    assert rho[5, 5, :].sum() == pytest.approx(0.75 * 0.75, rel=1e-15)       # y, t on a node: weights (1/8, 3/4, 1/8)
    return rho[5, 5, :] / (0.75 * 0.75)


@pytest.mark.parametrize("u", [3.0, 3.25, 3.5 - 2**-30, 3.5, 3.75, 4.0 - 2**-40, 6.125, 2.0009765625])
def test_weights_are_the_cell_average_of_the_cic_triangle(u):
    """Definition of the quadratic B-spline: B2 = B1 * box, i.e. the weight of node m is the integral of the CIC
    triangle centred on the particle over the node's cell [m-1/2, m+1/2].  Exact rational integral vs the oracle."""
    w = node_weights_1d(u)
    uf = Fraction(u)
    for m in range(12):
        ref = triangle_integral(Fraction(2 * m - 1, 2), Fraction(2 * m + 1, 2), uf)
        assert abs(Fraction(float(w[m])) - ref) <= Fraction(1, 2**50), (m, float(ref), w[m])


def test_moment_identities_of_the_quadratic_spline():
    """sum w = 1, sum w m = u (linear reproduction), sum w (m - u)^2 = 1/4 for every position."""
    rng = np.random.default_rng(3)
    m = np.arange(12, dtype=np.float64)
    for u in rng.uniform(1.0, 10.0, 50):
        w = node_weights_1d(u)
        assert np.count_nonzero(w) <= 3
        assert abs(w.sum() - 1.0) <= 4e-16
        assert abs((w * m).sum() - u) <= 1e-14
        assert abs((w * (m - u) ** 2).sum() - 0.25) <= 1e-14


def brute_tsc(x, y, t, shape, lo, d, qw, zscale):
    """R16 restated particle by particle with exact rational accumulation of the fp64 node values."""
    import math
    nx, ny, nz = shape
    rho = [[[Fraction(0) for _ in range(nx)] for _ in range(ny)] for _ in range(nz)]
    inside = 0
    for p in range(len(x)):
        q = (x[p], y[p], zscale * t[p])
        base, w = [], []
        for a, n in enumerate((nx, ny, nz)):
            u = (q[a] - lo[a]) * (1.0 / d[a])
            v = u + 0.5
            if not (v >= 1.0 and v < n - 1):
                break
            j = math.floor(v)
            dl = u - j
            w.append((0.5 * ((0.5 - dl) * (0.5 - dl)), 0.75 - dl * dl, 0.5 * ((0.5 + dl) * (0.5 + dl))))
            base.append(j - 1)
        else:
            inside += 1
            for dz in range(3):
                for dy in range(3):
                    for dx in range(3):
                        ww = (w[0][dx] * w[1][dy]) * w[2][dz]
                        rho[base[2] + dz][base[1] + dy][base[0] + dx] += Fraction(qw * ww)
    return np.array([[[float(v) for v in row] for row in plane] for plane in rho]), inside


@pytest.mark.parametrize("zscale", [1.0, -1.8])
def test_brute_force_tiny_grid(zscale):
    rng = np.random.default_rng(77)
    shape, lo, d = (5, 6, 4), (-1.0, -2.0, -0.5), (0.7, 1.1, 0.6)
    n = 14
    x = rng.uniform(-1.2, 2.0, n)
    y = rng.uniform(-2.2, 3.8, n)
    t = rng.uniform(-0.6, 1.4, n) / zscale
    ref, n_ref = brute_tsc(x, y, t, shape, lo, d, 1e-10, zscale)
    rho, n_in = O.deposit_cic(x, y, t, shape, lo, d, 1e-10, zscale, order=2)
    assert n_in == n_ref and 0 < n_in < n
    assert np.array_equal(rho, ref)


def test_total_charge_and_dipole_moment_are_conserved():
    rng = np.random.default_rng(9)
    shape, lo, d = (16, 16, 16), (-4e-3, -4e-3, -4e-3), (0.5e-3, 0.6e-3, 0.55e-3)
    n = 5000
    x, y, t = [rng.uniform(-2e-3, 2e-3, n) for _ in range(3)]
    qw = 1e-9 / n
    rho, n_in = O.deposit_cic(x, y, t, shape, lo, d, qw, order=2)
    assert n_in == n
    assert abs(rho.sum() - 1e-9) <= 1e-9 * 1e-13
    xn = lo[0] + d[0] * np.arange(16)
    assert abs((rho.sum(axis=(0, 1)) * xn).sum() - qw * x.sum()) <= 1e-13 * qw * np.abs(x).sum()


def test_gather_reproduces_linear_fields_and_offsets_quadratics_by_a_quarter():
    """Quadratic B-spline interpolation: exact on 1, x, y, z, xy, ...; on x^2 it returns x^2 + d^2/4."""
    rng = np.random.default_rng(10)
    shape, lo, d = (12, 11, 10), (-1.0, 0.5, 2.0), (0.25, 0.5, 0.125)
    nx, ny, nz = shape
    X = lo[0] + d[0] * np.arange(nx)[None, None, :] + 0 * np.zeros((nz, ny, nx))
    Y = lo[1] + d[1] * np.arange(ny)[None, :, None] + 0 * np.zeros((nz, ny, nx))
    Z = lo[2] + d[2] * np.arange(nz)[:, None, None] + 0 * np.zeros((nz, ny, nx))
    n = 200
    x = rng.uniform(lo[0] + 0.6 * d[0], lo[0] + (nx - 1.6) * d[0], n)
    y = rng.uniform(lo[1] + 0.6 * d[1], lo[1] + (ny - 1.6) * d[1], n)
    t = rng.uniform(lo[2] + 0.6 * d[2], lo[2] + (nz - 1.6) * d[2], n)
    E = (1.0 + 2.0 * X - 3.0 * Y + 0.5 * Z, X * Y * Z, X * X)
    ex, ey, ez = O.gather_field(x, y, t, shape, lo, d, E, order=2)
    assert np.max(np.abs(ex - (1.0 + 2.0 * x - 3.0 * y + 0.5 * t))) <= 1e-13
    assert np.max(np.abs(ey - x * y * t)) <= 1e-13
    assert np.max(np.abs(ez - (x * x + d[0] ** 2 / 4))) <= 1e-13
    # and it is a different interpolant from order 1: trilinear gives x^2 + w0 w1 d^2
    ez1 = O.gather_field(x, y, t, shape, lo, d, E, order=1)[2]
    assert np.max(np.abs(ez1 - ez)) > 1e-3 * d[0] ** 2


def test_deposit_gather_adjoint_identity():
    """sum_nodes rho * phi == q_w * sum_p gather(phi)(x_p): both sides use the same 27 weights."""
    rng = np.random.default_rng(12)
    shape, lo, d = (9, 8, 7), (0.0, 0.0, 0.0), (1.0, 0.5, 2.0)
    n = 300
    x = rng.uniform(0.0, 8.0, n)            # includes outside particles
    y = rng.uniform(0.0, 3.5, n)
    t = rng.uniform(0.0, 12.0, n)
    phi = rng.standard_normal((7, 8, 9))
    rho, n_in = O.deposit_cic(x, y, t, shape, lo, d, 0.37, order=2)
    g = O.gather_field(x, y, t, shape, lo, d, (phi, phi, phi), order=2)[0]
    assert 0 < n_in < n
    assert abs((rho * phi).sum() - 0.37 * g.sum()) <= 1e-12 * 0.37 * np.abs(g).sum()


def test_boundary_rule_R16():
    """Inside <=> 1 <= nearest node <= n-2, i.e. 0.5 <= u < n-1.5 on the rounded v = u + 0.5; NaN outside."""
    shape, lo, d = (6, 6, 6), (0.0, 0.0, 0.0), (1.0, 1.0, 1.0)
    mid = np.array([2.5])
    cases = [(0.5, True), (0.5 - 2**-53, False), (0.49, False), (4.5 - 2**-50, True), (4.5, False), (1.0, True),
             (np.nan, False), (-3.0, False), (np.inf, False)]
    for u, inside in cases:
        for axis in range(3):
            q = [mid.copy(), mid.copy(), mid.copy()]
            q[axis] = np.array([u])
            rho, n_in = O.deposit_cic(q[0], q[1], q[2], shape, lo, d, 1.0, order=2)
            assert n_in == int(inside), (u, axis)
            assert (rho.sum() > 0) == inside
    # the gather leaves outside particles untouched
    c = [np.array([0.2]), np.array([1.0]), mid.copy(), np.array([2.0]), mid.copy(), np.array([3.0])]
    E = tuple(np.ones((6, 6, 6)) for _ in range(3))
    assert O.gather_kick(c, shape, lo, d, E, (1.0, 1.0, 1.0), order=2) == 0
    assert c[1][0] == 1.0 and c[3][0] == 2.0 and c[5][0] == 3.0
