"""Pins for the oracle's non-linearised maps (readings R17 exact drift, R18 sinusoidal short RF;
PAPER.md l.168 "non-linear elements, RF-modeling").  Independent of the oracle's formulas: relativistic kinematics of a
free particle / of an energy kick written out in 50-digit arithmetic from (E, P), the linear limits R4 and R9,
symplecticity of numerical Jacobians, slice composition, periodicity."""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle as O
import workloads as W
from _util import J6

mp.mp.dps = 50
KIN, MASS = 2000.0, W.MASS_PROTON_MEV
G0, BG0, B0 = O.ref_from_kinetic(KIN, MASS)


def one(v, lattice, gamma=G0):
    c = [np.array([float(a)]) for a in v]
    g, _ = O.track(c, lattice, 1, gamma)
    return [float(a[0]) for a in c], g


def kin_free_flight(v, h):
    """A free particle crossing a slab of thickness h, from (E, P) only: velocity = P c^2 / E, straight line."""
    x, px, y, py, t, pt = [mp.mpf(a) for a in v]
    g0, bg0 = mp.mpf(G0), mp.sqrt(mp.mpf(G0) ** 2 - 1)
    b0 = bg0 / g0
    E = g0 - pt * bg0                         # total energy / mc^2   (pt = -(E - E0)/(p0 c), p0 = mc bg0)
    P = mp.sqrt(E * E - 1)                    # |momentum| / mc
    Px, Py = px * bg0, py * bg0
    Ps = mp.sqrt(P * P - Px * Px - Py * Py)
    bx, by, bs = Px / E, Py / E, Ps / E       # velocity / c
    cT = h / bs                               # c * time to cross the slab
    return [x + bx * cT, px, y + by * cT, py, t + cT - h / b0, pt]


@pytest.mark.parametrize("v", [(1e-3, 2e-3, -1e-3, 1e-3, 5e-4, 1e-3), (0.0, 3e-2, 0.0, -2e-2, 0.0, -2e-2),
                               (1e-4, 0.0, 0.0, 0.0, 1e-3, 0.1), (0.0, 0.2, 0.0, 0.1, 0.0, 0.0)])
def test_exact_drift_is_relativistic_free_flight(v):
    h = 0.73
    got, g = one(v, [("drift_exact", h, 1)])
    ref = kin_free_flight(v, mp.mpf(h))
    assert g == G0
    for a, b in zip(got, ref):
        # t: h ((1/b0 - pt)/ps - 1/b0) subtracts two numbers of order 1/b0, so its fp64 error is ~ eps h, not eps |dt|
        assert abs(mp.mpf(a) - b) <= 4e-16 * max(abs(b), mp.mpf(h)), (a, b)


def test_exact_drift_reduces_to_R4_at_small_amplitude_and_differs_at_large():
    h = 1.3
    for amp, tol in ((1e-7, 1e-13), (1e-5, 1e-9)):
        v = (amp, amp, -amp, 2 * amp, amp, -amp)
        a, _ = one(v, [("drift_exact", h, 1)])
        b, _ = one(v, [("drift", h, 1)])
        for i in (0, 2, 4):
            assert abs(a[i] - b[i]) <= tol * h * amp / 1e-7 * 1e-7 + 4 * amp * amp * h
    big = (0.0, 1e-2, 0.0, 1e-2, 0.0, 1e-2)
    a, _ = one(big, [("drift_exact", h, 1)])
    b, _ = one(big, [("drift", h, 1)])
    assert abs(a[0] - b[0]) > 1e-5 * abs(b[0])          # second-order terms are there


def numerical_jacobian(lattice, v0, eps):
    M = np.zeros((6, 6))
    for j in range(6):
        vp, vm = list(v0), list(v0)
        vp[j] += eps[j]
        vm[j] -= eps[j]
        a, _ = one(vp, lattice)
        b, _ = one(vm, lattice)
        M[:, j] = (np.array(a) - np.array(b)) / (2 * eps[j])
    return M


def test_exact_drift_jacobian_is_symplectic():
    v0 = (1e-3, 2e-2, -1e-3, -1e-2, 5e-4, 1e-2)
    M = numerical_jacobian([("drift_exact", 0.9, 1)], v0, [1e-6] * 6)
    assert np.max(np.abs(M.T @ J6 @ M - J6)) <= 1e-8
    assert abs(M[0, 1] - 0.9) > 1e-4                      # not the linear drift's matrix


def test_exact_drift_slices_compose():
    v = (1e-3, 2e-2, -1e-3, -1e-2, 5e-4, 1e-2)
    a, _ = one(v, [("drift_exact", 2.0, 1)])
    b, _ = one(v, [("drift_exact", 2.0, 7)])
    c, _ = one(v, [("drift_exact", 0.5, 1), ("drift_exact", 1.5, 3)])
    for i in range(6):
        assert abs(a[i] - b[i]) <= 4e-16 * max(abs(a[i]), 1e-3) and abs(a[i] - c[i]) <= 4e-16 * max(abs(a[i]), 1e-3)


VHAT, FREQ, PHI = 2.0e-3, 2.0e8, -30.0
KRF = 2 * np.pi * FREQ / 299792458.0


def kin_rf(v, vhat, freq, phi_deg):
    """Energy kick qV cos(omega dt + phi) on the particle, qV cos(phi) on the reference; everything else from (E, P)."""
    x, px, y, py, t, pt = [mp.mpf(a) for a in v]
    g0 = mp.mpf(G0)
    bg0 = mp.sqrt(g0 * g0 - 1)
    phi = mp.mpf(phi_deg) * mp.pi / 180
    k = 2 * mp.pi * mp.mpf(freq) / mp.mpf(299792458)
    E = g0 - pt * bg0
    E1 = E + mp.mpf(vhat) * mp.cos(k * t + phi)
    g1 = g0 + mp.mpf(vhat) * mp.cos(phi)
    bg1 = mp.sqrt(g1 * g1 - 1)
    # transverse momenta Px = px * p0 are unchanged by a purely longitudinal kick; renormalise by the new p0
    return [x, px * bg0 / bg1, y, py * bg0 / bg1, t, -(E1 - g1) / bg1], g1


@pytest.mark.parametrize("v", [(1e-3, 1e-3, 2e-3, -1e-3, 0.3, 1e-3), (0.0, 0.0, 0.0, 0.0, -0.11, -2e-3),
                               (1e-3, 2e-3, 0.0, 0.0, 0.0, 5e-3), (0.0, 1e-3, 0.0, 1e-3, 7.0, 0.0)])
def test_sinusoidal_rf_is_the_exact_energy_kick(v):
    got, g = one(v, [("shortrf_sin", 0.0, 1, VHAT, FREQ, PHI)])
    ref, g1 = kin_rf(v, VHAT, FREQ, PHI)
    assert abs(mp.mpf(g) - g1) <= 2e-16 * g1
    # the fp64 phase k t + phi carries an error ~ eps |k t + phi|, which the cosine passes on: scale the bar by it
    cond = (1 + abs(KRF * v[4] + np.radians(PHI))) * VHAT / BG0
    for a, b in zip(got, ref):
        assert abs(mp.mpf(a) - b) <= 4e-16 * max(abs(b), cond), (a, b)


def test_sinusoidal_rf_reduces_to_R9_and_differs_at_large_t():
    for t, tol in ((1e-6, 1e-15), (1e-4, 1e-11)):
        v = (0.0, 1e-3, 0.0, 1e-3, t, 1e-3)
        a, ga = one(v, [("shortrf_sin", 0.0, 1, VHAT, FREQ, PHI)])
        b, gb = one(v, [("shortrf", 0.0, 1, VHAT, FREQ, PHI)])
        assert ga == gb
        assert abs(a[5] - b[5]) <= VHAT / BG0 * (KRF * t) ** 2 + tol * 1e-3
        assert a[1] == b[1] and a[3] == b[3]
    v = (0.0, 0.0, 0.0, 0.0, 0.2, 0.0)
    a, _ = one(v, [("shortrf_sin", 0.0, 1, VHAT, FREQ, PHI)])
    b, _ = one(v, [("shortrf", 0.0, 1, VHAT, FREQ, PHI)])
    assert abs(a[5] - b[5]) > 0.05 * abs(b[5])


def test_sinusoidal_rf_jacobian_is_symplectic_up_to_the_momentum_rescaling():
    lat = [("shortrf_sin", 0.0, 1, VHAT, FREQ, PHI)]
    v0 = (1e-3, 1e-3, -1e-3, 2e-3, 0.25, 1e-3)
    M = numerical_jacobian(lat, v0, [1e-6, 1e-6, 1e-6, 1e-6, 1e-4, 1e-6])
    _, g1 = one(v0, lat)
    r = BG0 / np.sqrt(g1 * g1 - 1)
    assert np.max(np.abs(M.T @ J6 @ M - r * J6)) <= 1e-8
    assert abs(M[5, 4] - VHAT / np.sqrt(g1 * g1 - 1) * KRF * np.sin(KRF * 0.25 + np.radians(PHI))) <= 1e-9


def test_sinusoidal_rf_is_periodic_in_t_and_neutral_on_the_reference():
    lam = 299792458.0 / FREQ
    a, _ = one((0, 0, 0, 0, 0.1, 1e-3), [("shortrf_sin", 0.0, 1, VHAT, FREQ, PHI)])
    b, _ = one((0, 0, 0, 0, 0.1 + lam, 1e-3), [("shortrf_sin", 0.0, 1, VHAT, FREQ, PHI)])
    assert abs(a[5] - b[5]) <= 1e-15
    c, g = one((0, 0, 0, 0, 0.0, 0.0), [("shortrf_sin", 0.0, 1, VHAT, FREQ, PHI)])
    assert c == [0.0] * 6 and g == G0 + VHAT * np.cos(np.radians(PHI))


def test_nonlinear_elements_argument_checks():
    c = [np.zeros(1) for _ in range(6)]
    with pytest.raises(ValueError):
        O.track(c, [("shortrf_sin", 0.0, 2, VHAT, FREQ, PHI)], 1, G0)       # thin element: nslice must be 1
    with pytest.raises(ValueError):
        O.track(c, [("drift_exact", -1.0, 1)], 1, G0)


# ---- R20 chromatic quadrupole ----------------------------------------------------------------------------------------
def ode_quad(v, h, k, expanded):
    """40-digit integration of Hamilton's equations in s.  expanded=True: H with the square root expanded in (px, py) only
    (the reading's Hamiltonian); False: the full square root (SURVEY 8(c) derivation sketch with a quadrupole term)."""
    mp.mp.dps = 40
    x, px, y, py, t, pt = [mp.mpf(a) for a in v]
    g0 = mp.mpf(G0)
    b0 = mp.sqrt(g0 * g0 - 1) / g0
    opd = mp.sqrt(1 - 2 * pt / b0 + pt * pt)

    def rhs(s, u):
        X, PX, Y, PY, T = u
        if expanded:
            inv = 1 / opd
            tdot = (1 / b0 - pt) / opd * (1 + (PX * PX + PY * PY) / (2 * opd * opd)) - 1 / b0
        else:
            ps = mp.sqrt(opd * opd - PX * PX - PY * PY)
            inv = 1 / ps
            tdot = (1 / b0 - pt) / ps - 1 / b0
        return [PX * inv, -k * X, PY * inv, k * Y, tdot]

    sol = mp.odefun(rhs, 0, [x, px, y, py, t])
    out = sol(mp.mpf(h))
    mp.mp.dps = 50
    return [out[0], out[1], out[2], out[3], out[4], pt]


@pytest.mark.parametrize("k", [1.3, -0.8])
@pytest.mark.parametrize("v", [(1e-3, 2e-3, -1e-3, 1e-3, 5e-4, 1e-2), (2e-3, -1e-3, 1e-3, 2e-3, 0.0, -3e-2)])
def test_chromatic_quad_is_the_flow_of_its_hamiltonian(k, v):
    h = 0.6
    got, g = one(v, [("quad_chromatic", h, 1, k)])
    ref = ode_quad(v, h, k, expanded=True)
    assert g == G0
    for i, (a, b) in enumerate(zip(got, ref)):
        tol = 4e-16 * h if i == 4 else 4e-16 * max(abs(b), 1e-3)      # t: difference of two O(h/beta0) numbers
        assert abs(mp.mpf(a) - b) <= tol, (i, a, b)
    # and that Hamiltonian is the full square-root one up to fourth order in the transverse momenta: the velocities
    # px/ps and px/(1+d) differ by a relative p_perp^2/2, i.e. the coordinates by O(h p_perp^3); t by O(h p_perp^4)
    exact = ode_quad(v, h, k, expanded=False)
    pperp = math.hypot(max(abs(v[1]), abs(float(exact[1]))), max(abs(v[3]), abs(float(exact[3]))))
    for i in (0, 1, 2, 3):
        assert abs(mp.mpf(got[i]) - exact[i]) <= 2.0 * h * pperp ** 3 * max(1.0, abs(k) * h)
        assert abs(mp.mpf(got[i]) - exact[i]) > 0
    assert abs(mp.mpf(got[4]) - exact[4]) <= 2.0 * h * pperp ** 4 + 4e-16 * h


def test_chromatic_quad_limits_and_plane_exchange():
    h, k = 0.8, 1.1
    v = (1e-3, 2e-3, -1e-3, 1e-3, 5e-4, 0.0)
    a, _ = one(v, [("quad_chromatic", h, 1, k)])
    b, _ = one(v, [("quad", h, 1, k)])
    for i in range(4):                                   # on momentum: the transverse map is R5
        assert abs(a[i] - b[i]) <= 4e-16 * max(abs(b[i]), 1e-3)
    assert a[4] > b[4]                                   # ... but the path is longer than the reference's
    off = (1e-3, 2e-3, -1e-3, 1e-3, 5e-4, 2e-2)          # off momentum (pt > 0: lower energy): stronger focusing
    c, _ = one(off, [("quad_chromatic", h, 1, k)])
    d, _ = one(off, [("quad", h, 1, k)])
    assert abs(c[0] - d[0]) > 1e-3 * abs(d[0])
    # k < 0 is k > 0 with the planes exchanged
    sw = (v[2], v[3], v[0], v[1], v[4], 1e-2)
    e, _ = one((v[0], v[1], v[2], v[3], v[4], 1e-2), [("quad_chromatic", h, 1, -k)])
    f, _ = one(sw, [("quad_chromatic", h, 1, k)])
    assert [e[0], e[1], e[2], e[3], e[4]] == [f[2], f[3], f[0], f[1], f[4]]
    # k = 0: paraxial chromatic drift, continuous limit of small k
    z, _ = one(off, [("quad_chromatic", h, 1, 0.0)])
    s_, _ = one(off, [("quad_chromatic", h, 1, 1e-12)])
    for i in range(5):
        assert abs(z[i] - s_[i]) <= 1e-12 * max(abs(z[i]), 1e-3)


def test_chromatic_quad_jacobian_is_symplectic_and_slices_compose():
    v0 = (1e-3, 2e-3, -1e-3, 1e-3, 5e-4, 1e-2)
    M = numerical_jacobian([("quad_chromatic", 0.7, 1, 1.4)], v0, [1e-6] * 6)
    assert np.max(np.abs(M.T @ J6 @ M - J6)) <= 1e-8
    assert abs(M[0, 5]) > 1e-5                            # chromatic coupling: x depends on pt
    a, _ = one(v0, [("quad_chromatic", 0.7, 1, 1.4)])
    b, _ = one(v0, [("quad_chromatic", 0.7, 5, 1.4)])
    for i in range(6):
        assert abs(a[i] - b[i]) <= (5 * 4e-16 * 0.7 if i == 4 else 2e-15 * max(abs(a[i]), 1e-3))   # t: eps h per slice
