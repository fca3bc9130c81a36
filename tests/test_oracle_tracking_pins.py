"""Pins for the oracle's tracking maps (R1-R9) against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin is something OTHER than the oracle's own
formula: values printed in the paper (tests/golden/paper_values.txt), exact relativistic kinematics
and exact circular-orbit geometry evaluated in 50-digit mpmath, textbook closed forms, group
properties (symplecticity, slice composition) and conservation laws.
"""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle as O
import workloads as W
from _util import J6, matrix_of, paper_values, rms_emittance

mp.mp.dps = 50
ME, MP_ = W.MASS_ELECTRON_MEV, W.MASS_PROTON_MEV


def track_fn(lattice, gamma, nturns=1):
    def f(c):
        return O.track(c, lattice, nturns, gamma)
    return f


def M_of(lattice, gamma, nturns=1):
    return matrix_of(track_fn(lattice, gamma, nturns))


GAMMA_P2GEV = O.ref_from_kinetic(2000.0, MP_)[0]
GAMMA_E2GEV = O.ref_from_kinetic(2000.0, ME)[0]
GAMMA_E5GEV = O.ref_from_kinetic(5000.0, ME)[0]
GAMMA_P1GEV = O.ref_from_kinetic(1000.0, MP_)[0]


# ------------------------------------------------------------------------------------------------
# R2 reference particle
# ------------------------------------------------------------------------------------------------
def test_ref_kinetic_energy_reading():
    """PAPER.md l.138 '2.5 MeV proton beam': only a KINETIC reading gives gamma > 1 for a proton."""
    pv = paper_values()
    g, bg, b = O.ref_from_kinetic(pv["iota_proton_kinetic_MeV"], MP_)
    assert g > 1.0 and 0.0 < b < 1.0
    # textbook: gamma = 1 + T/mc^2 ; beta*gamma = sqrt(T(T+2mc^2))/mc^2
    T, m = mp.mpf(2.5), mp.mpf(MP_)
    assert abs(g - float(1 + T / m)) < 1e-15
    # R2 evaluates sqrt(gamma^2-1) in fp64: cancellation ~ ulp(1)/(gamma^2-1) = 2e-14 at 2.5 MeV
    assert abs(bg - float(mp.sqrt(T * (T + 2 * m)) / m)) < 1e-13 * bg
    assert abs(b - bg / g) < 1e-16


def test_ref_values_2gev_electron():
    g, bg, b = O.ref_from_kinetic(2000.0, ME)
    E, m = mp.mpf(2000) + mp.mpf(ME), mp.mpf(ME)
    assert abs(g - float(E / m)) / g < 1e-15
    assert abs(b - float(mp.sqrt(1 - (m / E) ** 2))) < 1e-15


# ------------------------------------------------------------------------------------------------
# R4 drift
# ------------------------------------------------------------------------------------------------
def test_drift_matrix_closed_form():
    h = 0.37
    M = M_of([("drift", h, 1)], GAMMA_P2GEV)
    bg = O.ref_from_kinetic(2000.0, MP_)[1]
    E = np.eye(6)
    E[0, 1] = h
    E[2, 3] = h
    E[4, 5] = h / bg**2
    assert np.max(np.abs(M - E)) < 1e-16


@pytest.mark.parametrize("kin,mass", [(2000.0, MP_), (2.5, MP_), (5000.0, ME)])
def test_drift_time_of_flight_exact_kinematics(kin, mass):
    """t-row pin: exact relativistic time of flight of an off-energy particle over length L,
    c*dt = L (1/beta(E) - 1/beta0), with pt = -(E-E0)/(p0 c); first order in pt."""
    L = mp.mpf("1.75")
    m = mp.mpf(mass)
    E0 = mp.mpf(kin) + m
    p0 = mp.sqrt(E0**2 - m**2)

    def ct(pt):
        E = E0 - pt * p0
        beta = mp.sqrt(E**2 - m**2) / E
        return L / beta - L / (p0 / E0)

    exact = mp.diff(ct, 0)
    g = O.ref_from_kinetic(kin, mass)[0]
    M = M_of([("drift", float(L), 1)], g)
    assert abs(M[4, 5] - float(exact)) / float(exact) < 1e-12


# ------------------------------------------------------------------------------------------------
# R5 quad
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("k", [1.0, -1.0, 2.3, -0.17])
def test_quad_matrix_closed_form(k):
    h = 0.8
    M = M_of([("quad", h, 1, k)], GAMMA_E2GEV)
    w = mp.sqrt(abs(k))
    F = np.array([[float(mp.cos(w * h)), float(mp.sin(w * h) / w)], [float(-w * mp.sin(w * h)), float(mp.cos(w * h))]])
    D = np.array([[float(mp.cosh(w * h)), float(mp.sinh(w * h) / w)], [float(w * mp.sinh(w * h)), float(mp.cosh(w * h))]])
    bg = O.ref_from_kinetic(2000.0, ME)[1]
    E = np.eye(6)
    E[0:2, 0:2] = F if k > 0 else D      # k > 0 focuses x (reading R5)
    E[2:4, 2:4] = D if k > 0 else F
    E[4, 5] = h / bg**2
    assert np.max(np.abs(M - E)) < 4e-16


def test_quad_solves_hill_equation():
    """x'' = -k x, y'' = +k y: compare against a 50-digit Taylor integration of the ODE."""
    k, h = 1.3, 0.6
    sol = mp.odefun(lambda s, v: [v[1], -k * v[0], v[3], k * v[2]], 0, [mp.mpf("1e-3"), mp.mpf("2e-4"), mp.mpf("-5e-4"), mp.mpf("1e-4")])
    ref = [float(v) for v in sol(h)]
    c = [np.array([1e-3]), np.array([2e-4]), np.array([-5e-4]), np.array([1e-4]), np.zeros(1), np.zeros(1)]
    O.track(c, [("quad", h, 1, k)], 1, GAMMA_E2GEV)
    for a, b in zip(c[:4], ref):
        assert abs(a[0] - b) < 1e-18 + 1e-15 * abs(b)


def test_quad_k0_is_drift():
    A = M_of([("quad", 0.7, 3, 0.0)], GAMMA_P2GEV)
    B = M_of([("drift", 0.7, 3)], GAMMA_P2GEV)
    assert np.array_equal(A, B)


# ------------------------------------------------------------------------------------------------
# paper values P1 / P2 (FODO cell of Listing 1)
# ------------------------------------------------------------------------------------------------
def fodo_cell_matrix(ns):
    return M_of(W.fodo_cell(ns), GAMMA_E2GEV)


def test_P1_fodo_phase_advance_paper_value():
    """'zero-current phase advance of 67.8 degrees per cell'."""
    pv = paper_values()
    M = fodo_cell_matrix(int(pv["listing_ns"]))
    for blk in (M[0:2, 0:2], M[2:4, 2:4]):
        cosmu = 0.5 * np.trace(blk)
        mu = math.degrees(math.acos(cosmu))
        assert round(mu, 1) == pv["fodo_phase_advance_deg"]
        # closed form of the cell trace (thick-lens FODO, phi = sqrt(k) L = 1, d = 0.5 m drift between)
        phi, d, k = 1.0, 0.5, 1.0
        closed = (math.cos(phi) * math.cosh(phi) + d * math.sqrt(k) * (math.cos(phi) * math.sinh(phi) - math.sin(phi) * math.cosh(phi))
                  - 0.5 * d * d * k * math.sin(phi) * math.sinh(phi))
        assert abs(cosmu - closed) < 5e-15


def test_P2_matched_beam_paper_listing():
    """the listing's matched-beam parameters are the periodic Twiss of the cell.
    sigma* are phase-ellipse intercepts: beta = sigmaX/(sigmaPx sqrt(1-mu^2)), |alpha| = |mu|/sqrt(1-mu^2),
    emittance = sigmaX sigmaPx / sqrt(1-mu^2) = 2 nm (l.66, l.112)."""
    pv = paper_values()
    M = fodo_cell_matrix(int(pv["listing_ns"]))
    mu_c = pv["listing_muxpx"]
    root = math.sqrt(1.0 - mu_c * mu_c)
    beta_paper = pv["listing_sigmaX"] / (pv["listing_sigmaPx"] * root)
    alpha_paper = abs(mu_c) / root
    eps_paper = pv["listing_sigmaX"] * pv["listing_sigmaPx"] / root
    assert abs(eps_paper - pv["fodo_emittance_m"]) / 2e-9 < 1e-9
    for blk, sign in ((M[0:2, 0:2], -1.0), (M[2:4, 2:4], +1.0)):
        cosmu = 0.5 * np.trace(blk)
        sinmu = math.copysign(math.sqrt(1 - cosmu**2), blk[0, 1])
        beta = blk[0, 1] / sinmu
        alpha = (blk[0, 0] - blk[1, 1]) / (2 * sinmu)
        assert abs(beta - beta_paper) / beta_paper < 2e-9       # the listing prints 11 digits
        assert abs(abs(alpha) - alpha_paper) / alpha_paper < 1e-8   # listing agrees to 3e-9 (9 digits)
        assert math.copysign(1.0, alpha) == sign                # alpha_x < 0 < alpha_y with k>0 focusing x
    assert pv["listing_muxpx"] == -pv["listing_muypy"]


def test_workload_twiss_values():
    """The Twiss numbers hard-coded in workloads/ are the periodic solution of the oracle's cell."""
    def twiss(blk):
        cosmu = 0.5 * np.trace(blk)
        sinmu = math.copysign(math.sqrt(1 - cosmu**2), blk[0, 1])
        return blk[0, 1] / sinmu, (blk[0, 0] - blk[1, 1]) / (2 * sinmu)

    M = fodo_cell_matrix(25)
    bx, ax = twiss(M[0:2, 0:2])
    by, ay = twiss(M[2:4, 2:4])
    assert abs(bx - W.FODO_BETA) < 1e-12 and abs(by - W.FODO_BETA) < 1e-12
    assert abs(ax - W.FODO_ALPHA_X) < 1e-12 and abs(ay + W.FODO_ALPHA_X) < 1e-12
    Mr = M_of(W.ring_cell(0.0, 0.0), GAMMA_P1GEV)
    bx, ax = twiss(Mr[0:2, 0:2])
    by, ay = twiss(Mr[2:4, 2:4])
    assert abs(bx - W.RING_TWISS_X[0]) < 1e-12 and abs(ax - W.RING_TWISS_X[1]) < 1e-12
    assert abs(by - W.RING_TWISS_Y[0]) < 1e-12 and abs(ay - W.RING_TWISS_Y[1]) < 1e-12
    # RF frequency of config 3 = h * beta0 * c / C at injection, h = 1
    beta0 = O.ref_from_kinetic(1000.0, MP_)[2]
    assert abs(W.RING_RF_FREQ_HZ - beta0 * W.C_LIGHT / W.RING_LENGTH_M) / W.RING_RF_FREQ_HZ < 1e-15
    lat = W.nonlinear_ring()
    assert len(lat) == 201 and abs(sum(e[1] for e in lat) - W.RING_LENGTH_M) < 1e-12
    # space-charge kick coefficients of config 4 (R12)
    g, bg, b = O.ref_from_kinetic(1000.0, MP_)
    sc = W.spacecharge_config("A", n=1)
    q_over_mc2 = 1.0 / (MP_ * 1e6)
    assert abs(sc.kick_coef[0] - q_over_mc2 * sc.ds / bg**2) / sc.kick_coef[0] < 1e-14
    assert abs(sc.kick_coef[2] - q_over_mc2 * sc.ds / bg) / sc.kick_coef[2] < 1e-14


# ------------------------------------------------------------------------------------------------
# symplecticity and group properties
# ------------------------------------------------------------------------------------------------
LINEAR_ELEMENTS = [
    [("drift", 0.33, 1)],
    [("quad", 0.9, 1, 1.7)],
    [("quad", 0.9, 4, -0.6)],
    [("sbend", 0.5, 1, 10.0)],
    [("sbend", 1.5, 3, -2.5)],
    [("dipedge", 0.0, 1, 0.05, 10.0, 0.02, 0.5)],
    [("dipedge", 0.0, 1, -0.3, -2.0, 0.0, 0.0)],
    [("multipole", 0.0, 1, 2, 0.4, -0.2)],
]


@pytest.mark.parametrize("lat", LINEAR_ELEMENTS)
@pytest.mark.parametrize("gamma", [GAMMA_P2GEV, GAMMA_E5GEV, 1.0026644])
def test_symplectic_linear_elements(lat, gamma):
    M = M_of(lat, gamma)
    assert np.max(np.abs(M.T @ J6 @ M - J6)) < 2e-15 * max(1.0, np.max(np.abs(M)) ** 2)


def test_symplectic_products():
    for lat, g in ((W.fodo_cell(10), GAMMA_P2GEV), (W.chicane(), GAMMA_E5GEV), (W.ring_cell(0, 0) * 3, GAMMA_P1GEV)):
        M = M_of(lat, g)
        assert np.max(np.abs(M.T @ J6 @ M - J6)) < 1e-13


@pytest.mark.parametrize("lat1,n", [(("quad", 1.0, 1, 1.0), 25), (("quad", 1.0, 1, -1.0), 10),
                                     (("sbend", 0.7, 1, 3.0), 7), (("drift", 0.5, 1), 5)])
def test_slice_composition(lat1, n):
    """R3: n maps of length L/n == one map of length L (group property of the flow)."""
    whole = M_of([lat1], GAMMA_P2GEV)
    sliced = M_of([(lat1[0], lat1[1], n) + tuple(lat1[3:])], GAMMA_P2GEV)
    assert np.max(np.abs(whole - sliced)) < 4e-15


def test_walk_order_and_turns():
    """nturns turns == the lattice concatenated nturns times; order matters (non-commuting maps)."""
    lat = W.fodo_cell(3)
    A = M_of(lat, GAMMA_P2GEV, nturns=3)
    B = M_of(lat * 3, GAMMA_P2GEV, nturns=1)
    assert np.array_equal(A, B)
    M1 = M_of(lat, GAMMA_P2GEV)
    assert np.max(np.abs(A - M1 @ M1 @ M1)) < 1e-13
    R = M_of(lat[::-1], GAMMA_P2GEV)
    assert np.max(np.abs(R - M1)) > 1e-3
    # element product in list order: M = M_last ... M_first
    Md, Mq = M_of([lat[0]], GAMMA_P2GEV), M_of([lat[1]], GAMMA_P2GEV)
    assert np.max(np.abs(M_of(lat[:2], GAMMA_P2GEV) - Mq @ Md)) < 1e-15


def test_reference_s_and_turn_bookkeeping():
    c = [np.zeros(1) for _ in range(6)]
    g, s = O.track(c, W.fodo_cell(2), 4, GAMMA_P2GEV, s=1.5)
    assert g == GAMMA_P2GEV and abs(s - (1.5 + 4 * 3.0)) < 1e-12


def test_invalid_lattices_rejected():
    c = [np.zeros(1) for _ in range(6)]
    for bad in ([("quad", 1.0, 0, 1.0)], [("sbend", 1.0, 1, 0.0)], [("multipole", 0.0, 1, 11, 1.0, 0.0)],
                [("multipole", 0.0, 2, 3, 1.0, 0.0)], [("drift", -1.0, 1)], [(99, 1.0, 1)]):
        with pytest.raises(ValueError):
            O.track(c, bad, 1, GAMMA_P2GEV)


# ------------------------------------------------------------------------------------------------
# R6 sector bend: exact circular-orbit geometry (50 digits), differentiated numerically
# ------------------------------------------------------------------------------------------------
def _sbend_exact(x0, px0, pt0, rho, h, kin, mass):
    """Exact hard-edge sector dipole for one particle in the mid-plane.  Reference: circle of radius
    rho about the origin, entering at (rho, 0) moving in +Y, bending towards the origin (rho>0);
    exit face = the ray at polar angle theta = h/rho.  Returns (x, px, t) at the exit face."""
    m = mp.mpf(mass)
    E0 = mp.mpf(kin) + m
    p0 = mp.sqrt(E0**2 - m**2)
    beta0 = p0 / E0
    E = E0 - pt0 * p0
    p = mp.sqrt(E**2 - m**2)
    beta = p / E
    R = rho * p / p0                      # radius scales with momentum in a fixed field
    a = mp.asin(px0 * p0 / p)             # angle to the reference direction; px = (P/p0) sin a
    th = h / rho
    P = (rho + x0, mp.mpf(0))
    # velocity direction (-sin a, cos a) rotated: +x outward; px>0 means moving outward
    v = (mp.sin(a), mp.cos(a))
    # centre of curvature: to the left of the velocity (counter-clockwise motion about the origin)
    C = (P[0] - R * v[1], P[1] + R * v[0])
    e = (mp.cos(th), mp.sin(th))
    # |s e - C|^2 = R^2  ->  s^2 - 2 s (e.C) + |C|^2 - R^2 = 0 ; outer root
    b = e[0] * C[0] + e[1] * C[1]
    cc = C[0] ** 2 + C[1] ** 2 - R**2
    s = b + mp.sqrt(b * b - cc)
    Q = (s * e[0], s * e[1])
    ang0 = mp.atan2(P[1] - C[1], P[0] - C[0])
    ang1 = mp.atan2(Q[1] - C[1], Q[0] - C[0])
    swept = ang1 - ang0
    path = R * swept
    # direction at Q: perpendicular to the radius from C, counter-clockwise
    vq = (-mp.sin(ang1), mp.cos(ang1))
    # reference direction at the exit face: (-sin th, cos th); outward normal e
    sin_a1 = vq[0] * e[0] + vq[1] * e[1]
    x1 = s - rho
    px1 = (p / p0) * sin_a1
    t1 = path / beta - h / beta0
    return x1, px1, t1


@pytest.mark.parametrize("rho,h,kin,mass", [(10.0, 0.5, 5000.0, ME), (2.5, 1.2, 1000.0, MP_), (1.0, 0.4, 2.5, MP_)])
def test_sbend_exact_geometry_first_order(rho, h, kin, mass):
    g, bg, beta = O.ref_from_kinetic(kin, mass)
    M = M_of([("sbend", h, 1, rho)], g)
    rho_, h_ = mp.mpf(rho), mp.mpf(h)
    cols = {0: lambda e: _sbend_exact(e, 0, 0, rho_, h_, kin, mass),
            1: lambda e: _sbend_exact(0, e, 0, rho_, h_, kin, mass),
            5: lambda e: _sbend_exact(0, 0, e, rho_, h_, kin, mass)}
    for col, fn in cols.items():
        for row_i, row in enumerate((0, 1, 4)):
            exact = float(mp.diff(lambda e: fn(e)[row_i], 0))
            assert abs(M[row, col] - exact) < 1e-11 * max(1.0, abs(exact)), (row, col, M[row, col], exact)
    # y-plane is a drift of the arc length; pt, px-py coupling absent
    assert abs(M[2, 3] - h) < 1e-16 and M[3, 3] == 1.0 and M[5, 5] == 1.0
    # t also picks up its own identity column
    assert M[4, 4] == 1.0


def test_sbend_limits_and_mirror():
    h = 0.8
    D = M_of([("drift", h, 1)], GAMMA_P2GEV)
    B = M_of([("sbend", h, 1, 1e9)], GAMMA_P2GEV)
    assert np.max(np.abs(D - B)) < 1e-8
    Mp = M_of([("sbend", h, 1, 3.0)], GAMMA_P2GEV)
    Mm = M_of([("sbend", h, 1, -3.0)], GAMMA_P2GEV)
    S = np.diag([-1.0, -1.0, 1.0, 1.0, 1.0, 1.0])       # x -> -x mirrors the bend
    assert np.max(np.abs(S @ Mp @ S - Mm)) < 1e-15


# ------------------------------------------------------------------------------------------------
# R7 dipole edge
# ------------------------------------------------------------------------------------------------
def test_dipedge_hard_edge_textbook():
    psi, rho = 0.21, 4.0
    M = M_of([("dipedge", 0.0, 1, psi, rho, 0.0, 0.0)], GAMMA_E5GEV)
    E = np.eye(6)
    E[1, 0] = math.tan(psi) / rho        # horizontally defocusing for psi > 0
    E[3, 2] = -math.tan(psi) / rho       # equal and opposite (curl B = 0)
    assert np.max(np.abs(M - E)) < 1e-16


def test_rectangular_magnet_geometry():
    """Sector body + exit edge psi = theta is a rectangular magnet entered normally: exact geometry says
    parallel rays stay parallel (R21 = 0), are displaced by x0 cos(theta) normal to the exit orbit
    (R11 = cos theta), and R12 = rho sin(theta), R22 = 1/cos(theta)."""
    rho, th = 10.0, 0.05
    M = M_of([("sbend", rho * th, 1, rho), ("dipedge", 0.0, 1, th, rho, 0.02, 0.5)], GAMMA_E5GEV)
    assert abs(M[1, 0]) < 1e-17
    assert abs(M[0, 0] - math.cos(th)) < 1e-16
    assert abs(M[0, 1] - rho * math.sin(th)) < 1e-15
    assert abs(M[1, 1] - 1.0 / math.cos(th)) < 1e-15


def test_dipedge_fringe_correction_direction():
    """Finite gap (g, K > 0) weakens the vertical edge focusing; g = 0 or K = 0 removes the correction.
    (Limits and sign only; the size of the correction is pinned by test_dipedge_fringe_term_vs_maxwell_ray_tracing.)"""
    psi, rho = 0.05, 10.0
    hard = M_of([("dipedge", 0.0, 1, psi, rho, 0.0, 0.5)], GAMMA_E5GEV)[3, 2]
    soft = M_of([("dipedge", 0.0, 1, psi, rho, 0.02, 0.5)], GAMMA_E5GEV)[3, 2]
    k0 = M_of([("dipedge", 0.0, 1, psi, rho, 0.02, 0.0)], GAMMA_E5GEV)[3, 2]
    assert hard == k0 == -math.tan(psi) / rho
    assert hard < soft < 0.0


# ---- R7 fringe term psi_c: pinned by ray tracing through an extended, Maxwell-consistent fringe field ----------
# Nothing below knows the expression for psi_c.  A pole face with normal e_n (pointing into the magnet at an entrance,
# out of it at an exit), e_tau along the face, e_y vertical, (e_n, e_tau, e_y) right-handed.  The mid-plane field falls
# off along the normal only: B_y(n, 0) = B0 f(n).  curl B = 0 then fixes the field off the mid-plane to first order in y:
#     B = B0 ( y f'(n), 0, f(n) )        (dB_n/dy = dB_y/dn; div B = 0 only adds -y^2 f''/2 to B_y, second order in y).
# A particle of momentum p and charge q obeys the Lorentz force, with path length s as the independent variable:
#     dr/ds = u,   du/ds = h u x b,   h = q B0 / p = 1/rho,   b = B / B0,   |u| = 1.
# The reference ray moves in the plane y = 0 and makes the angle psi with e_n where the field has vanished; rays started
# with a tiny vertical offset / slope give the 2 x 2 vertical transfer matrix M of the fringe region.  The hard-edge
# model of the same region (what a lattice of Sbend + DipEdge + Drift elements represents) is
#     M_model = D(L_body) . Edge . D(L_drift),
# the edge sitting where the field integral puts it (int f dn = length of full field), D(L) the vertical map of a drift
# or of a gradient-free sector-bend body of arc length L.  Hence Edge = D(-L_body) M D(-L_drift), and its (2,1) element is
# what the oracle's R43 = -tan(psi - psi_c)/rho has to equal, up to terms of second order in g/rho.  The fringe integral
# K = int f (1 - f) dn / g is computed from the profile by quadrature (its definition, include/bt.h).
def _fringe_profile(kind, g):
    if kind == "ramp":      # linear fall-off over 3 g  ->  K = 1/2, the value configs[2] uses
        w = 3.0 * g
        return (lambda n: min(max(n / w, 0.0), 1.0)), (lambda n: 1.0 / w if 0.0 < n < w else 0.0), [0.0, w], (0.0, w)
    lam = 0.7 * g           # smooth (tanh) fall-off: K = lam / (2 g) = 0.35
    return (lambda n: 0.5 * (1.0 + math.tanh(n / lam))), (lambda n: 0.5 / (lam * math.cosh(n / lam) ** 2)), [], (-22.0 * lam, 22.0 * lam)


def _trace_fringe(f, fp, breaks, span, h, theta0, y0, yp0):
    from scipy.integrate import solve_ivp

    def rhs(_s, w):
        n, _tau, y, un, ut, uy = w
        bn, bt, by = y * fp(n), 0.0, f(n)
        return [un, ut, uy, h * (ut * by - uy * bt), h * (uy * bn - un * by), h * (un * bt - ut * bn)]

    na, nb = span
    norm = math.sqrt(1.0 + yp0 * yp0)
    w = [na, 0.0, y0, math.cos(theta0) / norm, math.sin(theta0) / norm, yp0 / norm]
    s = 0.0
    for c in [b for b in breaks if na < b < nb] + [nb]:      # integrate from kink to kink of the profile
        def hit(_s, w, c=c):
            return w[0] - c
        hit.terminal, hit.direction = True, 1
        sol = solve_ivp(rhs, (s, s + 10.0 * (c - w[0]) + 1.0), w, method="DOP853", rtol=1e-13, atol=1e-18, events=hit,
                        max_step=(nb - na) / 50.0)
        assert sol.t_events[0].size == 1
        s, w = float(sol.t_events[0][0]), list(sol.y_events[0][0])
    return w


def _edge_matrix_from_ray_tracing(kind, g, rho, psi, face):
    """(Edge 2x2, K) for a face of a magnet with bending radius rho and TRANSPORT-sign edge angle psi (psi > 0 at both
    faces of a rectangular magnet)."""
    from scipy.integrate import quad
    h = 1.0 / rho
    f, fp, breaks, (na, nb) = _fringe_profile(kind, g)
    pts = breaks or None
    full = quad(f, na, nb, points=pts, epsabs=1e-15, epsrel=1e-13)[0]           # length of full field in the region
    K = quad(lambda n: f(n) * (1.0 - f(n)), na, nb, points=pts, epsabs=1e-15, epsrel=1e-13)[0] / g
    if face == "entrance":                      # field-free at na, full field at nb; the ray bends towards the normal
        theta0 = psi
        l_drift, arc = ((nb - full) - na) / math.cos(psi), None
    else:                                       # mirror image: full field at the start, the ray leaves at angle -psi
        f, fp = (lambda n, f=f: f(-n)), (lambda n, fp=fp: -fp(-n))
        breaks, (na, nb) = [-b for b in reversed(breaks)], (-nb, -na)
        theta0 = math.asin(-math.sin(psi) + h * full)    # d sin(theta)/dn = -h f  integrated over the region
        l_drift = (nb - (na + full)) / math.cos(psi)
    eps = 1e-7
    w0 = _trace_fringe(f, fp, breaks, (na, nb), h, theta0, 0.0, 0.0)
    wa = _trace_fringe(f, fp, breaks, (na, nb), h, theta0, eps, 0.0)
    wb = _trace_fringe(f, fp, breaks, (na, nb), h, theta0, 0.0, eps)
    assert w0[2] == 0.0 and w0[5] == 0.0                                        # the reference ray stays in the mid-plane
    M = np.array([[wa[2], wb[2]], [wa[5] / math.hypot(wa[3], wa[4]), wb[5] / math.hypot(wb[3], wb[4])]]) / eps
    theta1 = math.atan2(w0[4], w0[3])
    l_body = (theta0 - theta1) / h if face == "entrance" else (theta0 - (-psi)) / h   # arc of the hard-edge orbit in full field
    if face == "exit":
        assert abs(theta1 + psi) < 1e-9                                         # it does leave at -psi
    D = lambda L: np.array([[1.0, L], [0.0, 1.0]])
    E = D(-l_body) @ M @ D(-l_drift) if face == "entrance" else D(-l_drift) @ M @ D(-l_body)
    return E, K


def _oracle_r43(psi, rho, g, K):
    c = [np.zeros(1) for _ in range(6)]
    c[2][0] = 1e-3
    O.track(c, [("dipedge", 0.0, 1, psi, rho, g, K)], 1, GAMMA_E5GEV)
    return c[3][0] / 1e-3


@pytest.mark.parametrize("rho,g", [(10.0, 0.02), (10.0, 0.005), (2.5, 0.02), (-4.0, 0.01)])
@pytest.mark.parametrize("psi", [0.5, -0.4, 0.05, -0.05, 0.0])
@pytest.mark.parametrize("kind", ["ramp", "tanh"])
def test_dipedge_fringe_term_vs_maxwell_ray_tracing(rho, g, psi, kind):
    """R7's fringe term against the Lorentz force in an extended fringe field (see the comment block above): the
    vertical focusing of the oracle's thin edge must equal that of the ray-traced fringe region, once the drift and
    the bend body of the hard-edge model are divided out, to within 2 % of the fringe correction itself (the remainder
    is second order in g/rho: it measures 0.2 % at g/rho = 0.002 and 0.7 % at 0.008) -- for both signs of psi and of
    rho, configs[2]'s values (rho = 10, g = 0.02, K = 1/2, psi = +-0.05) included, two field profiles with different K.

    Mutants of oracle/bt_oracle.c:pass_dipedge that these pins kill (each was applied to a copy of the oracle and
    `pytest -k dipedge_fringe_term` run against it; `fail` = failing cases of 41 = 40 here + the remainder test below;
    the unmutated oracle passes all 41):
        (1 + sp*sp)  ->  (1 + cp*cp)                                                        fail 41
        (1 + sp*sp)  ->  1   (tan(theta(n)) averaged over the fringe, double-kick term lost) fail 17  (all with |psi| >= 0.4)
        "/ cp" dropped                                                                      fail 17  (all with |psi| >= 0.4)
        K  ->  2 K                                                                          fail 41
        g / rho  ->  g / (rho * rho)                                                        fail 41
        tan(psi - psi_c)  ->  tan(psi + psi_c)                                              fail 41
        tan(psi - psi_c)  ->  tan(psi) - psi_c                                              fail 17  (all with |psi| >= 0.4)
    """
    face = "entrance" if psi >= 0.0 or kind == "tanh" else "exit"              # both faces are exercised
    E, K = _edge_matrix_from_ray_tracing(kind, g, rho, psi, face)
    assert abs(K - (0.5 if kind == "ramp" else 0.35)) < 1e-9
    hard = -math.tan(psi) / rho
    got = _oracle_r43(psi, rho, g, K)
    corr = abs(got - hard)
    assert corr > 0.2 * K * g / rho ** 2                                        # there is a correction to compare
    assert abs(E[1, 0] - got) <= 0.02 * corr, (E[1, 0], got, hard)
    # the rest of the ray-traced edge is the identity to first order in g: a thin element at the effective edge
    assert abs(E[0, 0] - 1.0) < 1e-4 and abs(E[1, 1] - 1.0) < 1e-4
    assert abs(E[0, 1]) < 1e-4
    assert abs(np.linalg.det(E) - 1.0) < 1e-9


def test_dipedge_fringe_term_remainder_is_second_order():
    """Halving g quarters the distance between the ray-traced edge focusing and the oracle's first-order expression."""
    rho, psi = 2.5, 0.5
    d = []
    for g in (0.02, 0.01, 0.005):
        E, K = _edge_matrix_from_ray_tracing("ramp", g, rho, psi, "entrance")
        d.append(abs(E[1, 0] - _oracle_r43(psi, rho, g, K)))
    assert 3.5 < d[0] / d[1] < 4.5 and 3.5 < d[1] / d[2] < 4.5


# ------------------------------------------------------------------------------------------------
# chicane (config 2): paper invariant P5 + geometric path-length pin
# ------------------------------------------------------------------------------------------------
def test_chicane_dispersion_closed_P5():
    """'the initial emittance is recovered at the end of transport' <=> the chicane is
    achromatic: R16 = R26 = 0 (and by symplecticity R51 = R52 = 0); the x-plane is a pure drift."""
    M = M_of(W.chicane(), GAMMA_E5GEV)
    assert abs(M[0, 5]) < 1e-14 and abs(M[1, 5]) < 1e-15
    assert abs(M[4, 0]) < 1e-15 and abs(M[4, 1]) < 1e-14
    assert abs(M[0, 0] - 1) < 1e-14 and abs(M[1, 1] - 1) < 1e-14 and abs(M[1, 0]) < 1e-16
    Ld, Lm, rho, th = 5.0, 1.0, 10.0, 0.05
    R12 = 2 * Ld / math.cos(th) ** 2 + Lm + 4 * rho * math.tan(th)
    assert abs(M[0, 1] - R12) < 1e-13


def test_chicane_R56_exact_path_length():
    """t-row pin through the whole sbend+dipedge+drift chain: exact path length of a particle of momentum
    p through four rectangular magnets (projected length rho0 sin th0) with the outer drifts L_d along
    the inclined reference orbit, S(p) = 4 R phi + 2 L_d cos(th0)/cos(phi) + L_m, sin(phi) = rho0 sin(th0)/R;
    c*dt = S/beta - S0/beta0 differentiated w.r.t. pt."""
    Ld, Lm, rho0, th0 = mp.mpf(5), mp.mpf(1), mp.mpf(10), mp.mpf("0.05")
    m = mp.mpf(ME)
    E0 = mp.mpf(5000) + m
    p0 = mp.sqrt(E0**2 - m**2)
    S0 = 4 * rho0 * th0 + 2 * Ld + Lm

    def ct(pt):
        E = E0 - pt * p0
        p = mp.sqrt(E**2 - m**2)
        R = rho0 * p / p0
        phi = mp.asin(rho0 * mp.sin(th0) / R)
        S = 4 * R * phi + 2 * Ld * mp.cos(th0) / mp.cos(phi) + Lm
        return S / (p / E) - S0 / (p0 / E0)

    exact = float(mp.diff(ct, 0))
    M = M_of(W.chicane(), GAMMA_E5GEV)
    assert abs(M[4, 5] - exact) / exact < 1e-11
    assert abs(exact - 0.0267101968265) < 1e-12         # SURVEY 8(c) closed form, 5 GeV e-
    # bunch-length scaling for the config's chirp pt = -20 t:  |1 - 20 R56|
    assert abs(abs(1 - 20 * M[4, 5]) - 0.46580) < 1e-5


def test_chicane_compresses_config2_bunch():
    cfg = W.config(2, n=200_000)
    c = W.make_bunch(cfg)
    g = O.ref_from_kinetic(cfg.kin_energy_MeV, cfg.mass_MeV)[0]
    ex0, ey0, st0 = rms_emittance(c[0], c[1]), rms_emittance(c[2], c[3]), c[4].std()
    O.track(c, cfg.lattice, 1, g)
    assert abs(rms_emittance(c[0], c[1]) / ex0 - 1) < 1e-9     # emittance recovered (P5)
    assert abs(rms_emittance(c[2], c[3]) / ey0 - 1) < 1e-9
    assert abs(c[4].std() / st0 - 0.4658) < 2e-3              # compressed x2.147


# ------------------------------------------------------------------------------------------------
# R8 thin multipole
# ------------------------------------------------------------------------------------------------
def _kick(m, Kn, Ks, x, y):
    c = [np.array([x]), np.array([0.0]), np.array([y]), np.array([0.0]), np.array([0.3]), np.array([0.1])]
    O.track(c, [("multipole", 0.0, 1, m, Kn, Ks)], 1, GAMMA_P1GEV)
    assert c[0][0] == x and c[2][0] == y and c[4][0] == 0.3 and c[5][0] == 0.1
    return c[1][0], c[3][0]


def test_multipole_textbook_kicks():
    x, y = 1.3e-3, -0.7e-3
    K = 5.0
    dpx, dpy = _kick(3, K, 0.0, x, y)                       # sextupole: -(K/2)(x^2-y^2), +K x y
    assert abs(dpx + 0.5 * K * (x * x - y * y)) < 1e-20 and abs(dpy - K * x * y) < 1e-20
    K = 50.0
    dpx, dpy = _kick(4, K, 0.0, x, y)                       # octupole: -(K/6)(x^3-3xy^2), +(K/6)(3x^2y-y^3)
    assert abs(dpx + K / 6 * (x**3 - 3 * x * y * y)) < 1e-22 and abs(dpy - K / 6 * (3 * x * x * y - y**3)) < 1e-22
    dpx, dpy = _kick(1, 2e-3, 1e-3, x, y)                   # dipole kick
    assert dpx == -2e-3 and dpy == 1e-3
    dpx, dpy = _kick(2, 0.0, 0.4, x, y)                     # skew quad: +Ks y, +Ks x
    assert abs(dpx - 0.4 * y) < 1e-19 and abs(dpy - 0.4 * x) < 1e-19


@pytest.mark.parametrize("m", range(1, 11))
def test_multipole_general_order_vs_complex_power(m):
    x, y, Kn, Ks = 0.11, -0.07, 1.7, -0.9
    F = mp.mpc(Kn, Ks) * mp.mpc(x, y) ** (m - 1) / mp.factorial(m - 1)
    dpx, dpy = _kick(m, Kn, Ks, x, y)
    assert abs(dpx + float(F.real)) < 1e-15 * max(1.0, abs(F))
    assert abs(dpy - float(F.imag)) < 1e-15 * max(1.0, abs(F))


def test_multipole_m2_is_thin_quad_and_converges_to_thick():
    k, L = 1.0, 1.0
    thick = M_of([("quad", L, 1, k)], GAMMA_P2GEV)
    errs = []
    for n in (10, 100, 1000):
        h = L / n
        step = [("drift", h / 2, 1), ("multipole", 0.0, 1, 2, k * h, 0.0), ("drift", h / 2, 1)]
        M = M_of(step * n, GAMMA_P2GEV)
        errs.append(np.max(np.abs(M[:4, :4] - thick[:4, :4])))
    assert errs[0] < 5e-3 and errs[1] < errs[0] / 90 and errs[2] < errs[1] / 90     # O(n^-2)


def test_multipole_symplectic_jacobian():
    x, y, eps = 2e-3, 1e-3, 1e-7
    for m, Kn, Ks in ((3, 5.0, 1.0), (4, 50.0, -20.0)):
        def k(xx, yy):
            return _kick(m, Kn, Ks, xx, yy)
        dpx_dy = (k(x, y + eps)[0] - k(x, y - eps)[0]) / (2 * eps)
        dpy_dx = (k(x + eps, y)[1] - k(x - eps, y)[1]) / (2 * eps)
        assert abs(dpx_dy - dpy_dx) < 1e-9      # kick = gradient of a potential -> symplectic


# ------------------------------------------------------------------------------------------------
# R9 short RF
# ------------------------------------------------------------------------------------------------
def _rf_exact(t, px, pt, Vhat, freq, phase_deg, kin, mass):
    """Definition: E' = E + qV cos(k t + phi), reference E0' = E0 + qV cos(phi); transverse momenta
    Px unchanged, renormalised by the new p0; pt' = -(E'-E0')/(p0' c)."""
    m = mp.mpf(mass)
    E0 = mp.mpf(kin) + m
    p0 = mp.sqrt(E0**2 - m**2)
    qV = mp.mpf(Vhat) * m
    phi = mp.mpf(phase_deg) * mp.pi / 180
    k = 2 * mp.pi * mp.mpf(freq) / mp.mpf(W.C_LIGHT)
    E = E0 - pt * p0
    E1 = E + qV * mp.cos(k * t + phi)
    E01 = E0 + qV * mp.cos(phi)
    p01 = mp.sqrt(E01**2 - m**2)
    return px * p0 / p01, -(E1 - E01) / p01, E01 / m


@pytest.mark.parametrize("phase", [-30.0, -90.0, 25.0])
def test_shortrf_is_the_linearised_exact_energy_kick(phase):
    Vhat, freq, kin, mass = W.RING_RF_VHAT, W.RING_RF_FREQ_HZ, 1000.0, MP_
    g0 = O.ref_from_kinetic(kin, mass)[0]
    c = [np.zeros(7) for _ in range(6)]
    for j in range(6):
        c[j][j + 1] = 1.0
    g1, _ = O.track(c, [("shortrf", 0.0, 1, Vhat, freq, phase)], 1, g0)
    M = np.array([[c[i][j + 1] for j in range(6)] for i in range(6)])
    d_px = float(mp.diff(lambda e: _rf_exact(0, e, 0, Vhat, freq, phase, kin, mass)[0], 0))
    d_pt_pt = float(mp.diff(lambda e: _rf_exact(0, 0, e, Vhat, freq, phase, kin, mass)[1], 0))
    d_pt_t = float(mp.diff(lambda e: _rf_exact(e, 0, 0, Vhat, freq, phase, kin, mass)[1], 0))
    gamma_f = float(_rf_exact(0, 0, 0, Vhat, freq, phase, kin, mass)[2])
    assert abs(g1 - gamma_f) < 1e-15 * gamma_f
    assert abs(M[1, 1] - d_px) < 1e-14 and abs(M[3, 3] - d_px) < 1e-14
    assert abs(M[5, 5] - d_pt_pt) < 1e-14
    assert abs(M[5, 4] - d_pt_t) < 1e-14 * max(1.0, abs(d_pt_t) * 1e4)
    assert M[0, 0] == M[2, 2] == M[4, 4] == 1.0
    r = d_px
    assert np.max(np.abs(M.T @ J6 @ M - r * J6)) < 1e-15       # conformal-symplectic, factor (bg)_i/(bg)_f
    if phase == -90.0:
        assert abs(r - 1.0) < 1e-15 and abs(g1 - g0) < 1e-15


def test_shortrf_updates_reference_for_later_maps():
    """R9: after the cavity all later maps use the new beta0 gamma0 (here: the drift's t-row)."""
    Vhat = 0.5
    g0 = GAMMA_P1GEV
    lat = [("shortrf", 0.0, 1, Vhat, 1e6, 0.0), ("drift", 2.0, 1)]
    c = [np.zeros(1) for _ in range(6)]
    c[5][0] = 1e-3
    g1, _ = O.track(c, lat, 1, g0)
    assert abs(g1 - (g0 + Vhat)) < 1e-15
    bg0, bg1 = math.sqrt(g0 * g0 - 1), math.sqrt(g1 * g1 - 1)
    assert abs(c[4][0] - 2.0 / bg1**2 * (1e-3 * bg0 / bg1)) < 1e-18
    # config 3: gamma after 100 turns
    c = [np.zeros(1) for _ in range(6)]
    g100, s100 = O.track(c, W.nonlinear_ring(), 100, GAMMA_P1GEV)
    assert abs(g100 - (GAMMA_P1GEV + 100 * W.RING_RF_VHAT * math.cos(math.radians(-30.0)))) < 1e-13
    assert abs(s100 - 7500.0) < 1e-9


def test_shortrf_longitudinal_focusing_below_transition():
    """Buncher phase (-90 deg) in a straight channel: negative-mass-free (below transition) longitudinal
    motion is stable, |tr M_long| < 2, and unstable for +90 deg."""
    def tr(phase):
        lat = W.fodo_cell(1) + [("shortrf", 0.0, 1, 1e-3, 1e8, phase)]
        M = M_of(lat, GAMMA_P1GEV)
        return M[4, 4] + M[5, 5]
    assert abs(tr(-90.0)) < 2.0 < abs(tr(+90.0))


# ------------------------------------------------------------------------------------------------
# whole tracker: invariants the paper's benchmarks check (P3, P6)
# ------------------------------------------------------------------------------------------------
def test_P3_emittance_conserved_and_moments_periodic_fodo():
    cfg = W.config(1, n=100_000)
    cfg.lattice = W.fodo_cell(25) * 3
    c = W.make_bunch(cfg)
    g = O.ref_from_kinetic(cfg.kin_energy_MeV, cfg.mass_MeV)[0]
    e0 = [rms_emittance(c[0], c[1]), rms_emittance(c[2], c[3]), rms_emittance(c[4], c[5])]
    s0 = [c[0].std(), c[2].std(), c[1].std(), c[3].std()]
    O.track(c, cfg.lattice, 1, g)
    e1 = [rms_emittance(c[0], c[1]), rms_emittance(c[2], c[3]), rms_emittance(c[4], c[5])]
    s1 = [c[0].std(), c[2].std(), c[1].std(), c[3].std()]
    for a, b in zip(e0, e1):
        assert abs(a / b - 1) < 1e-10
    for a, b in zip(s0, s1):
        assert abs(a / b - 1) < 1e-2          # matched to sampling noise of 1e5 particles (P3: "remain matched")
    assert abs(e0[0] / 1e-6 - 1) < 1e-2


def test_P6_normalised_emittance_conserved_with_rf_linear_ring():
    cfg = W.config(3, n=50_000)
    lat = W.nonlinear_ring(rf=True, sext=0.0, octu=0.0)
    c = W.make_bunch(cfg)
    g0 = O.ref_from_kinetic(cfg.kin_energy_MeV, cfg.mass_MeV)[0]
    e0 = rms_emittance(c[0], c[1]) * math.sqrt(g0 * g0 - 1)
    g1, _ = O.track(c, lat, 5, g0)
    e1 = rms_emittance(c[0], c[1]) * math.sqrt(g1 * g1 - 1)
    assert g1 > g0 and abs(e1 / e0 - 1) < 1e-10


def test_config0_tracks_and_is_deterministic():
    cfg = W.config(0)
    a, b = W.make_bunch(cfg), W.make_bunch(cfg)
    g = O.ref_from_kinetic(cfg.kin_energy_MeV, cfg.mass_MeV)[0]
    O.set_num_threads(1)
    O.track(a, cfg.lattice, cfg.nturns, g)
    O.set_num_threads(4)
    O.track(b, cfg.lattice, cfg.nturns, g)
    for u, v in zip(a, b):
        assert np.array_equal(u, v) and np.all(np.isfinite(u))
    assert np.array_equal(a[5], W.make_bunch(cfg)[5])     # pt untouched by drifts and quads
