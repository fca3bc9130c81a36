"""Pins for the oracle's beam statistics (oracle.moments / oracle.rms_emittances; "beam statistics",
l.112 "beam second moments ... emittances").  Each pin is independent of the oracle's own code: exact rational
arithmetic, closed forms, the covariance law of affine maps, the paper's printed matched-beam numbers, and the
emittance invariant of a symplectic transport."""
from fractions import Fraction

import numpy as np

import oracle as O
import workloads as W
from _util import paper_values


def _rand_dyadic(rng, n, scale_bits=20):
    """Random values k / 2^scale_bits: exactly representable, so rational arithmetic sees the same numbers."""
    return rng.integers(-(1 << 24), 1 << 24, size=n).astype(np.float64) / float(1 << scale_bits)


def test_moments_exact_rational_brute_force():
    """Definition evaluated in exact rational arithmetic on a tiny ensemble; every one of the 6 + 36 outputs."""
    rng = np.random.default_rng(11)
    n = 9
    c = [_rand_dyadic(rng, n) for _ in range(6)]
    c[4] = c[4] + 4096.0                      # a coordinate with a large offset (exact in fp64)
    mean, cov = O.moments(c)
    fr = [[Fraction(float(v)) for v in a] for a in c]
    for i in range(6):
        mi = sum(fr[i]) / n
        assert abs(Fraction(float(mean[i])) - mi) <= abs(mi) * Fraction(1, 2**51)
        for j in range(6):
            mj = sum(fr[j]) / n
            cij = sum((a - mi) * (b - mj) for a, b in zip(fr[i], fr[j])) / n
            scale = max(abs(cij), Fraction(1, 10**30))
            assert abs(Fraction(float(cov[i, j])) - cij) <= scale * Fraction(1, 2**50), (i, j)


def test_moments_closed_form_integer_lattice():
    """x = 0..m-1: mean (m-1)/2, variance (m^2-1)/12; px = 3 - 2x: <x px> = -2 var, <px px> = 4 var; y = const."""
    m = 1001
    x = np.arange(m, dtype=np.float64)
    c = [x, 3.0 - 2.0 * x, np.full(m, 7.5), np.zeros(m), x * x, np.ones(m)]
    mean, cov = O.moments(c)
    var = (m * m - 1) / 12.0
    assert mean[0] == (m - 1) / 2.0 and mean[1] == 3.0 - (m - 1) and mean[2] == 7.5 and mean[5] == 1.0
    assert abs(cov[0, 0] - var) <= 1e-15 * var
    assert abs(cov[0, 1] + 2.0 * var) <= 1e-15 * 2 * var and cov[1, 0] == cov[0, 1]
    assert abs(cov[1, 1] - 4.0 * var) <= 1e-15 * 4 * var
    assert np.all(cov[2, :] == 0.0) and np.all(cov[:, 3] == 0.0) and np.all(cov[5, :] == 0.0)
    # <x, x^2> for the integer lattice: (m-1)(m^2-1)/12
    assert abs(cov[0, 4] - (m - 1) * (m * m - 1) / 12.0) <= 1e-14 * (m - 1) * (m * m - 1) / 12.0
    # variance of k^2, k = 0..m-1: sum k^4/m - (sum k^2/m)^2, in exact integers
    s2 = sum(k * k for k in range(m))
    s4 = sum(k ** 4 for k in range(m))
    v4 = Fraction(s4, m) - Fraction(s2, m) ** 2
    assert abs(Fraction(float(cov[4, 4])) - v4) <= v4 * Fraction(1, 2**50)


def test_moments_affine_covariance_law():
    """q' = A q + b  =>  mean' = A mean + b, cov' = A cov A^T, with a non-symmetric A (a transposed operand or a
    swapped index in the oracle breaks this)."""
    rng = np.random.default_rng(5)
    n = 4000
    q = rng.standard_normal((6, n)) * np.array([1e-3, 2e-3, 5e-4, 1e-3, 3e-3, 1e-4])[:, None]
    A = rng.standard_normal((6, 6))
    b = rng.standard_normal(6) * 1e-2
    qp = A @ q + b[:, None]
    m0, c0 = O.moments([np.ascontiguousarray(r) for r in q])
    m1, c1 = O.moments([np.ascontiguousarray(r) for r in qp])
    assert np.allclose(m1, A @ m0 + b, rtol=0, atol=1e-15)
    ref = A @ c0 @ A.T
    assert np.max(np.abs(c1 - ref)) <= 1e-12 * np.max(np.abs(ref))
    assert np.array_equal(c1, c1.T)


def test_moments_translation_invariance_large_offset():
    """Second moments about the mean do not see a common offset of 10^6 sigma (a one-pass sum-of-squares would)."""
    rng = np.random.default_rng(6)
    n = 20000
    c = [rng.standard_normal(n) * 1e-3 for _ in range(6)]
    _, cov0 = O.moments(c)
    shifted = [a + 1024.0 for a in c]                # ~10^6 sigma; the addition rounds each value to 2^-43 ~ 1e-13
    _, cov1 = O.moments(shifted)
    d = np.sqrt(np.diag(cov0))
    assert np.max(np.abs(cov1 - cov0) / np.outer(d, d)) <= 1e-8


def test_emittance_of_the_papers_matched_beam():
    """PAPER.md l.72-80 prints sigmaX, sigmaPx, muxpx of the FODO listing and l.66/l.112 its 'unnormalized rms emittance
    of 2 nm'.  With the sigmas read as phase-ellipse intercepts, an ensemble with second moments
    <xx> = sX^2/(1-mu^2), <pp> = sP^2/(1-mu^2), <xp> = mu sX sP/(1-mu^2) must have emittance 2.000000e-9 m."""
    pv = paper_values()
    sx, sp, mu = pv["listing_sigmaX"], pv["listing_sigmaPx"], pv["listing_muxpx"]
    f = 1.0 / (1.0 - mu * mu)
    target = np.array([[sx * sx * f, mu * sx * sp * f], [mu * sx * sp * f, sp * sp * f]])
    # deterministic ensemble with EXACTLY this covariance: 4 points +-L e1, +-L e2 of a Cholesky factor, scaled by sqrt(2)
    L = np.linalg.cholesky(target)
    pts = np.sqrt(2.0) * np.concatenate([L.T, -L.T])          # rows: points (x, px); mean 0, cov = L L^T
    z = np.zeros(4)
    c = [np.ascontiguousarray(pts[:, 0]), np.ascontiguousarray(pts[:, 1]), z.copy(), z.copy(), z.copy(), z.copy()]
    mean, cov = O.moments(c)
    assert np.max(np.abs(mean)) <= 1e-20
    assert np.max(np.abs(cov[:2, :2] - target) / np.abs(target)) <= 1e-14
    ex, ey, et = O.rms_emittances(cov)
    assert abs(ex - pv["fodo_emittance_m"]) <= 1e-9 * pv["fodo_emittance_m"]      # the paper's 2 nm
    assert ey == 0.0 and et == 0.0
    # Twiss from the moments: beta = <xx>/eps, alpha = -<xp>/eps  (the cell's periodic values)
    assert abs(cov[0, 0] / ex - 2.8216194100) <= 1e-8 and abs(-cov[0, 1] / ex - 1.59050035) <= 1e-8


def test_emittance_conserved_by_symplectic_transport():
    """'emittances remain constant' through the FODO cell -- the three rms emittances from the
    oracle's moments are invariants of the (uncoupled, linear) transport, to rounding."""
    cfg = W.config(0, n=5000)
    c = W.make_bunch(cfg)
    _, cov0 = O.moments(c)
    e0 = O.rms_emittances(cov0)
    O.track(c, cfg.lattice, 3, O.ref_from_kinetic(cfg.kin_energy_MeV, cfg.mass_MeV)[0])
    _, cov1 = O.moments(c)
    e1 = O.rms_emittances(cov1)
    for a, b in zip(e0, e1):
        assert abs(a - b) <= 1e-11 * a
    # and the moments themselves transform with the cell matrix: second moments are NOT constant for an unmatched beam
    assert abs(cov1[0, 0] - cov0[0, 0]) > 1e-3 * cov0[0, 0]


def test_moments_match_numpy_cov_on_random_data():
    rng = np.random.default_rng(8)
    c = [rng.standard_normal(3001) * s for s in (1e-3, 1e-3, 2e-3, 5e-4, 1e-2, 1e-4)]
    mean, cov = O.moments(c)
    ref = np.cov(np.stack(c), bias=True)
    assert np.allclose(mean, [a.mean() for a in c], rtol=0, atol=1e-18)
    d = np.sqrt(np.diag(ref))
    assert np.max(np.abs(cov - ref) / np.outer(d, d)) <= 1e-13
