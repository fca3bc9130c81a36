"""Typo guard: the oracle against (a) a 40-digit mpmath restatement of readings R1-R9 and (b) the
worked examples W1-W3 printed in SURVEY.md 8(c).  Not a pin in the sense of the task statement (it
retypes the formulas at higher precision); it bounds the oracle's fp64 rounding error (R14 margin)."""
import os

import mpmath as mp
import numpy as np

import oracle as O
import workloads as W

mp.mp.dps = 40
HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "survey_worked_examples.txt")):
        line = line.split("#", 1)[0].strip()
        if line:
            k, v = line.split("=")
            out[k.strip()] = [float(s) for s in v.split()]
    return out


def mp_track(v, lattice, nturns, kin, mass):
    """R1-R9 restated in mpmath for ONE particle; input numbers are the fp64 values."""
    x, px, y, py, t, pt = [mp.mpf(a) for a in v]
    gamma = 1 + mp.mpf(kin) / mp.mpf(mass)
    for _ in range(nturns):
        for el in lattice:
            kind, ds, ns = el[0], mp.mpf(el[1]), el[2]
            par = [mp.mpf(p) for p in el[3:]]
            bg = mp.sqrt(gamma**2 - 1)
            beta = bg / gamma
            h = ds / ns
            for _s in range(ns):
                if kind == "drift" or (kind == "quad" and par[0] == 0):
                    x, y, t = x + h * px, y + h * py, t + h / bg**2 * pt
                elif kind == "quad":
                    w = mp.sqrt(abs(par[0]))
                    c, s, ch, sh = mp.cos(w * h), mp.sin(w * h), mp.cosh(w * h), mp.sinh(w * h)
                    f = lambda q, p: (c * q + s / w * p, -w * s * q + c * p)
                    d = lambda q, p: (ch * q + sh / w * p, w * sh * q + ch * p)
                    (x, px), (y, py) = (f(x, px), d(y, py)) if par[0] > 0 else (d(x, px), f(y, py))
                    t = t + h / bg**2 * pt
                elif kind == "sbend":
                    rho = par[0]
                    th = h / rho
                    C, S = mp.cos(th), mp.sin(th)
                    x, px, y, t = (C * x + rho * S * px - rho * (1 - C) / beta * pt,
                                   -S / rho * x + C * px - S / beta * pt,
                                   y + h * py,
                                   t + S / beta * x + rho * (1 - C) / beta * px + rho * (S / beta**2 - th) * pt)
                elif kind == "dipedge":
                    psi, rho, g, K = par
                    psi_c = K * g / rho * (1 + mp.sin(psi) ** 2) / mp.cos(psi)
                    px, py = px + mp.tan(psi) / rho * x, py - mp.tan(psi - psi_c) / rho * y
                elif kind == "multipole":
                    m = int(par[0])
                    F = mp.mpc(par[1], par[2]) * mp.mpc(x, y) ** (m - 1) / mp.factorial(m - 1)
                    px, py = px - F.real, py + F.imag
                elif kind == "shortrf":
                    Vh, f_, ph = par
                    phi = ph * mp.pi / 180
                    gf = gamma + Vh * mp.cos(phi)
                    bgf = mp.sqrt(gf**2 - 1)
                    r = bg / bgf
                    krf = 2 * mp.pi * f_ / mp.mpf(W.C_LIGHT)
                    px, py, pt = r * px, r * py, r * pt + Vh * krf * mp.sin(phi) / bgf * t
                    gamma = gf
    return [x, px, y, py, t, pt], gamma


V0 = (1e-3, 2e-4, -5e-4, 1e-4, 1e-3, 1e-3)


def orc(v, lattice, nturns, kin, mass):
    c = [np.array([a]) for a in v]
    g0 = O.ref_from_kinetic(kin, mass)[0]
    g, _ = O.track(c, lattice, nturns, g0)
    return [a[0] for a in c], g


def close(a, b, rel):
    scale = max(abs(float(x)) for x in b)
    return all(abs(float(x) - float(y)) <= rel * max(abs(float(y)), 1e-1 * scale) for x, y in zip(a, b))


def test_W1_config0():
    G = golden()
    lat = W.config(0).lattice
    for nt, key in ((1, "W1_turn1"), (10, "W1_turn10")):
        ref, _ = mp_track(V0, lat, nt, 2000.0, W.MASS_PROTON_MEV)
        got, _ = orc(V0, lat, nt, 2000.0, W.MASS_PROTON_MEV)
        assert close(got, ref, 1e-13)
        assert close(G[key], ref, 1e-15)


def test_W2_chicane():
    G = golden()
    ref, _ = mp_track(G["W2_in"], W.chicane(), 1, 5000.0, W.MASS_ELECTRON_MEV)
    got, _ = orc(G["W2_in"], W.chicane(), 1, 5000.0, W.MASS_ELECTRON_MEV)
    assert close(got, ref, 1e-13)
    assert close(G["W2_out"], ref, 1e-15)


def test_W3_ring_with_rf():
    G = golden()
    lat = W.nonlinear_ring()
    for nt, key, gk in ((1, "W3_turn1", "W3_gamma1"), (2, "W3_turn2", "W3_gamma2")):
        ref, gref = mp_track(V0, lat, nt, 1000.0, W.MASS_PROTON_MEV)
        got, g = orc(V0, lat, nt, 1000.0, W.MASS_PROTON_MEV)
        assert close(got, ref, 1e-13)
        assert abs(g - float(gref)) < 1e-15 * g
        assert close(G[key], ref, 1e-15)
        assert abs(G[gk][0] - float(gref)) < 1e-15 * g
