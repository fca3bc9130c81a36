"""Measured parity margins at the full BASELINE sizes (not a test: the tests assert the bars, this prints how far inside
them the CUDA path is; the numbers go into BASELINE.md section 4 and profiles/).

    python tests/parity_report.py            # on a GPU box; about two minutes

R14: max over particles and coordinates of |gpu - oracle| / max(|oracle|, rms(oracle)); bar 1e-11.
R15 (i): max relative error over the non-zero nodes of an isolated deposit (identical zero sets asserted); bar 1e-12.
"""
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)

import oracle as O  # noqa: E402
import paper_2208_02382_b200 as bt  # noqa: E402
import workloads as W  # noqa: E402
from _gpu import gpu_track, oracle_track, r15_isolated  # noqa: E402
from _util import r14_error  # noqa: E402


def main():
    for idx in (0, 1, 2, 3):
        cfg = W.config(idx)
        c = W.make_bunch(cfg)
        got, _ref, _l = gpu_track(cfg, c)
        stride = 64 if idx == 3 else 1          # configs[3]: the oracle tracks the subset i % 64 == 0
        sub = [a[::stride].copy() for a in c]
        del c
        ref, _ = oracle_track(cfg, sub)
        err = max(r14_error([a[::stride] for a in got], ref))
        print("configs[%d] %-14s %9d particles (oracle on every %d-th): R14 max %.2e  (bar 1e-11)" % (idx, cfg.name, cfg.n, stride, err), flush=True)
    for variant in ("A", "B"):
        sc = W.spacecharge_config(variant)
        c = W.make_spacecharge_bunch(sc)
        E = W.gaussian_bunch_field(sc)
        beam, grid = bt.Beam(sc.n), bt.Grid(sc.shape, sc.lo, sc.d)
        beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, sc.charge_qe)
        grid.set_field(*E)
        beam.upload(c)
        beam.sort_by_cell(grid, sc.zscale)
        beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
        rho = grid.download_rho()
        rho_ref, _n = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight, sc.zscale)
        e15 = r15_isolated(rho, rho_ref)
        beam.gather_kick(grid, sc.kick_coef, sc.zscale, sc.ds / 2, sc.ds / 2)
        got = beam.download()
        ref = [a.copy() for a in c]
        g0 = O.ref_from_kinetic(sc.kin_energy_MeV, sc.mass_MeV)[0]
        O.track(ref, [("drift", sc.ds / 2, 1)], 1, g0)
        O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale)
        O.track(ref, [("drift", sc.ds / 2, 1)], 1, g0)
        e14 = max(r14_error(got, ref))
        print("configs[4] %s  %d particles, %dx%dx%d nodes: deposit R15(i) max %.2e (bar 1e-12); half drift + gather + kick + half drift "
              "R14 max %.2e (bar 1e-11)" % ((variant, sc.n) + tuple(sc.shape) + (e15, e14)), flush=True)
        beam.close()
        grid.close()


if __name__ == "__main__":
    main()
