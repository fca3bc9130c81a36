"""GPU-side helpers for the parity tests: everything goes through the C-ABI binding."""
import numpy as np

import oracle as O
import paper_2208_02382_b200 as bt


def gpu_track(cfg, coords, nturns=None, lattice=None, storage=None):
    """Upload coords, set reference + lattice, bt_track, download.  Returns (coords_out, (gamma, s, turn), launch)."""
    n = coords[0].shape[0]
    beam = bt.Beam(n, storage=storage)
    try:
        beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
        beam.lattice_set(cfg.lattice if lattice is None else lattice)
        beam.upload(coords)
        beam.track(cfg.nturns if nturns is None else nturns)
        out = beam.download()
        return out, beam.get_ref(), beam.last_launch()
    finally:
        beam.close()


def oracle_track(cfg, coords, nturns=None, lattice=None):
    c = [a.copy() for a in coords]
    g0 = O.ref_from_kinetic(cfg.kin_energy_MeV, cfg.mass_MeV)[0]
    g, s = O.track(c, cfg.lattice if lattice is None else lattice, cfg.nturns if nturns is None else nturns, g0)
    return c, (g, s)


def r15_isolated(rho_gpu, rho_ref):
    """strict relative error on every non-zero node + identical zero set."""
    assert np.array_equal(rho_gpu == 0.0, rho_ref == 0.0), "zero-node sets differ"
    nzm = rho_ref != 0.0
    if not nzm.any():
        return 0.0
    return float(np.max(np.abs(rho_gpu[nzm] - rho_ref[nzm]) / np.abs(rho_ref[nzm])))
