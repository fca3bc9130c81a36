"""Order-2 particle shape (bt_grid_set_particle_shape(2): quadratic B-spline, reading R16) through the C-ABI against the
oracle.  Same bars as order 1: deposit R15 (isolated: every non-zero node within relative 1e-12, identical zero set; total
charge 1e-13), gather/kick R14 1e-11."""
import math

import numpy as np
import pytest

import oracle as O
import paper_2208_02382_b200 as bt
import workloads as W
from _gpu import r15_isolated
from _util import r14_error

pytestmark = pytest.mark.gpu


def run_deposit(c, sc, zscale=None, sort=False, storage=None, twice=False):
    beam = bt.Beam(c[0].shape[0], storage=storage)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    try:
        grid.set_particle_shape(2)
        beam.upload(c)
        zs = sc.zscale if zscale is None else zscale
        if sort:
            beam.sort_by_cell(grid, zs)
        beam.deposit_cic(grid, sc.q_weight, zs, zero_first=True)
        if twice:
            beam.deposit_cic(grid, sc.q_weight, zs, zero_first=False)
        return grid.download_rho()
    finally:
        beam.close()
        grid.close()


@pytest.mark.parametrize("mode", [0, 1, 3])
@pytest.mark.parametrize("variant", ["A", "B"])
@pytest.mark.parametrize("n,shape,sort", [(1, (8, 8, 8), False), (257, (16, 12, 10), False), (200_003, (32, 32, 32), False),
                                          (200_003, (32, 32, 32), True), (300_000, (128, 128, 128), True)])
def test_deposit_order2(mode, variant, n, shape, sort, knobs):
    knobs("deposit_mode", mode)
    sc = W.spacecharge_config(variant, n=n, shape=shape)
    c = W.make_spacecharge_bunch(sc)
    rho = run_deposit(c, sc, sort=sort)
    ref, n_in = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight, order=2)
    assert r15_isolated(rho, ref) <= 1e-12
    total = math.fsum(rho.ravel())
    assert abs(total - sc.q_weight * n_in) <= 1e-13 * sc.q_weight * max(n_in, 1)


def test_deposit_order2_boundaries_zscale_unaligned_accumulate():
    import torch
    sc = W.spacecharge_config("A", n=5001, shape=(16, 16, 16))
    c = W.make_spacecharge_bunch(sc)
    lo, d = sc.lo[0], sc.d[0]
    c[0][:9] = [lo + 0.5 * d, lo + 14.5 * d, np.nextafter(lo + 0.5 * d, -1), lo + 14.5 * d - 1e-12, np.nan, np.inf, -np.inf, lo, 0.5]
    c[2][9:13] = [lo, lo + 15 * d, np.nan, 7.0]
    backing = [torch.empty(sc.n + 1, dtype=torch.float64, device="cuda") for _ in range(6)]
    for zs in (1.0, -1.8, 0.25):
        rho = run_deposit(c, sc, zscale=zs, storage=[b[1:] for b in backing])
        ref, n_in = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight, zs, order=2)
        assert 0 < n_in < sc.n
        assert r15_isolated(rho, ref) <= 1e-12
    twice = run_deposit(c, sc, twice=True)
    ref1, _ = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight, order=2)
    ref2, _ = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight, rho=ref1.copy(), order=2)
    assert r15_isolated(twice, ref2) <= 1e-12


@pytest.mark.parametrize("mode", [0, 1, 2, 3, 4, 5])
@pytest.mark.parametrize("offset", [0, 1])
def test_gather_order2(mode, offset, knobs):
    import torch
    knobs("gather_mode", mode)
    sc = W.spacecharge_config("A", n=70_001, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    c[0][:5] = [1.0, np.nan, -1.0, 5.9e-3, -5.9e-3]
    E = W.gaussian_bunch_field(sc)
    backing = [torch.empty(sc.n + 2, dtype=torch.float64, device="cuda") for _ in range(6)]
    beam = bt.Beam(sc.n, storage=[b[offset:offset + sc.n] for b in backing])
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    grid.set_particle_shape(2)
    beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, 1.0)
    grid.set_field(*E)
    beam.upload(c)
    beam.sort_by_cell(grid, sc.zscale)
    beam.gather_kick(grid, sc.kick_coef, sc.zscale, sc.ds / 2, sc.ds)
    beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, 0.0)
    got = beam.download()
    g0 = O.ref_from_kinetic(sc.kin_energy_MeV, sc.mass_MeV)[0]
    ref = [a.copy() for a in c]
    O.track(ref, [("drift", sc.ds / 2, 1)], 1, g0)
    O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale, order=2)
    O.track(ref, [("drift", sc.ds, 1)], 1, g0)
    O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale, order=2)
    ok = np.isfinite(ref[0])
    assert max(r14_error([a[ok] for a in got], [a[ok] for a in ref])) <= 1e-11
    # and order 2 really is a different interpolant from order 1
    ref1 = [a.copy() for a in c]
    O.gather_kick(ref1, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale, order=1)
    ref2 = [a.copy() for a in c]
    O.gather_kick(ref2, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale, order=2)
    assert np.nanmax(np.abs(ref1[1] - ref2[1])) > 1e-9 * np.nanmax(np.abs(ref2[1] - c[1]))
    beam.close()
    grid.close()


def test_spacecharge_steps_order2_in_run():
    """Three deposit + gather/kick/drift steps with the order-2 shape on sorted storage against the oracle's loop."""
    sc = W.spacecharge_config("A", n=150_000, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    E = W.gaussian_bunch_field(sc)
    g0 = O.ref_from_kinetic(sc.kin_energy_MeV, sc.mass_MeV)[0]
    beam = bt.Beam(sc.n)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    grid.set_particle_shape(2)
    beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, 1.0)
    grid.set_field(*E)
    beam.upload(c)
    beam.sort_by_cell(grid, sc.zscale)
    ref = [a.copy() for a in c]
    for step in range(3):
        beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
        rho = grid.download_rho()
        rref, n_in = O.deposit_cic(ref[0], ref[2], ref[4], sc.shape, sc.lo, sc.d, sc.q_weight, sc.zscale, order=2)
        assert np.max(np.abs(rho - rref) / np.maximum(rref, sc.q_weight)) <= 1e-12          # R15 in-run
        beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, sc.ds)
        O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale, order=2)
        O.track(ref, [("drift", sc.ds, 1)], 1, g0)
    got = beam.download()
    assert max(r14_error(got, ref)) <= 1e-11
    beam.close()
    grid.close()


def test_shape_argument_errors():
    grid = bt.Grid((8, 8, 8), (0, 0, 0), (1, 1, 1))
    assert bt.lib.bt_grid_set_particle_shape(grid._h, 3) == bt.BT_ERR_UNSUPPORTED
    assert bt.lib.bt_grid_set_particle_shape(grid._h, 0) == bt.BT_ERR_UNSUPPORTED
    assert bt.lib.bt_grid_set_particle_shape(None, 2) == bt.BT_ERR_INVALID
    grid.close()
    small = bt.Grid((2, 8, 8), (0, 0, 0), (1, 1, 1))
    assert bt.lib.bt_grid_set_particle_shape(small._h, 2) == bt.BT_ERR_INVALID
    small.close()


@pytest.mark.parametrize("order", [1, 2])
@pytest.mark.parametrize("n", [1, 255, 256, 257, 513])
def test_gather_small_counts_around_the_chunk_size(order, n, knobs):
    """Pipeline chunks are 256 particles: counts below, at and just above one chunk (ragged tail kernel), tile mode forced."""
    knobs("gather_mode", 4)
    sc = W.spacecharge_config("A", n=n, shape=(16, 16, 16))
    c = W.make_spacecharge_bunch(sc)
    E = W.gaussian_bunch_field(sc)
    beam = bt.Beam(n)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    grid.set_particle_shape(order)
    beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, 1.0)
    grid.set_field(*E)
    beam.upload(c)
    beam.sort_by_cell(grid, sc.zscale)
    beam.gather_kick(grid, sc.kick_coef, sc.zscale, sc.ds / 2, sc.ds / 2)
    got = beam.download()
    g0 = O.ref_from_kinetic(sc.kin_energy_MeV, sc.mass_MeV)[0]
    ref = [a.copy() for a in c]
    O.track(ref, [("drift", sc.ds / 2, 1)], 1, g0)
    O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale, order=order)
    O.track(ref, [("drift", sc.ds / 2, 1)], 1, g0)
    assert max(r14_error(got, ref)) <= 1e-11
    beam.close()
    grid.close()


def test_everything_outside_the_grid_is_a_no_op():
    sc = W.spacecharge_config("A", n=3000, shape=(8, 8, 8))
    c = W.make_spacecharge_bunch(sc)
    c[0] += 1.0                                     # the whole bunch is a metre away from the grid
    E = W.gaussian_bunch_field(sc)
    for order in (1, 2):
        beam = bt.Beam(sc.n)
        grid = bt.Grid(sc.shape, sc.lo, sc.d)
        grid.set_particle_shape(order)
        beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, 1.0)
        grid.set_field(*E)
        beam.upload(c)
        beam.sort_by_cell(grid, sc.zscale)
        beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
        assert not grid.download_rho().any()
        beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, 0.0)
        got = beam.download()
        for a, b in zip(got, c):
            assert np.array_equal(a, b)
        beam.close()
        grid.close()
