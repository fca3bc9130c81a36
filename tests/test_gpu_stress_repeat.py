"""Stand-in for compute-sanitizer, which is closed on this GPU pool (profiles/r02_summary.md): the kernels with hand-placed
barriers, mbarrier pipelines, double-buffered shared memory and warp-private scratch are run

  * on particle arrays that sit between guard bands (a sentinel bit pattern on both sides of every array, checked after
    every call): an out-of-bounds write of a chunk / tail / vector path shows up as a damaged band;
  * repeatedly from the same input: everything deterministic (walk, gather + kick, sort, statistics, diagnostics) must come
    out bit-identical on every repetition and in every kernel mode that shares the arithmetic; a race on a shared-memory
    stage, a missed barrier or a re-used buffer shows up as a difference.  The deposit (fp64 atomics: order not
    deterministic) must meet R15 against the oracle on every repetition.

Sizes span several chunks of every kernel plus a ragged tail.
"""
import numpy as np
import pytest

import oracle as O
import paper_2208_02382_b200 as bt
import workloads as W
from _gpu import r15_isolated

pytestmark = pytest.mark.gpu

SENTINEL = np.int64(0x7FF8DEADBEEF1234)  # a NaN payload no kernel would produce


def banded_storage(n, band, lead=0):
    """Six views of n doubles inside ONE allocation, `band` sentinel doubles before and after each (lead: extra doubles in
    front, to make the arrays 8- but not 16-byte aligned).  Returns (views, check) -- check() asserts the bands are intact."""
    import torch
    total = lead + 6 * n + 7 * band
    buf = torch.empty(total, dtype=torch.float64, device="cuda")
    buf.view(torch.int64).fill_(int(SENTINEL))
    views, off = [], lead + band
    mask = torch.ones(total, dtype=torch.bool, device="cuda")
    for _ in range(6):
        views.append(buf[off:off + n])
        mask[off:off + n] = False
        off += n + band
    for v in views:
        v.zero_()

    def check(where):
        torch.cuda.synchronize()
        bad = (buf.view(torch.int64)[mask] != int(SENTINEL)).nonzero()
        assert bad.numel() == 0, "%s wrote outside its arrays (%d guard words damaged)" % (where, bad.numel())
    return views, check


@pytest.mark.parametrize("n,lead", [(1, 0), (255, 0), (4097, 0), (4097, 1), (100_003, 0), (100_003, 1), (262_144, 0)])
def test_no_kernel_writes_outside_the_particle_arrays(n, lead, knobs):
    sc = W.spacecharge_config("A", n=n, shape=(24, 20, 16))
    c = W.make_spacecharge_bunch(sc)
    E = W.gaussian_bunch_field(sc)
    views, check = banded_storage(n, band=1024, lead=lead)
    aligned16 = all(v.data_ptr() % 16 == 0 for v in views)   # odd n or lead: every other array starts 8 bytes off
    beam = bt.Beam(n, storage=views)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    try:
        beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, sc.charge_qe)
        grid.set_field(*E)
        beam.upload(c)
        check("bt_beam_upload")
        # fused walk: every particles-per-thread variant, static and per-turn tables
        for lattice in (W.fodo_cell(7), W.nonlinear_ring()[:40] + [W.nonlinear_ring()[-1]]):
            beam.lattice_set(lattice)
            for ppt in (1, 2, 4):
                if ppt > 1 and not aligned16:
                    continue  # vector variants need 16-byte aligned arrays (rejected by the library otherwise)
                knobs("track_ppt", ppt)
                beam.track(2)
                check("bt_track ppt=%d" % ppt)
            knobs("track_ppt", -1)
        beam.upload(c)
        beam.lattice_set(W.fodo_cell(3))
        beam.track_diagnostics(1, 5, "element")
        check("bt_track_diagnostics(element)")
        beam.track_diagnostics(1, 9, "slice")
        check("bt_track_diagnostics(slice)")
        beam.moments()
        check("bt_beam_moments")
        beam.upload(c)
        for order in (1, 2):
            grid.set_particle_shape(order)
            for mode in (0, 1, 2, 3):
                knobs("deposit_mode", mode)
                beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
                check("bt_deposit_cic order %d mode %d" % (order, mode))
            knobs("deposit_mode", -1)
            for mode in (0, 1, 2, 3, 4, 5):
                knobs("gather_mode", mode)
                beam.gather_kick(grid, sc.kick_coef, sc.zscale, sc.ds / 2, sc.ds / 2)
                check("bt_gather_kick order %d mode %d" % (order, mode))
                beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, 0.0)
                check("bt_gather_kick (kick only) order %d mode %d" % (order, mode))
            knobs("gather_mode", -1)
        grid.set_particle_shape(1)
        # the sort moves the bunch into the library's partner arrays and back; the lent arrays' bands must survive both
        for _ in range(3):
            beam.sort_by_cell(grid, sc.zscale)
            beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
            beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, sc.ds)
            check("sort + deposit + gather on sorted storage")
        got = beam.download()
        check("bt_beam_download")
        assert all(np.isfinite(g).all() for g in got)
    finally:
        beam.close()
        grid.close()


@pytest.mark.parametrize("variant,order", [("A", 1), ("B", 1), ("A", 2)])
def test_gather_sort_and_deposit_repeat_identically(variant, order, knobs):
    n = 200_003
    sc = W.spacecharge_config(variant, n=n, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    E = W.gaussian_bunch_field(sc)
    beam = bt.Beam(n)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    try:
        beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, sc.charge_qe)
        grid.set_particle_shape(order)
        grid.set_field(*E)
        ref_rho, _ = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight, sc.zscale, order=order)
        first = None
        for sorted_storage in (False, True):
            for mode in (0, 1, 2, 3, 4, 5):
                knobs("gather_mode", mode)
                for rep in range(4):
                    beam.upload(c)
                    if sorted_storage:
                        beam.sort_by_cell(grid, sc.zscale)
                    beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
                    assert r15_isolated(grid.download_rho(), ref_rho) <= 1e-12, (sorted_storage, mode, rep)
                    beam.gather_kick(grid, sc.kick_coef, sc.zscale, sc.ds / 2, sc.ds / 2)
                    got = beam.download()          # caller's order, whatever the storage order
                    if first is None:
                        first = got
                    else:                          # same arithmetic in every mode and storage order: bit-identical
                        for a, b in zip(got, first):
                            assert np.array_equal(a, b), (sorted_storage, mode, rep)
            knobs("gather_mode", -1)
    finally:
        beam.close()
        grid.close()


def test_resorting_a_wandering_beam_keeps_every_particle(knobs):
    """20 steps with a re-sort every 3 deposits (ping-pong storage, id permutation): the caller's-order download must be
    bit-identical to the same steps on a beam that is never sorted."""
    n = 150_001
    sc = W.spacecharge_config("A", n=n, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    E = W.gaussian_bunch_field(sc)
    outs = []
    for interval in (0, 3):
        beam = bt.Beam(n)
        grid = bt.Grid(sc.shape, sc.lo, sc.d)
        try:
            beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, sc.charge_qe)
            grid.set_field(*E)
            beam.upload(c)
            beam.set_resort_interval(interval)
            for _ in range(20):
                beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
                beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, 40 * sc.ds)   # large steps: particles change cell
            outs.append(beam.download())
            rho = grid.download_rho()
        finally:
            beam.close()
            grid.close()
    for a, b in zip(*outs):
        assert np.array_equal(a, b)
    assert np.isfinite(rho).all()


def test_walk_statistics_and_diagnostics_repeat_identically(knobs):
    cfg = W.config(3, n=70_001)
    c = W.make_bunch(cfg)
    lattice = cfg.lattice
    ref = None
    for rep in range(3):
        for ppt in (1, 2, 4):
            knobs("track_ppt", ppt)
            beam = bt.Beam(cfg.n)
            try:
                beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
                beam.lattice_set(lattice)
                beam.upload(c)
                beam.track(3)
                got = beam.download()
                mom = beam.moments()
                beam.upload(c)
                beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
                dm, dc = beam.track_diagnostics(1, len(lattice), "element")
                after_diag = beam.download()
            finally:
                beam.close()
            if ref is None:
                ref = (got, mom)
                ref_diag = {}
            for a, b in zip(got, ref[0]):          # the walk's arithmetic does not depend on particles per thread
                assert np.array_equal(a, b), (rep, ppt)
            assert np.array_equal(mom[0], ref[1][0]) and np.array_equal(mom[1], ref[1][1]), (rep, ppt)
            if ppt not in ref_diag:                # rows are per warp: the reduction order depends on ppt, not on the run
                ref_diag[ppt] = (dm, dc, after_diag)
            assert np.array_equal(dm, ref_diag[ppt][0]) and np.array_equal(dc, ref_diag[ppt][1]), (rep, ppt)
            for a, b in zip(after_diag, ref_diag[ppt][2]):
                assert np.array_equal(a, b), (rep, ppt)
    knobs("track_ppt", -1)
