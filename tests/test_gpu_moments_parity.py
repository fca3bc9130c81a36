"""bt_beam_moments (CUDA, through the C-ABI) against the oracle's two-pass long-double definition.

Tolerance: the device sums fp64 products in a fixed tree; for N terms the error of a tree sum
is <= ~log2(N) eps sum|terms| and |d_i d_j| sums to at most N sqrt(c_ii c_jj)(1 + 1/4096), so
|cov - ref| <= 1e-12 sqrt(ref_ii ref_jj) and |mean - ref| <= 1e-12 sigma_i + 4 eps |ref| hold with two orders of margin."""
import numpy as np
import pytest

import oracle as O
import paper_2208_02382_b200 as bt
import workloads as W

pytestmark = pytest.mark.gpu


def check(c, beam=None):
    own = beam is None
    if own:
        beam = bt.Beam(c[0].shape[0])
        beam.upload(c)
    mean, cov = beam.moments()
    rm, rc = O.moments(c)
    sig = np.sqrt(np.diag(rc))
    assert np.all(np.abs(mean - rm) <= 1e-12 * sig + 4 * np.finfo(float).eps * np.abs(rm)), (mean - rm, sig)
    scale = np.outer(sig, sig)
    if np.all(scale > 0):
        assert np.max(np.abs(cov - rc) / scale) <= 1e-12, np.max(np.abs(cov - rc) / scale)
    else:
        assert np.max(np.abs(cov - rc)) <= 1e-12 * max(np.max(scale), 1e-300)
    assert np.array_equal(cov, cov.T)
    if own:
        beam.close()
    return mean, cov


@pytest.mark.parametrize("n", [1, 2, 3, 255, 4097, 100_003, 1_000_000, 64_000_000])
def test_moments_gaussian_sizes(n):
    cfg = W.config(0, n=n)
    check(W.make_bunch(cfg))


def test_moments_offset_and_correlated_bunch():
    """Centre 10^3 sigma away from the origin, strong x-px and t-pt correlations (the chicane's chirped bunch)."""
    cfg = W.config(2, n=300_001)
    c = W.make_bunch(cfg)
    c[0] += 1.0
    c[4] -= 3.0
    c[1] += 0.7 * c[0]
    check(c)


def test_moments_on_a_cell_sorted_offset_bunch_at_bench_size():
    """configs[4]'s 8e6-particle bunch, shifted by five sigma and cell-sorted: the first particles of the storage then all sit
    in one corner of the grid, so the provisional centre must come from a sample spread over the whole storage."""
    sc = W.spacecharge_config("A")
    c = W.make_spacecharge_bunch(sc)
    c[0] += 5e-3
    c[3] -= 2e-3
    beam = bt.Beam(sc.n)
    grid = bt.Grid(sc.shape, [l + (5e-3 if a == 0 else 0.0) for a, l in enumerate(sc.lo)], sc.d)
    beam.upload(c)
    beam.sort_by_cell(grid, sc.zscale)
    check(c, beam)
    beam.close()
    grid.close()


def test_moments_unaligned_storage_and_odd_count():
    import torch
    cfg = W.config(0, n=70_001)
    c = W.make_bunch(cfg)
    backing = [torch.empty(cfg.n + 1, dtype=torch.float64, device="cuda") for _ in range(6)]
    beam = bt.Beam(cfg.n, storage=[b[1:] for b in backing])
    beam.upload(c)
    check(c, beam)
    beam.close()


def test_moments_independent_of_storage_order_and_deterministic():
    sc = W.spacecharge_config("A", n=200_000, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    beam = bt.Beam(sc.n)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    beam.upload(c)
    m0, c0 = check(c, beam)
    m1, c1 = beam.moments()
    assert np.array_equal(m0, m1) and np.array_equal(c0, c1)          # bit-reproducible
    beam.sort_by_cell(grid, sc.zscale)
    check(c, beam)                                                     # same ensemble, other storage order
    beam.close()
    grid.close()


def test_moments_after_tracking_match_and_emittance_is_conserved():
    """second moments stay matched, emittances constant -- from the DEVICE statistics after bt_track."""
    cfg = W.config(1, n=200_000)
    c = W.make_bunch(cfg)
    beam = bt.Beam(cfg.n)
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
    beam.lattice_set(cfg.lattice[:5])            # one FODO cell of the channel
    beam.upload(c)
    _, cov0 = beam.moments()
    beam.track(1)
    _, cov1 = beam.moments()
    ref = [a.copy() for a in c]
    O.track(ref, cfg.lattice[:5], 1, O.ref_from_kinetic(cfg.kin_energy_MeV, cfg.mass_MeV)[0])
    _, rc = O.moments(ref)
    sig = np.sqrt(np.diag(rc))
    assert np.max(np.abs(cov1 - rc) / np.outer(sig, sig)) <= 1e-11    # R14 tracking differences enter here
    e0, e1 = O.rms_emittances(cov0), O.rms_emittances(cov1)
    for a, b in zip(e0, e1):
        assert abs(a - b) <= 1e-10 * a
    assert abs(cov1[0, 0] - cov0[0, 0]) <= 2e-2 * cov0[0, 0]          # matched beam: <xx> periodic up to sampling noise ~ sqrt(2/N)
    beam.close()


def test_moments_argument_errors():
    beam = bt.Beam(10)
    assert bt.lib.bt_beam_moments(beam._h, None, None) == bt.BT_ERR_INVALID
    assert bt.lib.bt_beam_moments(None, None, None) == bt.BT_ERR_INVALID
    beam.close()


def _slice_lattice(lat):
    """Every element cut into its slices as separate single-slice elements of length ds/nslice (the oracle then stops after
    every slice; h = ds/nslice is the same rounded division on both sides)."""
    out = []
    for el in lat:
        kind, ds, ns = el[0], el[1], el[2]
        out += [(kind, ds / ns, 1) + tuple(el[3:])] * ns
    return out


@pytest.mark.parametrize("idx,n,granularity,ppt,block", [
    (0, 20_000, "element", -1, -1), (0, 20_000, "slice", -1, -1), (3, 20_000, "element", -1, -1), (3, 70_001, "element", -1, -1),
    (1, 70_001, "slice", -1, -1),
    # the geometry large bunches get by default (eight particles per thread: n >= 524 288), forced here at a size the oracle
    # can follow boundary by boundary, with both block sizes and a ragged last block
    (3, 70_001, "element", 8, 128), (1, 70_001, "slice", 8, 128), (3, 70_001, "element", 8, 64), (0, 20_000, "slice", 8, 64),
    (3, 70_001, "element", 2, 128)])
def test_track_diagnostics_inside_the_walk(idx, n, granularity, ppt, block, knobs):
    """bt_track_diagnostics (statistics taken inside the fused walk): final state bit-identical to bt_track; every record
    equals the oracle's moments of the oracle's bunch at that boundary of the walk -- after every element or after every
    slice (config 0: FODO cell with 10-slice quads; config 3: ring with kicks and an RF cavity that moves the reference
    energy; config 1's cell with 25-slice quads; 70 001 particles = four particles per thread + a ragged last block); and
    the whole table costs O(1) launches."""
    cfg = W.config(idx, n=n)
    lat = {0: cfg.lattice, 1: cfg.lattice[:5], 3: cfg.lattice[:16] + cfg.lattice[-1:]}[idx]
    nturns = 2
    c = W.make_bunch(cfg)
    beam = bt.Beam(cfg.n)
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
    beam.lattice_set(lat)
    beam.upload(c)
    beam.track(nturns)
    plain, ref_state = beam.download(), beam.get_ref()
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
    beam.upload(c)
    steps = _slice_lattice(lat) if granularity == "slice" else lat
    n0 = bt.launch_count()
    knobs("track_ppt", ppt)
    knobs("track_block", block)
    mean, cov = beam.track_diagnostics(nturns, len(steps), granularity)
    if ppt > 0:
        assert beam.last_launch()["particles_per_thread"] == ppt and beam.last_launch()["block"] == block
    knobs("track_ppt", -1)
    knobs("track_block", -1)
    launches = bt.launch_count() - n0
    assert launches <= 1 + 2 * 2, launches             # centre + (walk, combine) per record table; RF lattices: one table per turn here
    got = beam.download()
    for a, b in zip(got, plain):
        assert np.array_equal(a, b)
    assert beam.get_ref() == ref_state
    ref = [a.copy() for a in c]
    g = O.ref_from_kinetic(cfg.kin_energy_MeV, cfg.mass_MeV)[0]
    for t in range(nturns):
        for e, el in enumerate(steps):
            g, _ = O.track(ref, [el], 1, g)
            rm, rc = O.moments(ref)
            sig = np.sqrt(np.diag(rc))
            assert np.max(np.abs(cov[t, e] - rc) / np.outer(sig, sig)) <= 1e-11, (t, e)
            assert np.all(np.abs(mean[t, e] - rm) <= 1e-11 * sig + 1e-15 * np.abs(rm)), (t, e)
    beam.close()


def test_track_diagnostics_many_boundaries_are_cut_into_launches():
    """More boundaries than one row buffer / one record table holds (config 1's channel, slice granularity: 10 600 rows per
    warp over 2 turns, 1000 records): the launches are cut, elements split between launches, and the records still line up."""
    cfg = W.config(1, n=20_000)
    c = W.make_bunch(cfg)
    beam = bt.Beam(cfg.n)
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
    beam.lattice_set(cfg.lattice)
    beam.upload(c)
    nb = cfg.slice_maps_per_turn
    mean, cov = beam.track_diagnostics(2, nb, "slice")
    got = beam.download()
    final = [a.copy() for a in c]
    O.track(final, cfg.lattice, 2, O.ref_from_kinetic(cfg.kin_energy_MeV, cfg.mass_MeV)[0])
    rm, rc = O.moments(final)
    sig = np.sqrt(np.diag(rc))
    assert np.max(np.abs(cov[1, nb - 1] - rc) / np.outer(sig, sig)) <= 1e-11          # the last record = the final bunch
    gm, gc = O.moments(got)
    assert np.max(np.abs(cov[1, nb - 1] - gc) / np.outer(sig, sig)) <= 1e-12
    # a matched beam in a periodic channel: the records at the cell ends repeat (P:l.112 "second moments remain matched")
    per_cell = nb // 100
    ends = cov[0, per_cell - 1::per_cell, 0, 0]
    assert ends.shape == (100,) and np.max(np.abs(ends / ends[0] - 1.0)) < 2e-2
    assert np.all(np.isfinite(cov)) and np.all(np.isfinite(mean))
    assert bt.lib.bt_track_diagnostics(beam._h, 1, 7, np.zeros(42).ctypes.data_as(bt._dp)) == bt.BT_ERR_INVALID
    # the output is sized by the library's own count; a buffer that is too small is refused before anything runs
    import ctypes
    need = ctypes.c_int64()
    assert bt.lib.bt_track_diagnostics_records(beam._h, 2, 1, ctypes.byref(need)) == bt.BT_OK and need.value == 2 * nb
    assert bt.lib.bt_track_diagnostics_records(beam._h, 3, 0, ctypes.byref(need)) == bt.BT_OK and need.value == 3 * len(cfg.lattice)
    before, turn = bt.launch_count(), beam.get_ref()[2]
    small = np.zeros((nb - 1, 42))
    assert bt.lib.bt_track_diagnostics_n(beam._h, 1, 1, small.ctypes.data_as(bt._dp), nb - 1) == bt.BT_ERR_INVALID
    assert b"records" in bt.lib.bt_last_error() and bt.launch_count() == before and beam.get_ref()[2] == turn
    with pytest.raises(ValueError):
        beam.track_diagnostics(1, nb - 1, "slice")
    # the buffers the walk keeps on the beam can be given back and come back on demand
    beam.release_scratch()
    m2, c2 = beam.track_diagnostics(1, granularity="element")
    assert m2.shape == (1, len(cfg.lattice), 6) and np.all(np.isfinite(c2))
    beam.close()


def test_moments_device_variant_is_bit_identical_and_asynchronous():
    """bt_beam_moments_device leaves the 42 numbers in device memory (no synchronisation): same bits as bt_beam_moments."""
    import torch
    cfg = W.config(1, n=300_001)
    c = W.make_bunch(cfg)
    beam = bt.Beam(cfg.n)
    beam.upload(c)
    mean, cov = beam.moments()
    out = torch.full((3, 42), float("nan"), dtype=torch.float64, device="cuda")
    for k in range(3):                       # three calls back to back on the stream, read once at the end
        beam.moments_device(out[k])
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    for k in range(3):
        assert np.array_equal(got[k, :6], mean) and np.array_equal(got[k, 6:].reshape(6, 6), cov)
    assert bt.lib.bt_beam_moments_device(beam._h, None) == bt.BT_ERR_INVALID
    beam.close()
