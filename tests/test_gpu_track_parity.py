"""Parity of the fused lattice walk (bt_track, through the C-ABI) against the CPU oracle.

Bar (BASELINE.json north_star, made well-posed by reading R14): for every coordinate c and particle i
    |gpu - oracle| <= 1e-11 * max(|oracle_ci|, rms_c(oracle))        after the full run.
"""
import numpy as np
import pytest

import workloads as W
from _gpu import gpu_track, oracle_track
from _util import r14_error

pytestmark = pytest.mark.gpu
TOL = 1e-11


def check(got, ref, tol=TOL):
    errs = r14_error(got, ref)
    assert max(errs) <= tol, dict(zip(W.COORD_NAMES, errs))
    for g in got:
        assert np.all(np.isfinite(g))
    return errs


def test_config0_tiny_fodo_full():
    cfg = W.config(0)
    c = W.make_bunch(cfg)
    got, (g, s, turn), launch = gpu_track(cfg, c)
    ref, (g_ref, s_ref) = oracle_track(cfg, c)
    check(got, ref)
    assert g == g_ref and abs(s - s_ref) < 1e-9 and turn == 10
    assert np.array_equal(got[5], c[5])            # pt untouched by drifts and quads: bit exact


# sizes: several 512-particle tiles (P=4 x 128 threads) plus a ragged tail, and sub-warp sizes
@pytest.mark.parametrize("n", [1, 31, 33, 513, 4 * 128 * 5 + 77, 50_001])
def test_config1_fodo_channel_reduced(n):
    cfg = W.config(1, n=n)
    c = W.make_bunch(cfg)
    got, _, launch = gpu_track(cfg, c)
    ref, _ = oracle_track(cfg, c)
    check(got, ref)


@pytest.mark.parametrize("ppt,block", [(1, 32), (1, 128), (2, 64), (2, 128), (4, 128), (4, 96), (4, 32), (4, 64)])
def test_all_kernel_variants_agree(ppt, block, knobs):
    """Every (particles-per-thread, block size) instantiation against the oracle, config-3 ring (all op kinds except
    sbend/edge; 7 turns of per-turn tables = 2 launches) and the chicane."""
    knobs("track_ppt", ppt)
    knobs("track_block", block)
    n = 4 * 128 * 3 + 201
    cfg = W.config(3, n=n)
    c = W.make_bunch(cfg)
    got, ref_state, launch = gpu_track(cfg, c, nturns=7)
    assert launch["particles_per_thread"] == ppt and launch["block"] == block
    ref, (g_ref, _) = oracle_track(cfg, c, nturns=7)
    check(got, ref)
    assert abs(ref_state[0] - g_ref) <= 1e-15 * g_ref
    cfg = W.config(2, n=n)
    c = W.make_bunch(cfg)
    got, _, _ = gpu_track(cfg, c)
    ref, _ = oracle_track(cfg, c)
    check(got, ref)


def test_record_fusion_is_bit_identical(knobs):
    """Peephole fusion of adjacent thin kicks / trailing drift into one record changes the dispatch count, not the
    arithmetic: with the knob track_fuse = 0 (one record per element) the walk must give the same bits.  configs[3]'s ring
    exercises all three fusions: SEXTOCT, TAILDRIFT and the half-cell runs (one dispatch per 25 half cells)."""
    cfg = W.config(3, n=5000)
    c = W.make_bunch(cfg)
    fused, _, _ = gpu_track(cfg, c, nturns=3)
    knobs("track_fuse", 0)
    plain, _, _ = gpu_track(cfg, c, nturns=3)
    assert all(np.array_equal(a, b) for a, b in zip(fused, plain))


def test_lattice_longer_than_one_launch_table():
    """> 510 records per turn: the walk is split into several launches per turn (static and per-turn tables)."""
    cell = [("quad", 0.2, 1, 1.3), ("multipole", 0.0, 1, 3, 0.2, 0.0), ("drift", 0.1, 1), ("quad", 0.2, 7, -1.3),
            ("multipole", 0.0, 1, 4, 2.0, 0.0), ("multipole", 0.0, 1, 3, -0.2, 0.0), ("multipole", 0.0, 1, 4, 0.9, 0.0), ("drift", 0.1, 2)]
    lat = cell * 300                                   # 2400 elements -> 2400 records (one fused pair, one split quad per cell)
    cfg = W.config(0, n=2500)
    c = W.make_bunch(cfg)
    got, _, _ = gpu_track(cfg, c, nturns=2, lattice=lat)
    ref, _ = oracle_track(cfg, c, nturns=2, lattice=lat)
    check(got, ref)
    lat_rf = lat + [("shortrf", 0.0, 1, 1e-3, 1e7, -20.0)]
    got, (g, _, _), _ = gpu_track(cfg, c, nturns=3, lattice=lat_rf)
    ref, (g_ref, _) = oracle_track(cfg, c, nturns=3, lattice=lat_rf)
    check(got, ref)
    assert abs(g - g_ref) <= 1e-15 * g_ref


@pytest.mark.parametrize("window", [1, 700, 3000])
def test_walk_planned_in_windows_is_bit_identical(window, knobs):
    """bt_track / bt_track_host build the per-turn coefficient tables one window of records at a time (bounded host memory for
    any nturns) and carry the reference energy from window to window.  Forced here to windows of one turn, of a few turns and
    of about a turn (lattice longer than one launch table): the same bits and the same final gamma as the whole-call plan."""
    import torch
    import paper_2208_02382_b200 as bt
    cfg = W.config(3, n=20_003)
    c = W.make_bunch(cfg)
    cell = [("quad", 0.2, 1, 1.3), ("multipole", 0.0, 1, 3, 0.2, 0.0), ("drift", 0.1, 1), ("quad", 0.2, 7, -1.3),
            ("multipole", 0.0, 1, 4, 2.0, 0.0), ("multipole", 0.0, 1, 3, -0.2, 0.0), ("multipole", 0.0, 1, 4, 0.9, 0.0), ("drift", 0.1, 2)]
    long_static = cell * 300                                                   # 2400 records per turn, no RF
    long_rf = long_static + [("shortrf", 0.0, 1, 1e-3, 1e7, -20.0)]
    for lat, nturns in ((cfg.lattice, 7), (long_static, 3), (long_rf, 3)):    # cfg 3: RF ring, 7 turns = 2 launches unwindowed
        results = []
        for w in (-1, window):
            knobs("plan_window", w)
            beam = bt.Beam(cfg.n)
            beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
            beam.lattice_set(lat)
            beam.upload(c)
            beam.track(nturns)
            plain, ref = beam.download(), beam.get_ref()
            beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
            pinned = [torch.from_numpy(a.copy()).pin_memory() for a in c]
            out = [torch.empty(cfg.n, dtype=torch.float64).pin_memory() for _ in range(6)]
            beam.track_host(pinned, out, nturns=nturns, nchunks=3)
            assert beam.get_ref() == ref
            for a, b in zip(out, plain):
                assert np.array_equal(a.numpy(), b)
            results.append((plain, ref))
            beam.close()
        for a, b in zip(results[0][0], results[1][0]):
            assert np.array_equal(a, b)
        assert results[0][1] == results[1][1]


def test_two_beams_with_different_lattices_interleaved():
    """The record table travels with each launch (kernel parameters): beams with different lattices on different
    streams, interleaved, must each see their own table."""
    import torch
    import paper_2208_02382_b200 as bt
    cfg_a, cfg_b = W.config(1, n=40_000), W.config(3, n=30_000)
    ca, cb = W.make_bunch(cfg_a), W.make_bunch(cfg_b)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    a = bt.Beam(cfg_a.n, stream=sa.cuda_stream)
    b = bt.Beam(cfg_b.n, stream=sb.cuda_stream)
    for beam, cfg, c in ((a, cfg_a, ca), (b, cfg_b, cb)):
        beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, 1.0)
        beam.lattice_set(cfg.lattice)
        beam.upload(c)
    for _ in range(3):
        a.track(1)
        b.track(2)
    got_a, got_b = a.download(), b.download()
    check(got_a, oracle_track(cfg_a, ca, nturns=3)[0])
    check(got_b, oracle_track(cfg_b, cb, nturns=6)[0])
    a.close()
    b.close()


def test_config2_chicane_reduced():
    cfg = W.config(2, n=300_007)
    c = W.make_bunch(cfg)
    got, _, _ = gpu_track(cfg, c)
    ref, _ = oracle_track(cfg, c)
    check(got, ref)
    assert abs(got[4].std() / c[4].std() - 0.4658) < 2e-3     # compression by |1 - 20 R56|


def test_config3_ring_reduced_100_turns():
    cfg = W.config(3, n=20_003)
    c = W.make_bunch(cfg)
    got, (g, s, turn), _ = gpu_track(cfg, c)
    ref, (g_ref, s_ref) = oracle_track(cfg, c)
    errs = check(got, ref)
    assert abs(g - g_ref) <= 1e-15 * g_ref and abs(s - 7500.0) < 1e-6 and turn == 100
    assert abs(g - 2.1580889531834284) < 1e-12       # gamma after 100 turns


def test_general_multipoles_sbend_slices_and_skew():
    """Ops that no BASELINE config exercises: general-order / skew multipoles (OP_MULT), sliced sbend, sliced drift,
    k = 0 quad, dipole kick."""
    lat = [("drift", 0.3, 3), ("quad", 0.4, 2, 0.0), ("sbend", 0.9, 4, 3.0), ("dipedge", 0.0, 1, 0.1, 3.0, 0.01, 0.45),
           ("multipole", 0.0, 1, 1, 1e-4, -2e-4), ("multipole", 0.0, 1, 2, 0.3, 0.1), ("multipole", 0.0, 1, 3, 4.0, 2.0),
           ("multipole", 0.0, 1, 4, 30.0, -10.0), ("multipole", 0.0, 1, 5, 1e3, 5e2), ("multipole", 0.0, 1, 10, 1e9, 1e9),
           ("sbend", 0.9, 1, -3.0), ("quad", 0.5, 7, -2.0), ("shortrf", 0.0, 1, 1e-3, 1e8, -90.0), ("drift", 1.0, 1)]
    cfg = W.config(0, n=3000)
    c = W.make_bunch(cfg)
    got, _, _ = gpu_track(cfg, c, nturns=3, lattice=lat)
    ref, _ = oracle_track(cfg, c, nturns=3, lattice=lat)
    check(got, ref)


def test_repeated_calls_continue_and_zero_turns():
    import paper_2208_02382_b200 as bt
    cfg = W.config(3, n=1000)
    c = W.make_bunch(cfg)
    beam = bt.Beam(cfg.n)
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, 1.0)
    beam.lattice_set(cfg.lattice)
    beam.upload(c)
    beam.track(0)
    assert all(np.array_equal(a, b) for a, b in zip(beam.download(), c))
    beam.track(2)
    beam.track(3)
    got = beam.download()
    ref, (g_ref, _) = oracle_track(cfg, c, nturns=5)
    check(got, ref)
    assert beam.get_ref()[2] == 5 and abs(beam.get_ref()[0] - g_ref) < 1e-15 * g_ref
    # bit-reproducible run to run
    beam.upload(c)
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, 1.0)
    beam.track(5)
    again = beam.download()
    assert all(np.array_equal(a, b) for a, b in zip(got, again))
    beam.close()


def test_borrowed_unaligned_and_library_storage():
    import torch
    cfg = W.config(1, n=5000)
    cfg.lattice = W.fodo_cell(25) * 2
    c = W.make_bunch(cfg)
    ref, _ = oracle_track(cfg, c)
    # borrowed tensors whose data pointers are only 8-byte aligned -> scalar path
    backing = [torch.empty(cfg.n + 1, dtype=torch.float64, device="cuda") for _ in range(6)]
    views = [b[1:] for b in backing]
    got, _, launch = gpu_track(cfg, c, storage=views)
    assert launch["particles_per_thread"] == 1
    check(got, ref)
    assert all(np.array_equal(v.cpu().numpy(), g) for v, g in zip(views, got))      # zero-copy view sees the result
    got, _, _ = gpu_track(cfg, c, storage="library")
    check(got, ref)


def test_error_paths_on_device():
    import paper_2208_02382_b200 as bt
    beam = bt.Beam(100)
    with pytest.raises(bt.BtError) as ei:
        beam.track(1)
    assert ei.value.code == bt.BT_ERR_STATE
    beam.lattice_set(W.fodo_cell(2))
    with pytest.raises(bt.BtError) as ei:
        beam.track(1)
    assert ei.value.code == bt.BT_ERR_STATE          # no reference particle yet
    for bad in ([("quad", 1.0, 0, 1.0)], [("sbend", 1.0, 1, 0.0)], [("multipole", 0.0, 1, 11, 1.0, 0.0)],
                [("dipedge", 0.0, 2, 0.1, 1.0, 0.0, 0.0)], [("drift", -1.0, 1)], [(9, 1.0, 1)]):
        with pytest.raises(bt.BtError) as ei:
            beam.lattice_set(bad)
        assert ei.value.code == bt.BT_ERR_INVALID
    with pytest.raises(bt.BtError):
        beam.set_ref(-1.0, 1.0)
    beam.close()


# ---- BASELINE full sizes, in the launch configuration bench.py times ------------------------------------
def test_config1_full_size_every_particle():
    cfg = W.config(1)
    c = W.make_bunch(cfg)
    got, _, launch = gpu_track(cfg, c)
    ref, _ = oracle_track(cfg, c)
    check(got, ref)
    assert launch["particles_per_thread"] == 2      # long records: smaller tasks fill the tail better (track.cu)


def test_config2_full_size_every_particle():
    cfg = W.config(2)
    c = W.make_bunch(cfg)
    got, _, _ = gpu_track(cfg, c)
    ref, _ = oracle_track(cfg, c)
    check(got, ref)


def test_config3_full_size_sampled():
    """64M particles x 100 turns on the GPU; the oracle tracks the strided subset i % 64 == 0 (particles are
    independent, so the subset's result is the full run's result for those particles) + global invariants.
    Then the call bench.py's e2e leg times -- bt_track_host(pinned in, pinned out, 100 turns, 16 chunks) on the same bunch --
    must leave, in the host buffers, the same bits as bt_track left on the device, for every particle."""
    import torch
    import paper_2208_02382_b200 as bt
    cfg = W.config(3)
    c = W.make_bunch(cfg)
    got, (g, s, turn), _ = gpu_track(cfg, c)
    sub = [a[::64].copy() for a in c]
    pinned = [torch.from_numpy(a).pin_memory() for a in c]
    del c
    out = [torch.empty(cfg.n, dtype=torch.float64).pin_memory() for _ in range(6)]
    beam = bt.Beam(cfg.n)
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
    beam.lattice_set(cfg.lattice)
    beam.track_host(pinned, out, nturns=cfg.nturns, nchunks=16)
    assert beam.get_ref() == (g, s, turn)
    beam.close()
    del pinned
    for a, b in zip(out, got):
        assert np.array_equal(a.numpy(), b)
    del out
    ref, (g_ref, _) = oracle_track(cfg, sub)
    check([a[::64] for a in got], ref)
    assert abs(g - g_ref) <= 1e-15 * g_ref and turn == 100
    for a in got:
        assert np.all(np.isfinite(a))
    # normalised transverse emittances stay within a few % (nonlinear ring, no losses)
    from _util import rms_emittance
    bg = np.sqrt(g * g - 1)
    bg0 = 1.807618289845165
    ex = rms_emittance(got[0], got[1]) * bg / bg0
    assert 0.9e-6 < ex < 1.5e-6


@pytest.mark.parametrize("nchunks", [1, 3, 8, 64])
def test_track_host_pipelined_is_bit_identical(nchunks):
    """bt_track_host (chunks on three streams, copies overlapped) == upload + bt_track + download, bit for bit, and
    within R14 of the oracle; ragged chunking (n not a multiple of anything), in-place host buffers."""
    import torch
    import paper_2208_02382_b200 as bt
    cfg = W.config(1, n=70_001)
    lat = cfg.lattice[:10]
    c = W.make_bunch(cfg)
    beam = bt.Beam(cfg.n)
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
    beam.lattice_set(lat)
    beam.upload(c)
    beam.track(2)
    plain = beam.download()
    pinned = [torch.from_numpy(a.copy()).pin_memory() for a in c]
    beam.track_host(pinned, None, nturns=2, nchunks=nchunks)           # in place
    got = [t.numpy() for t in pinned]
    for a, b in zip(got, plain):
        assert np.array_equal(a, b)
    dev = beam.download()                                               # the device copy holds the result too
    for a, b in zip(dev, plain):
        assert np.array_equal(a, b)
    ref, _ = oracle_track(cfg, c, nturns=2, lattice=lat)
    assert max(r14_error(got, ref)) <= 1e-11
    g, s, turn = beam.get_ref()
    assert turn == 4
    beam.close()


@pytest.mark.parametrize("nchunks", [3, 8])
def test_track_host_with_rf_lattice_is_pipelined_and_bit_identical(nchunks):
    """A lattice whose RF changes the reference energy (per-turn tables, 7 turns = 2 launches per chunk) through the chunked
    host path: every launch carries its own table, so the chunk streams need no serialisation.  Bit-identical to
    upload + bt_track + download, same reference energy, one walk launch per (chunk, plan launch)."""
    import torch
    import paper_2208_02382_b200 as bt
    cfg = W.config(3, n=20_003)
    c = W.make_bunch(cfg)
    beam = bt.Beam(cfg.n)
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
    beam.lattice_set(cfg.lattice)
    beam.upload(c)
    n0 = bt.launch_count()
    beam.track(7)
    per_call = bt.launch_count() - n0
    plain, g_plain = beam.download(), beam.get_ref()[0]
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
    pinned = [torch.from_numpy(a.copy()).pin_memory() for a in c]
    out = [torch.empty(cfg.n, dtype=torch.float64).pin_memory() for _ in range(6)]
    n0 = bt.launch_count()
    beam.track_host(pinned, out, nturns=7, nchunks=nchunks)
    chunk_len = -(-(-(-cfg.n // nchunks)) // 1024) * 1024               # chunks are whole 1024-particle granules
    assert per_call == 2 and bt.launch_count() - n0 == per_call * -(-cfg.n // chunk_len)
    for a, b in zip(out, plain):
        assert np.array_equal(a.numpy(), b)
    g, s, turn = beam.get_ref()
    assert g == g_plain and turn == 7
    ref, _ = oracle_track(cfg, c, nturns=7)
    assert max(r14_error([t.numpy() for t in out], ref)) <= 1e-11
    assert bt.lib.bt_track_host(beam._h, None, None, 1, 8) == bt.BT_ERR_INVALID
    beam.close()


def _nonlinear_ring():
    """FODO cells with exact drifts, thin sextupoles and one sinusoidal RF cavity per turn (NEXT-3 elements)."""
    cell = [("quad", 1.0, 5, 1.0), ("multipole", 0.0, 1, 3, 5.0, 0.0), ("drift_exact", 0.5, 3),
            ("quad", 1.0, 5, -1.0), ("multipole", 0.0, 1, 3, -5.0, 0.0), ("drift_exact", 0.5, 1)]
    return cell * 4 + [("shortrf_sin", 0.0, 1, 1.0 / 938.27208816, 3.4976811924685272e6 * 40, -30.0)]


@pytest.mark.parametrize("n,nturns", [(1, 3), (10_007, 5), (300_001, 2)])
def test_nonlinear_maps_match_oracle(n, nturns):
    """R17 exact drift + R18 sinusoidal RF inside the fused walk (per-turn tables: the RF moves the reference energy)."""
    cfg = W.config(3, n=n)
    lat = _nonlinear_ring()
    c = W.make_bunch(cfg)
    c[4] *= 30.0                                     # spread t over a good fraction of the RF wavelength (2.1 m)
    got, (g, s, turn), _ = gpu_track(cfg, c, nturns=nturns, lattice=lat)
    ref, (g_ref, s_ref) = oracle_track(cfg, c, nturns=nturns, lattice=lat)
    assert max(r14_error(got, ref)) <= 1e-11
    assert abs(g - g_ref) <= 4e-16 * g_ref and abs(s - s_ref) <= 1e-12 and turn == nturns
    # and they are different maps from their linearised versions (R4, R9) on this bunch
    lin = [("drift",) + e[1:] if e[0] == "drift_exact" else ("shortrf",) + e[1:] if e[0] == "shortrf_sin" else e for e in lat]
    ref_lin, _ = oracle_track(cfg, c, nturns=nturns, lattice=lin)
    if n > 1:
        assert max(r14_error(ref_lin, ref)) > 1e-6


def test_exact_drift_only_lattice_static_table_and_host_pipeline():
    import torch
    import paper_2208_02382_b200 as bt
    cfg = W.config(0, n=50_001)
    lat = [("drift_exact", 0.25, 1), ("quad", 1.0, 10, 1.0), ("drift_exact", 0.5, 4), ("quad", 1.0, 10, -1.0), ("drift_exact", 0.25, 1)]
    c = W.make_bunch(cfg)
    got, _, _ = gpu_track(cfg, c, nturns=4, lattice=lat)
    ref, _ = oracle_track(cfg, c, nturns=4, lattice=lat)
    assert max(r14_error(got, ref)) <= 1e-11
    beam = bt.Beam(cfg.n)
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
    beam.lattice_set(lat)
    out = beam.track_host(c, [np.empty_like(a) for a in c], nturns=4, nchunks=5)
    for a, b in zip(out, got):
        assert np.array_equal(a, b)
    beam.close()


def test_nonlinear_element_validation():
    import paper_2208_02382_b200 as bt
    beam = bt.Beam(8)
    with pytest.raises(bt.BtError):
        beam.lattice_set([("shortrf_sin", 0.0, 2, 1e-3, 1e8, 0.0)])
    with pytest.raises(bt.BtError):
        beam.lattice_set([("drift_exact", -1.0, 1)])
    beam.close()


@pytest.mark.parametrize("n,nturns", [(1, 2), (20_011, 3), (200_001, 1)])
def test_chromatic_quad_matches_oracle(n, nturns):
    """R20 chromatic quadrupole (both signs, k = 0, sliced) mixed with exact drifts and linear elements in one walk."""
    cfg = W.config(0, n=n)
    lat = [("drift_exact", 0.25, 1), ("quad_chromatic", 1.0, 4, 1.0), ("drift", 0.5, 2), ("quad_chromatic", 1.0, 3, -1.0),
           ("quad_chromatic", 0.3, 1, 0.0), ("quad", 0.2, 2, 0.7), ("drift_exact", 0.25, 1)]
    c = W.make_bunch(cfg)
    c[5] *= 10.0                                       # percent-level momentum spread: the chromatic effect is visible
    got, (g, s, turn), _ = gpu_track(cfg, c, nturns=nturns, lattice=lat)
    ref, (g_ref, s_ref) = oracle_track(cfg, c, nturns=nturns, lattice=lat)
    assert max(r14_error(got, ref)) <= 1e-11
    assert g == g_ref and abs(s - s_ref) <= 1e-12
    if n > 1:
        lin = [("quad",) + e[1:] if e[0] == "quad_chromatic" else e for e in lat]
        ref_lin, _ = oracle_track(cfg, c, nturns=nturns, lattice=lin)
        assert max(r14_error(ref_lin, ref)) > 1e-4      # a different map from R5 on this bunch


@pytest.mark.parametrize("seed", [0, 1, 2, 3, 4, 5])
def test_random_lattices_of_all_element_kinds(seed):
    """Seeded random lattices mixing all nine element kinds (random order, parameters, slice counts; with and without
    energy-changing cavities), several turns: exercises every opcode, the peephole fusions and the per-turn tables."""
    rng = np.random.default_rng(1000 + seed)
    cfg = W.config(0, n=3001 + 64 * seed)
    lat = []
    for _ in range(int(rng.integers(8, 24))):
        kind = int(rng.integers(0, 9))
        ns = int(rng.integers(1, 8))
        L = float(rng.uniform(0.05, 0.6))
        if kind == 0:
            lat.append(("drift", L, ns))
        elif kind == 1:
            lat.append(("quad", L, ns, float(rng.choice([-0.6, -0.3, 0.0, 0.4, 0.7]))))
        elif kind == 2:
            lat.append(("sbend", L, ns, float(rng.choice([-8.0, 5.0, 12.0]))))
        elif kind == 3:
            lat.append(("dipedge", 0.0, 1, float(rng.uniform(-0.2, 0.2)), float(rng.choice([-8.0, 5.0])), 0.02, 0.5))
        elif kind == 4:
            m = int(rng.integers(1, 7))
            lat.append(("multipole", 0.0, 1, m, float(rng.uniform(-0.5, 0.5)) * (1e-3 if m == 1 else 1.0),
                        float(rng.choice([0.0, rng.uniform(-0.3, 0.3)])) * (1e-3 if m == 1 else 1.0)))
        elif kind == 5 and seed % 2 == 0:
            lat.append(("shortrf", 0.0, 1, 1e-3, 2e8, float(rng.choice([-90.0, -30.0, 20.0]))))
        elif kind == 6:
            lat.append(("drift_exact", L, ns))
        elif kind == 7 and seed % 2 == 0:
            lat.append(("shortrf_sin", 0.0, 1, 5e-4, 1e8, float(rng.choice([-90.0, -45.0, 10.0]))))
        else:
            lat.append(("quad_chromatic", L, ns, float(rng.choice([-1.0, 0.0, 0.8]))))
    c = W.make_bunch(cfg)
    nturns = 2
    got, (g, s, turn), _ = gpu_track(cfg, c, nturns=nturns, lattice=lat)
    ref, (g_ref, s_ref) = oracle_track(cfg, c, nturns=nturns, lattice=lat)
    assert all(np.all(np.isfinite(a)) for a in ref), lat        # the lattices are tame enough for the bunch to survive
    assert max(r14_error(got, ref)) <= 1e-11, lat
    assert abs(g - g_ref) <= 8e-16 * g_ref and abs(s - s_ref) <= 1e-10 and turn == nturns


def test_track_host_edge_cases():
    """nturns = 0 copies through unchanged; more chunks than 1024-particle granules; tiny bunch."""
    import paper_2208_02382_b200 as bt
    cfg = W.config(0, n=1500)
    c = W.make_bunch(cfg)
    beam = bt.Beam(cfg.n)
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, cfg.charge_qe)
    beam.lattice_set(cfg.lattice)
    out = beam.track_host(c, [np.empty_like(a) for a in c], nturns=0, nchunks=4)
    for a, b in zip(out, c):
        assert np.array_equal(a, b)
    out = beam.track_host(c, [np.empty_like(a) for a in c], nturns=2, nchunks=200)
    ref, _ = oracle_track(cfg, c, nturns=2)
    assert max(r14_error(out, ref)) <= 1e-11
    assert bt.lib.bt_track_host(beam._h, None, None, 1, 0) == bt.BT_ERR_INVALID
    beam.close()
