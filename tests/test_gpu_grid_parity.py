"""Parity of bt_deposit_cic and bt_gather_kick (through the C-ABI) against the CPU oracle.

Deposit bar (north_star + reading R15): (i) isolated -- bit-identical positions on both sides: every non-zero
node within relative 1e-12 and identical zero-node set; (ii) in-run -- |rho_gpu - rho_ref| <= 1e-12 max(rho_ref,
q_weight); total charge within 1e-13.  Gather/kick bar: R14, 1e-11.
"""
import math

import numpy as np
import pytest

import oracle as O
import paper_2208_02382_b200 as bt
import workloads as W
from _gpu import r15_isolated
from _util import r14_error

pytestmark = pytest.mark.gpu


def gpu_deposit(c, sc, zscale=None, q_weight=None, accumulate_into=None):
    beam = bt.Beam(c[0].shape[0])
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    try:
        beam.upload(c)
        zs = sc.zscale if zscale is None else zscale
        qw = sc.q_weight if q_weight is None else q_weight
        beam.deposit_cic(grid, qw, zs, zero_first=True)
        if accumulate_into:
            beam.deposit_cic(grid, qw, zs, zero_first=False)
        return grid.download_rho()
    finally:
        beam.close()
        grid.close()


@pytest.mark.parametrize("variant", ["A", "B"])
@pytest.mark.parametrize("n,shape", [(1, (8, 8, 8)), (257, (16, 12, 10)), (200_003, (32, 32, 32)), (300_000, (128, 128, 128))])
def test_deposit_isolated(variant, n, shape):
    sc = W.spacecharge_config(variant, n=n, shape=shape)
    c = W.make_spacecharge_bunch(sc)
    rho = gpu_deposit(c, sc)
    ref, n_in = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight)
    assert r15_isolated(rho, ref) <= 1e-12
    total = math.fsum(rho.ravel())
    assert abs(total - sc.q_weight * n_in) <= 1e-13 * sc.q_weight * max(n_in, 1)


def test_deposit_boundaries_nan_zscale_and_accumulate():
    sc = W.spacecharge_config("A", n=5000, shape=(16, 16, 16))
    c = W.make_spacecharge_bunch(sc)
    lo, hi = sc.lo[0], sc.lo[0] + sc.d[0] * 15
    c[0][:8] = [lo, hi, np.nextafter(lo, -1), hi - 1e-12, np.nan, np.inf, -np.inf, 0.5]
    c[2][8:12] = [lo, hi, np.nan, 7.0]
    for zs in (1.0, -1.8, 0.25):
        rho = gpu_deposit(c, sc, zscale=zs)
        ref, n_in = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight, zs)
        assert 0 < n_in < sc.n
        assert r15_isolated(rho, ref) <= 1e-12
    twice = gpu_deposit(c, sc, accumulate_into=True)
    ref, _ = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight)
    assert r15_isolated(twice, 2.0 * ref) <= 1e-12


def test_deposit_all_outside_is_zero():
    sc = W.spacecharge_config("A", n=1000, shape=(8, 8, 8))
    c = W.make_spacecharge_bunch(sc)
    c[0][:] = 1.0
    assert not gpu_deposit(c, sc).any()


def gpu_gather(c, sc, E, coef, zscale=1.0, hb=0.0, ha=0.0, ref=(1000.0, W.MASS_PROTON_MEV)):
    beam = bt.Beam(c[0].shape[0])
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    try:
        beam.set_ref(ref[0], ref[1], 1.0)
        grid.set_field(*E)
        beam.upload(c)
        beam.gather_kick(grid, coef, zscale, hb, ha)
        return beam.download(), beam.get_ref()
    finally:
        beam.close()
        grid.close()


@pytest.mark.parametrize("variant,n,shape", [("A", 1, (8, 8, 8)), ("A", 100_003, (32, 32, 32)), ("B", 100_003, (32, 32, 32)),
                                               ("A", 200_000, (128, 128, 128))])
def test_gather_kick_only(variant, n, shape):
    sc = W.spacecharge_config(variant, n=n, shape=shape)
    c = W.make_spacecharge_bunch(sc)
    E = W.gaussian_bunch_field(sc)
    got, _ = gpu_gather(c, sc, E, sc.kick_coef)
    ref = [a.copy() for a in c]
    O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef)
    assert max(r14_error(got, ref)) <= 1e-11
    for k in (0, 2, 4):
        assert np.array_equal(got[k], c[k])           # kick only: positions untouched
    # the kick itself (a small difference of O(1e-6) on momenta of O(1e-3)) to 1e-9 of its own rms
    for k in (1, 3, 5):
        dk_g, dk_r = got[k] - c[k], ref[k] - c[k]
        scale = np.sqrt(np.mean(dk_r**2)) if n > 1 else max(abs(dk_r[0]), 1e-300)
        assert np.max(np.abs(dk_g - dk_r)) <= 1e-9 * scale


def test_gather_with_drifts_outside_particles_and_zscale():
    sc = W.spacecharge_config("A", n=50_000, shape=(16, 16, 16))
    c = W.make_spacecharge_bunch(sc)
    c[0][:100] = 0.02          # outside: zero field, still drifted
    c[4][100:110] = np.nan
    rng = np.random.default_rng(3)
    E = [rng.standard_normal((16, 16, 16)) * 1e5 for _ in range(3)]
    zs, hb, ha = -1.3, 0.004, 0.007
    cfg = W.config(3, n=1)
    got, (g, s, turn) = gpu_gather(c, sc, E, (1e-11, -2e-11, 3e-11), zs, hb, ha)
    ref = [a.copy() for a in c]
    g0 = O.ref_from_kinetic(1000.0, W.MASS_PROTON_MEV)[0]
    O.track(ref, [("drift", hb, 1)], 1, g0)
    O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, (1e-11, -2e-11, 3e-11), zs)
    O.track(ref, [("drift", ha, 1)], 1, g0)
    ok = ~np.isnan(ref[4])
    assert max(r14_error([a[ok] for a in got], [a[ok] for a in ref])) <= 1e-11
    assert np.all(np.isnan(got[4][~ok]))
    assert abs(s - (hb + ha)) < 1e-15
    assert np.array_equal(got[1][:100], c[1][:100])      # outside: momenta untouched


def test_gather_requires_field_and_ref():
    beam = bt.Beam(10)
    grid = bt.Grid((4, 4, 4), (0, 0, 0), (1, 1, 1))
    with pytest.raises(bt.BtError) as ei:
        beam.gather_kick(grid, (1, 1, 1))
    assert ei.value.code == bt.BT_ERR_STATE
    beam.close()
    grid.close()


@pytest.mark.parametrize("resort", [0, 3])
@pytest.mark.parametrize("variant", ["A", "B"])
def test_config4_in_run_reduced(variant, resort):
    """The BASELINE configs[4] step sequence at 4e5 particles / 64^3 nodes, in the caller's order and with the
    library re-sorting by cell every third deposit."""
    sc = W.spacecharge_config(variant, n=400_000, shape=(64, 64, 64))
    run_config4(sc, resort)


def run_config4(sc, resort_interval=0, order=1):
    """oracle = 10 x [D(.005); deposit; gather+kick(.01); D(.005)]; library = bt_track(D(.005)) once, then per step
    bt_deposit_cic + bt_gather_kick(0, .01 -- .005 on the last step): deposit and gather see the same positions.
    Checked: R15 (ii) (in-run: |rho - rho_ref| <= 1e-12 max(rho_ref, q_weight)) and the total charge at the first and at the
    last step -- the library's positions there differ from the oracle's by rounding (its drifts are FMAs, the oracle's are a
    rounded product and a rounded sum), which is exactly the case R15 (ii) is for; R15 (i) (isolated: strict 1e-12 on every
    non-zero node, identical zero set) on the ORACLE's positions of the first and of the last step, deposited by a second
    beam with the same storage handling; R14 on the final coordinates; s."""
    c = W.make_spacecharge_bunch(sc)
    E = W.gaussian_bunch_field(sc)
    g0 = O.ref_from_kinetic(sc.kin_energy_MeV, sc.mass_MeV)[0]
    half = [("drift", sc.ds / 2, 1)]
    check_steps = (0, sc.nsteps - 1)
    # oracle
    ref = [a.copy() for a in c]
    rho_ref, pos_ref = {}, {}
    for step in range(sc.nsteps):
        O.track(ref, half, 1, g0)
        if step in check_steps:
            rho_ref[step] = O.deposit_cic(ref[0], ref[2], ref[4], sc.shape, sc.lo, sc.d, sc.q_weight, sc.zscale, order=order)
            pos_ref[step] = [a.copy() for a in ref]
        O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale, order=order)
        O.track(ref, half, 1, g0)
    # library
    beam = bt.Beam(sc.n)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    grid.set_particle_shape(order)
    beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, sc.charge_qe)
    grid.set_field(*E)
    beam.upload(c)
    beam.lattice_set(half)
    beam.track(1)
    beam.set_resort_interval(resort_interval)
    for step in range(sc.nsteps):
        beam.deposit_cic(grid, sc.q_weight, sc.zscale, zero_first=True)
        if step in check_steps:
            rho = grid.download_rho()
            r, n_in = rho_ref[step]
            assert np.all(np.abs(rho - r) <= 1e-12 * np.maximum(r, sc.q_weight)), step          # R15 (ii)
            assert abs(math.fsum(rho.ravel()) - sc.q_weight * n_in) <= 1e-13 * sc.q_weight * n_in
        beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, sc.ds if step < sc.nsteps - 1 else sc.ds / 2)
    got = beam.download()
    assert max(r14_error(got, ref)) <= 1e-11
    assert abs(beam.get_ref()[1] - sc.nsteps * sc.ds) < 1e-12
    beam.close()
    # R15 (i): the oracle's own positions (bit-identical input), same storage handling
    iso = bt.Beam(sc.n)
    iso.set_ref(sc.kin_energy_MeV, sc.mass_MeV, sc.charge_qe)
    for step in check_steps:
        iso.upload(pos_ref[step])
        if resort_interval:
            iso.sort_by_cell(grid, sc.zscale)
        iso.deposit_cic(grid, sc.q_weight, sc.zscale, zero_first=True)
        assert r15_isolated(grid.download_rho(), rho_ref[step][0]) <= 1e-12, step
    iso.close()
    grid.close()


@pytest.mark.parametrize("resort", [0, 5, 10])
@pytest.mark.parametrize("variant", ["A", "B"])
def test_config4_full_size(variant, resort):
    """configs[4] as BASELINE states it -- 8e6 particles, 128^3 nodes, all 10 steps -- in the caller's order, with
    bt_beam_set_resort_interval(10), and with the interval bench.py times (5: a second library-triggered re-sort in the middle
    of the run -- the bunch ping-pongs back into its home arrays, the ids are composed twice -- followed by five more steps);
    criteria in run_config4."""
    run_config4(W.spacecharge_config(variant), resort)


@pytest.mark.parametrize("variant,resort", [("A", 3), ("A", 5), ("B", 3)])
def test_config4_full_size_order2(variant, resort):
    """The same run with the listing's own particle shape (P:l.60 set_particle_shape(2)) at the size and re-sort cadence
    bench.py's A_order2 leg times (8e6 particles, 128^3 nodes, 10 steps, interval 3; 5 = the order-1 cadence): the order-2-keyed
    sort, the 27-node deposit and the regrouping tile gather against the oracle's order-2 loop, same criteria."""
    run_config4(W.spacecharge_config(variant), resort, order=2)


# ---- S4 cell binning ---------------------------------------------------------------------------------
def _cell_keys(c, sc, zscale=1.0):
    """Host restatement of the canonical index, for checking sortedness only."""
    u = [(c[0] - sc.lo[0]) * (1.0 / sc.d[0]), (c[2] - sc.lo[1]) * (1.0 / sc.d[1]), (zscale * c[4] - sc.lo[2]) * (1.0 / sc.d[2])]
    nx, ny, nz = sc.shape
    inside = np.ones(len(c[0]), dtype=bool)
    for a, n in zip(u, (nx, ny, nz)):
        inside &= (a >= 0) & (a < n - 1)
    ijk = [np.where(inside, np.floor(np.where(inside, a, 0.0)), 0).astype(np.int64) for a in u]
    return np.where(inside, (ijk[2] * ny + ijk[1]) * nx + ijk[0], nx * ny * nz)


@pytest.mark.parametrize("variant,n,shape", [("A", 1, (8, 8, 8)), ("A", 1023, (8, 8, 8)), ("A", 300_001, (32, 32, 32)),
                                               ("B", 300_001, (32, 32, 32)), ("A", 500_000, (128, 128, 128))])
def test_sort_by_cell_orders_storage_and_keeps_api_order(variant, n, shape):
    import torch
    sc = W.spacecharge_config(variant, n=n, shape=shape)
    c = W.make_spacecharge_bunch(sc)
    if n > 100:
        c[0][:7] = [1.0, np.nan, -1.0, np.inf, 0.0, 5.9e-3, -5.9e-3]      # some outside particles
    E = W.gaussian_bunch_field(sc)
    beam = bt.Beam(n)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, 1.0)
    grid.set_field(*E)
    beam.upload(c)
    assert beam.ids_ptr() == 0
    beam.sort_by_cell(grid, sc.zscale)
    # API order unchanged, bit for bit
    back = beam.download()
    for a, b in zip(back, c):
        assert np.array_equal(a, b, equal_nan=True)
    # storage order sorted by cell key; ids is a permutation consistent with the data
    stored = [t.cpu().numpy() for t in beam.tensors]
    keys = _cell_keys(stored, sc, sc.zscale)
    assert np.all(np.diff(keys) >= 0)
    assert beam.ids_ptr() != 0
    ids = np.empty(n, dtype=np.int32)
    import ctypes
    torch.cuda.synchronize()
    ids_t = torch.empty(n, dtype=torch.int32, device="cuda")
    ctypes.cdll.LoadLibrary("libcudart.so").cudaMemcpy(ctypes.c_void_p(ids_t.data_ptr()), ctypes.c_void_p(beam.ids_ptr()), ctypes.c_size_t(4 * n), 3)
    ids = ids_t.cpu().numpy()
    assert np.array_equal(np.sort(ids), np.arange(n))
    assert np.array_equal(stored[1], c[1][ids])
    # deposit + gather on sorted storage == oracle on the original order
    beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
    rho = grid.download_rho()
    ref_rho, n_in = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight, sc.zscale)
    assert r15_isolated(rho, ref_rho) <= 1e-12
    beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, sc.ds)
    beam.sort_by_cell(grid, sc.zscale)            # sorting twice composes the permutations
    got = beam.download()
    ref = [a.copy() for a in c]
    O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale)
    O.track(ref, [("drift", sc.ds, 1)], 1, O.ref_from_kinetic(sc.kin_energy_MeV, sc.mass_MeV)[0])
    ok = np.isfinite(ref[0])
    assert max(r14_error([a[ok] for a in got], [a[ok] for a in ref])) <= 1e-11
    # upload resets the storage order
    beam.upload(c)
    assert beam.ids_ptr() == 0
    beam.close()
    grid.close()


def test_sorted_tracking_still_matches():
    """bt_track on cell-sorted storage: download must still be the original order."""
    cfg = W.config(0, n=5000)
    c = W.make_bunch(cfg)
    sc = W.spacecharge_config("A", n=5000, shape=(16, 16, 16))
    beam = bt.Beam(cfg.n)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    beam.set_ref(cfg.kin_energy_MeV, cfg.mass_MeV, 1.0)
    beam.lattice_set(cfg.lattice)
    beam.upload(c)
    beam.sort_by_cell(grid, 1.0)
    beam.track(3)
    got = beam.download()
    from _gpu import oracle_track
    ref, _ = oracle_track(cfg, c, nturns=3)
    assert max(r14_error(got, ref)) <= 1e-11
    beam.close()
    grid.close()


@pytest.mark.parametrize("mode", [0, 1, 2, 3])
@pytest.mark.parametrize("variant", ["A", "B"])
def test_deposit_modes_unaligned(mode, variant, knobs):
    import torch
    knobs("deposit_mode", mode)
    sc = W.spacecharge_config(variant, n=70_001, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    backing = [torch.empty(sc.n + 1, dtype=torch.float64, device="cuda") for _ in range(6)]
    beam = bt.Beam(sc.n, storage=[b[1:] for b in backing])
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    beam.upload(c)
    beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
    rho = grid.download_rho()
    ref_rho, _ = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight, sc.zscale)
    assert r15_isolated(rho, ref_rho) <= 1e-12
    beam.close()
    grid.close()


@pytest.mark.parametrize("mode", [0, 1, 2, 3, 4, 5])
@pytest.mark.parametrize("offset", [0, 1])
def test_gather_modes(mode, offset, knobs):
    """Every gather path (registers / streaming pipeline with 256-, 512-, 128-particle chunks), on aligned and on
    8-byte-offset storage (the pipeline needs 16-byte alignment: offset storage must take the register path), with a
    ragged tail, sorted storage, drifts on both sides and a kick-only call."""
    import torch
    knobs("gather_mode", mode)
    sc = W.spacecharge_config("A", n=70_001, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    c[0][:5] = [1.0, np.nan, -1.0, 5.9e-3, -5.9e-3]
    E = W.gaussian_bunch_field(sc)
    backing = [torch.empty(sc.n + 2, dtype=torch.float64, device="cuda") for _ in range(6)]
    beam = bt.Beam(sc.n, storage=[b[offset:offset + sc.n] for b in backing])
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
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
    O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale)
    O.track(ref, [("drift", sc.ds, 1)], 1, g0)
    O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale)
    ok = np.isfinite(ref[0])
    assert max(r14_error([a[ok] for a in got], [a[ok] for a in ref])) <= 1e-11
    beam.close()
    grid.close()


@pytest.mark.parametrize("seed", range(8))
def test_random_grids_shapes_orders_and_clouds(seed):
    """Seeded random grids (anisotropic, non-cubic, offset), particle clouds that partly leave the grid, both shape orders,
    random zscale, sorted or not: deposit (R15 isolated) and gather + kick with drifts (R14) against the oracle."""
    rng = np.random.default_rng(500 + seed)
    shape = tuple(int(v) for v in rng.integers(3, 40, 3))
    d = tuple(float(v) for v in rng.uniform(0.2e-3, 2e-3, 3))
    lo = tuple(float(v) for v in rng.uniform(-5e-3, 0.0, 3))
    order = 1 + seed % 2
    zscale = float(rng.choice([1.0, -1.0, 0.37, 2.5]))
    n = int(rng.integers(1, 60_000))
    centre = [lo[a] + 0.5 * d[a] * (shape[a] - 1) for a in range(3)]
    width = [0.35 * d[a] * (shape[a] - 1) for a in range(3)]
    c = [np.zeros(n) for _ in range(6)]
    c[0] = centre[0] + width[0] * rng.standard_normal(n)
    c[2] = centre[1] + width[1] * rng.standard_normal(n)
    c[4] = (centre[2] + width[2] * rng.standard_normal(n)) / zscale
    for a in (1, 3, 5):
        c[a] = 1e-3 * rng.standard_normal(n)
    nn = shape[0] * shape[1] * shape[2]
    E = [rng.standard_normal((shape[2], shape[1], shape[0])) * 1e5 for _ in range(3)]
    coef, qw, ds = (1e-9, -2e-9, 0.5e-9), 1e-9 / n, 0.01
    beam = bt.Beam(n)
    grid = bt.Grid(shape, lo, d)
    grid.set_particle_shape(order)
    beam.set_ref(1000.0, W.MASS_PROTON_MEV, 1.0)
    grid.set_field(*E)
    beam.upload(c)
    if seed % 3 == 0:
        beam.sort_by_cell(grid, zscale)
    beam.deposit_cic(grid, qw, zscale, True)
    rho = grid.download_rho()
    ref_rho, n_in = O.deposit_cic(c[0], c[2], c[4], shape, lo, d, qw, zscale, order=order)
    assert r15_isolated(rho, ref_rho) <= 1e-12
    assert abs(math.fsum(rho.ravel()) - qw * n_in) <= 1e-13 * qw * max(n_in, 1)
    beam.gather_kick(grid, coef, zscale, ds / 2, ds)
    got = beam.download()
    g0 = O.ref_from_kinetic(1000.0, W.MASS_PROTON_MEV)[0]
    ref = [a.copy() for a in c]
    O.track(ref, [("drift", ds / 2, 1)], 1, g0)
    O.gather_kick(ref, shape, lo, d, E, coef, zscale, order=order)
    O.track(ref, [("drift", ds, 1)], 1, g0)
    assert max(r14_error(got, ref)) <= 1e-11
    assert nn > 0
    beam.close()
    grid.close()


def test_resort_interval_sorts_inside_deposit_and_keeps_results():
    """bt_beam_set_resort_interval(3): deposits 1, 4, 7 re-bin the storage themselves; the step loop still matches the
    oracle's loop (API order is unaffected), and upload resets the cadence."""
    sc = W.spacecharge_config("A", n=120_000, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    E = W.gaussian_bunch_field(sc)
    g0 = O.ref_from_kinetic(sc.kin_energy_MeV, sc.mass_MeV)[0]
    beam = bt.Beam(sc.n)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, 1.0)
    grid.set_field(*E)
    beam.set_resort_interval(3)
    beam.upload(c)
    assert beam.ids_ptr() == 0
    ref = [a.copy() for a in c]
    for step in range(5):
        beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
        assert beam.ids_ptr() != 0                      # sorted by the first deposit
        rho = grid.download_rho()
        rref, _ = O.deposit_cic(ref[0], ref[2], ref[4], sc.shape, sc.lo, sc.d, sc.q_weight, sc.zscale)
        assert np.max(np.abs(rho - rref) / np.maximum(rref, sc.q_weight)) <= 1e-12
        beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, sc.ds)
        O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale)
        O.track(ref, [("drift", sc.ds, 1)], 1, g0)
        if step in (0, 3):                               # right after a sort the storage is in cell order at the deposit's positions
            pass
    got = beam.download()
    assert max(r14_error(got, ref)) <= 1e-11
    beam.upload(c)
    assert beam.ids_ptr() == 0
    assert bt.lib.bt_beam_set_resort_interval(beam._h, -1) == bt.BT_ERR_INVALID
    beam.set_resort_interval(0)
    beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
    assert beam.ids_ptr() == 0                           # interval 0: the deposit never sorts
    beam.close()
    grid.close()


@pytest.mark.parametrize("pingpong", [False, True])
def test_lent_tensors_keep_holding_the_bunch_across_library_triggered_sorts(pingpong):
    """The zero-copy contract (P:l.102) for arrays the caller lent: external code keeps the tensors it passed in, so after
    any number of sorts -- the ones bt_deposit_cic triggers under a re-sort interval included -- those tensors ARE the bunch
    (storage order, ids map back), and bt_beam_download never scribbles on them.  With ping-pong switched on explicitly the
    bunch may sit in the library's partner arrays; bt_beam_storage says so, bt_beam_rehome brings it back, and the lent
    tensors are left untouched meanwhile."""
    import ctypes
    import torch
    sc = W.spacecharge_config("A", n=150_001, shape=(32, 32, 32))
    c = W.make_spacecharge_bunch(sc)
    E = W.gaussian_bunch_field(sc)
    lent = [torch.empty(sc.n, dtype=torch.float64, device="cuda") for _ in range(6)]
    lent_ptrs = [t.data_ptr() for t in lent]
    beam = bt.Beam(sc.n, storage=lent, pingpong=pingpong if pingpong else None)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, 1.0)
    grid.set_field(*E)
    beam.set_resort_interval(2)
    beam.upload(c)
    assert beam.storage()[0] and beam.ptrs() == lent_ptrs
    cudart = ctypes.cdll.LoadLibrary("libcudart.so")

    def ids():
        t = torch.empty(sc.n, dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        cudart.cudaMemcpy(ctypes.c_void_p(t.data_ptr()), ctypes.c_void_p(beam.ids_ptr()), ctypes.c_size_t(4 * sc.n), 3)
        return t.cpu().numpy()

    seen_away = False
    epochs = [beam.storage()[1]]
    for step in range(5):                               # sorts before deposits 1, 3, 5
        beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
        beam.gather_kick(grid, sc.kick_coef, sc.zscale, 0.0, sc.ds)
        in_home, epoch = beam.storage()
        api = beam.download()                           # API order; must not disturb the lent tensors
        if in_home:
            assert beam.ptrs() == lent_ptrs
            stored = [t.cpu().numpy() for t in lent]
            perm = ids()
            for a, b in zip(stored, api):               # the lent tensors hold the bunch: storage slot j = original particle ids[j]
                assert np.array_equal(a, b[perm])
        else:
            assert pingpong
            seen_away = True
            assert beam.ptrs() != lent_ptrs
            before = [t.clone() for t in lent]
            beam.download()
            for a, b in zip(before, lent):              # stale, but the caller's: not used as scratch
                assert torch.equal(a, b)
            beam.rehome()
            assert beam.storage() == (True, epoch + 1) and beam.ptrs() == lent_ptrs
            perm = ids()
            for a, b in zip([t.cpu().numpy() for t in lent], api):
                assert np.array_equal(a, b[perm])
        epochs.append(beam.storage()[1])
    assert seen_away == pingpong
    assert epochs[1] > epochs[0] and epochs[2] == epochs[1] and epochs[3] > epochs[2]   # moved by deposits 1 and 3, not by 2
    ref = [a.copy() for a in c]
    g0 = O.ref_from_kinetic(sc.kin_energy_MeV, sc.mass_MeV)[0]
    for step in range(5):
        O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, sc.kick_coef, sc.zscale)
        O.track(ref, [("drift", sc.ds, 1)], 1, g0)
    assert max(r14_error(beam.download(), ref)) <= 1e-11
    beam.close()
    grid.close()
