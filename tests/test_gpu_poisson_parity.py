"""bt_grid_solve_poisson (zero-padded FFT convolution, cuFFT + this library's kernels, through the C-ABI) against the
oracle's direct O(N^2) sum (reading R19), and the closed space-charge step deposit -> solve -> gather/kick.

Tolerances.  The FFT convolution errs by ~ eps log2(8N) relative to max|phi| on every node:
|phi - ref| <= 1e-12 max|ref|.  The field differences neighbouring potentials, so that absolute error is divided by d:
|E - ref| <= 1e-12 max|phi| / min(d') per component (d' the rest-frame spacings), i.e. ~1e-10 max|E| on the grids below."""
import math

import numpy as np
import pytest

import oracle as O
import paper_2208_02382_b200 as bt
import workloads as W
from _util import r14_error

pytestmark = pytest.mark.gpu


def gpu_solve(rho, lo, d, gz):
    import ctypes
    import torch
    nz, ny, nx = rho.shape
    grid = bt.Grid((nx, ny, nz), lo, d)
    dev = torch.from_numpy(np.ascontiguousarray(rho)).cuda()
    torch.cuda.synchronize()
    ctypes.cdll.LoadLibrary("libcudart.so").cudaMemcpy(ctypes.c_void_p(grid.rho_ptr()), ctypes.c_void_p(dev.data_ptr()),
                                                      ctypes.c_size_t(8 * rho.size), 3)
    grid.solve_poisson(gz)
    phi, E = grid.download_phi(), grid.download_field()
    grid.close()
    return phi, E


def check(rho, d, gz):
    phi, E = gpu_solve(rho, (0.0, 0.0, 0.0), d, gz)
    ref = O.poisson(rho, d, gz)
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(phi - ref)) <= 1e-12 * scale
    Eref = O.efield(ref, d, gz)
    dmin = min(d[0], d[1], gz * d[2])
    for a, b in zip(E, Eref):
        assert np.max(np.abs(a - b)) <= 1e-12 * scale / dmin
    # the stencil applied to the device's own potential is reproduced to rounding
    Eself = O.efield(phi, d, gz)
    for a, b in zip(E, Eself):
        assert np.max(np.abs(a - b)) <= 1e-14 * scale / dmin
    return phi, E


@pytest.mark.parametrize("shape,d,gz", [((8, 8, 8), (1e-3, 1e-3, 1e-3), 1.0), ((20, 12, 28), (1e-3, 2e-3, 0.5e-3), 2.0657889247894516),
                                        ((32, 32, 32), (0.4e-3, 0.4e-3, 0.4e-3), 1.0), ((2, 3, 5), (1.0, 1.0, 1.0), 0.5)])
def test_poisson_matches_direct_sum(shape, d, gz):
    rng = np.random.default_rng(sum(shape))
    nx, ny, nz = shape
    rho = rng.uniform(-1e-12, 3e-12, (nz, ny, nx))
    rho[rng.uniform(size=rho.shape) < 0.3] = 0.0
    check(rho, d, gz)


@pytest.mark.parametrize("shape", [(32, 32, 32), (16, 24, 128), (40, 12, 32)])
def test_poisson_more_grid_shapes(shape):
    """Non-cubic grids with power-of-two and other plane counts; the 128-plane case on sampled nodes."""
    rng = np.random.default_rng(7)
    nx, ny, nz = shape
    rho = rng.uniform(-1e-12, 3e-12, (nz, ny, nx))
    rho[rng.uniform(size=rho.shape) < 0.5] = 0.0
    d, gz = (1e-3, 0.8e-3, 0.5e-3), 1.7
    if nz <= 32:
        check(rho, d, gz)
    else:
        phi, E = gpu_solve(rho, (0.0, 0.0, 0.0), d, gz)
        idx = rng.integers(0, rho.size, 64)
        ref = O.poisson_sample(rho, d, gz, idx)
        assert np.max(np.abs(phi.reshape(-1)[idx] - ref)) <= 1e-12 * np.max(np.abs(phi))


def test_point_charge_and_resolve_with_another_gz():
    """Coulomb potential of one node charge; the cached Green transform is rebuilt when gz changes."""
    rho = np.zeros((9, 10, 11))
    rho[4, 5, 6] = 1e-9
    d = (1e-3, 1e-3, 1e-3)
    K = 1.0 / (4.0 * math.pi * O.EPS0)
    for gz in (1.0, 3.0, 1.0):
        phi, _ = check(rho, d, gz)
        assert abs(phi[4, 5, 8] - K * 1e-9 / 2e-3) <= 1e-12 * phi.max()
        assert abs(phi[6, 5, 6] - K * 1e-9 / (2e-3 * gz)) <= 1e-12 * phi.max()


def test_full_size_grid_on_sampled_nodes():
    """configs[4] size: 128^3 nodes, rho deposited from 10^6 particles by the library; potential checked against the oracle's
    direct sum at 48 nodes (all 2.1e6 sources each)."""
    sc = W.spacecharge_config("A", n=1_000_000)
    c = W.make_spacecharge_bunch(sc)
    beam = bt.Beam(sc.n)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    beam.upload(c)
    beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
    gz = O.ref_from_kinetic(sc.kin_energy_MeV, sc.mass_MeV)[0]
    grid.solve_poisson(gz)
    rho, phi = grid.download_rho(), grid.download_phi()
    rng = np.random.default_rng(0)
    idx = np.concatenate([rng.integers(0, rho.size, 40), [0, rho.size - 1, (64 * 128 + 64) * 128 + 64, 127, 128 * 128 * 127, 12345, 999999, 2000000]])
    ref = O.poisson_sample(rho, sc.d, gz, idx)
    assert np.max(np.abs(phi.reshape(-1)[idx] - ref)) <= 1e-12 * np.max(np.abs(phi))
    E = grid.download_field()
    Eself = O.efield(phi, sc.d, gz)
    for a, b in zip(E, Eself):
        assert np.max(np.abs(a - b)) <= 1e-14 * np.max(np.abs(phi)) / min(sc.d)
    beam.close()
    grid.close()


@pytest.mark.parametrize("side_stream", [False, True])
def test_closed_space_charge_step_deposit_solve_gather(side_stream):
    """The paper's split-operator step with its own field (P:l.49): deposit -> Poisson (rest frame) -> gather + kick + drift,
    two steps, against the oracle chain.  The kick coefficients are the caller's (R12); any finite values test the plumbing.
    side_stream: the beam lives on a non-blocking side stream while the solve runs on the default stream -- the grid's
    operations must be ordered across the two (deposit -> solve -> gather hand the grid over with an event)."""
    import torch
    n, shape = (60_000, (24, 24, 24)) if not side_stream else (1_500_000, (48, 48, 48))   # long enough kernels to race
    sc = W.spacecharge_config("A", n=n, shape=shape)
    c = W.make_spacecharge_bunch(sc)
    g0 = O.ref_from_kinetic(sc.kin_energy_MeV, sc.mass_MeV)[0]
    coef = (2.0e-9, 2.0e-9, -1.0e-9)
    if side_stream:
        cs = torch.cuda.Stream()                     # torch side streams are non-blocking w.r.t. the default stream
        beam = bt.Beam(sc.n, storage="library", stream=cs.cuda_stream)
    else:
        beam = bt.Beam(sc.n)
    grid = bt.Grid(sc.shape, sc.lo, sc.d)
    beam.set_ref(sc.kin_energy_MeV, sc.mass_MeV, 1.0)
    beam.upload(c)
    beam.sort_by_cell(grid, sc.zscale)
    ref = [a.copy() for a in c]
    for step in range(2):
        beam.deposit_cic(grid, sc.q_weight, sc.zscale, True)
        grid.solve_poisson(g0)
        beam.gather_kick(grid, coef, sc.zscale, 0.0, sc.ds)
        rho, _ = O.deposit_cic(ref[0], ref[2], ref[4], sc.shape, sc.lo, sc.d, sc.q_weight, sc.zscale)
        E = O.efield(O.poisson(rho, sc.d, g0), sc.d, g0)
        O.gather_kick(ref, sc.shape, sc.lo, sc.d, E, coef, sc.zscale)
        O.track(ref, [("drift", sc.ds, 1)], 1, g0)
    got = beam.download()
    assert max(r14_error(got, ref)) <= 1e-11
    kick = np.max(np.abs(ref[1] - c[1]))
    assert kick > 1e-6 * np.sqrt(np.mean(c[1] ** 2))          # the space-charge kick is not negligible in this test
    beam.close()
    grid.close()


def test_poisson_argument_errors():
    grid = bt.Grid((4, 4, 4), (0, 0, 0), (1, 1, 1))
    assert bt.lib.bt_grid_solve_poisson(grid._h, 0.0, None) == bt.BT_ERR_INVALID
    assert bt.lib.bt_grid_solve_poisson(None, 1.0, None) == bt.BT_ERR_INVALID
    out = np.zeros(64)
    assert bt.lib.bt_grid_download_phi(grid._h, out.ctypes.data) == bt.BT_ERR_STATE
    assert bt.lib.bt_grid_download_field(grid._h, out.ctypes.data, out.ctypes.data, out.ctypes.data) == bt.BT_ERR_STATE
    grid.close()
