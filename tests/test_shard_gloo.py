"""N > 1 host logic on CPU: two gloo ranks.  Particles are sharded by index; tracking needs no
exchange (checked: a shard tracked alone is bit-identical to the same particles tracked in the whole bunch); the
one exchange step is the sum of the ranks' private charge grids (paper_2208_02382_b200.shard.allreduce_rho)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank), OMP_NUM_THREADS="1")
    import oracle as O
    import workloads as W
    from paper_2208_02382_b200 import shard

    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert shard.rank_world() == (rank, rank, world)
        # ---- tracking shards independently ----
        cfg = W.config(0, n=2001)
        whole = W.make_bunch(cfg)
        lo, hi = shard.shard_bounds(cfg.n, rank, world)
        mine = [a[lo:hi].copy() for a in whole]
        g0 = O.ref_from_kinetic(cfg.kin_energy_MeV, cfg.mass_MeV)[0]
        O.track(mine, cfg.lattice, 2, g0)
        ref = [a.copy() for a in whole]
        O.track(ref, cfg.lattice, 2, g0)
        for a, b in zip(mine, ref):
            assert np.array_equal(a, b[lo:hi])
        # ---- deposit: private grids + one all-reduce == deposit of the whole bunch ----
        sc = W.spacecharge_config("A", n=30_001, shape=(16, 16, 16))
        c = W.make_spacecharge_bunch(sc)
        lo, hi = shard.shard_bounds(sc.n, rank, world)
        rho_mine, n_in_mine = O.deposit_cic(c[0][lo:hi], c[2][lo:hi], c[4][lo:hi], sc.shape, sc.lo, sc.d, sc.q_weight, sc.zscale)
        t = torch.from_numpy(rho_mine.copy())
        got = shard.allreduce_rho(t)
        assert got is t
        rho_all, n_in = O.deposit_cic(c[0], c[2], c[4], sc.shape, sc.lo, sc.d, sc.q_weight, sc.zscale)
        cnt = torch.tensor([float(n_in_mine)], dtype=torch.float64)
        dist.all_reduce(cnt)
        assert int(cnt.item()) == n_in
        r = t.numpy()
        assert np.array_equal(r == 0.0, rho_all == 0.0)
        nz = rho_all != 0.0
        assert np.max(np.abs(r[nz] - rho_all[nz]) / rho_all[nz]) <= 1e-12
        # ---- the closed space-charge step, driven through shard.spacecharge_step with the oracle standing in for the kernels:
        # two ranks, each with half the particles and a private grid == one rank with the whole bunch (R15 on rho, R14 after) ----
        sc = W.spacecharge_config("A", n=20_001, shape=(12, 12, 12))
        c = W.make_spacecharge_bunch(sc)
        coef = (2.0e-9, 2.0e-9, -1.0e-9)
        gsc = O.ref_from_kinetic(sc.kin_energy_MeV, sc.mass_MeV)[0]
        drift = [("drift", sc.ds, 1)]

        def run(coords, reduce_fn, rhos):
            st = {}

            def deposit():
                st["rho"] = torch.from_numpy(O.deposit_cic(coords[0], coords[2], coords[4], sc.shape, sc.lo, sc.d, sc.q_weight, sc.zscale)[0].copy())

            def solve():
                rho = st["rho"].numpy()
                rhos.append(rho.copy())
                st["E"] = O.efield(O.poisson(rho, sc.d, gsc), sc.d, gsc)

            def gather():
                O.gather_kick(coords, sc.shape, sc.lo, sc.d, st["E"], coef, sc.zscale)
                O.track(coords, drift, 1, gsc)

            phases = []
            for _ in range(2):
                shard.spacecharge_step(deposit, lambda: reduce_fn(st["rho"]), solve, gather, mark=phases.append)
            assert phases == ["deposit", "allreduce", "solve", "gather"] * 2
            return coords

        lo, hi = shard.shard_bounds(sc.n, rank, world)
        rhos_mine, rhos_whole = [], []
        mine = run([a[lo:hi].copy() for a in c], shard.allreduce_rho, rhos_mine)
        whole = run([a.copy() for a in c], lambda t: t, rhos_whole)          # one rank, the whole bunch, no collective
        for a, b in zip(rhos_mine, rhos_whole):
            assert np.all(np.abs(a - b) <= 1e-12 * np.maximum(b, sc.q_weight))     # R15 (ii)
        from _util import r14_error
        assert max(r14_error(mine, [a[lo:hi] for a in whole])) <= 1e-11             # R14
        assert np.max(np.abs(whole[1] - c[1])) > 0.0
        # ---- timing reduction: slowest rank ----
        assert shard.max_over_ranks([rank + 1.0, 5.0 - rank]) == [float(world), 5.0]
        assert W.rank_seed(1, rank) == 1 + 1000 * rank
        with open(os.path.join(out_dir, "ok%d" % rank), "w") as f:
            f.write("ok")
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_shard_track_and_allreduce_rho(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    assert all((tmp_path / ("ok%d" % r)).exists() for r in range(world))


@pytest.mark.parametrize("n,world", [(0, 1), (1, 2), (10, 3), (64_000_000, 8), (7, 8)])
def test_shard_bounds_partition(n, world):
    from paper_2208_02382_b200.shard import shard_bounds
    b = [shard_bounds(n, r, world) for r in range(world)]
    assert b[0][0] == 0 and b[-1][1] == n
    assert all(b[r][1] == b[r + 1][0] for r in range(world - 1))
    sizes = [hi - lo for lo, hi in b]
    assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_bounds(n, world, world)


def test_single_process_helpers_are_noops():
    from paper_2208_02382_b200 import shard
    t = torch.arange(4, dtype=torch.float64)
    assert shard.allreduce_rho(t) is t and t.tolist() == [0.0, 1.0, 2.0, 3.0]
    assert shard.max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
