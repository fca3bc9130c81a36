"""Multi-rank host logic: one process per GPU, particles sharded by index, lattice and field
replicated.  bt_track and bt_gather_kick need NO communication (particles never interact: ranks
own particle subsets); the one exchange step of the method is the sum of the ranks' private charge grids after
bt_deposit_cic and before the field solve (one Poisson problem per bunch) -- `allreduce_rho`.

Plumbing only (torch.distributed: NCCL on GPUs, gloo in the CPU tests); no arithmetic of the method lives here.
"""
import os

__all__ = ["rank_world", "shard_bounds", "max_over_ranks", "allreduce_rho", "spacecharge_step"]


def rank_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) outside it."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def shard_bounds(n_total, rank, world):
    """Contiguous, disjoint, exhaustive particle ranges [lo, hi) whose sizes differ by at most one
    (strong scaling of ONE bunch: equal particle counts per rank, SURVEY 8e "load balance")."""
    if not (world >= 1 and 0 <= rank < world and n_total >= 0):
        raise ValueError("shard_bounds: need 0 <= rank < world and n_total >= 0")
    base, rem = divmod(int(n_total), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def _dist():
    import torch.distributed as dist
    return dist if (dist.is_available() and dist.is_initialized()) else None


def max_over_ranks(values, device=None):
    """Element-wise MAX of a short list of floats over all ranks (timings are reported as the slowest rank's)."""
    import torch
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist = _dist()
    if dist is not None and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def allreduce_rho(rho, always=False):
    """In-place SUM over ranks of the charge grid: `rho` is a bt.Grid (its device array is wrapped zero-copy and
    reduced by NCCL on the current stream -- 128^3 doubles = 16.8 MB over NVLink/NVSwitch) or any torch tensor
    (gloo in the CPU tests).  fp64 summation order across ranks is the collective's; R15 already accepts that.
    No-op at world size 1 unless always=True (bench.py: the collective is issued on the zero-copy view even in a
    one-rank group, so the path NCCL takes on device memory is exercised on a single GPU)."""
    dist = _dist()
    t = rho.rho_tensor() if hasattr(rho, "rho_tensor") else rho
    if dist is not None and (dist.get_world_size() > 1 or always):
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t


def spacecharge_step(deposit, allreduce, solve, gather, mark=None):
    """One closed space-charge step of the split-operator scheme as a rank of a sharded bunch runs it:
        deposit()    this rank's particles onto its private copy of the charge grid        (bt_deposit_cic)
        allreduce()  sum of the private grids over the ranks: the method's ONE collective (allreduce_rho)
        solve()      the bunch's single Poisson problem, solved redundantly on every rank  (bt_grid_solve_poisson)
        gather()     field at this rank's particles, kick, drift                           (bt_gather_kick)
    The four steps are the caller's callables -- the library's calls on a GPU, the oracle's functions in the CPU tests --
    so that the ORDER and the place of the collective are one piece of code for both.  mark(name), if given, is called after
    each phase (bench.py records a CUDA event there)."""
    for name, fn in (("deposit", deposit), ("allreduce", allreduce), ("solve", solve), ("gather", gather)):
        fn()
        if mark is not None:
            mark(name)
