"""Host-side logic of the N > 1 path.

The D_w solve shards by right-hand side ("solution of this system for many right-hand sides"): every
rank holds the replicated gauge field and works on its own right-hand sides; there is no data-path collective.
Only the timing uses torch.distributed: a barrier on both sides of the timed region and the MAX over ranks of the
device time.  This module has no CUDA dependency, so the world_size-2 `gloo` tests on CPU cover it
(tests/test_sharding_gloo.py); bench.py uses the same functions under NCCL.
"""
from __future__ import annotations


def shard_rhs(nrhs: int, world: int, rank: int) -> list[int]:
    """Right-hand sides of `rank`: contiguous blocks, sizes differing by at most one, every index exactly once."""
    if nrhs < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError("shard_rhs: need nrhs >= 0, world >= 1, 0 <= rank < world")
    base, extra = divmod(nrhs, world)
    lo = rank * base + min(rank, extra)
    return list(range(lo, lo + base + (1 if rank < extra else 0)))


def rhs_seed(global_rhs: int, base_seed: int = 3) -> int:
    """Seed of the synthetic source of a right-hand side (DESIGN.md input recipe: sources seed 3 + rhs): depends on
    the GLOBAL index only, so a run on N ranks solves the same systems as a run on one."""
    return base_seed + int(global_rhs)


def max_over_ranks(x: float, dist=None, device=None) -> float:
    """MAX over ranks of a local scalar (device time); identity without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, seconds_local: float, dist=None, device=None) -> tuple[float, float]:
    """(units of ALL ranks) / (max over ranks of the local time).  Returns (rate, seconds_max).  The units are summed
    with an all-reduce, so ragged shards (nrhs not a multiple of the world size) are counted exactly."""
    sec = max_over_ranks(seconds_local, dist, device)
    total = float(units_per_rank)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        import torch
        t = torch.tensor([float(units_per_rank)], dtype=torch.float64, device=device if device is not None else "cpu")
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        total = float(t.item())
    return total / sec, sec
