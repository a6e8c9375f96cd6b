"""Band sharding for N > 1 GPUs.

Every band is an independent transform that shares one read-only plan ("the same offset
array can be used for all wavefunctions"; the paper itself splits the batch dimension once ranks
exceed the axis length).  So the path shards over BANDS: contiguous band ranges per
rank, plan tables and V(r) replicated, NO data-path collective.  The only communication is the
max-over-ranks of the measured time in benchmarks.
"""
from __future__ import annotations


def band_range(n_bands: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous [lo, hi) band range of `rank`; the first n_bands % world ranks get one band more."""
    if world < 1 or not (0 <= rank < world) or n_bands < 0:
        raise ValueError("bad sharding arguments")
    q, r = divmod(n_bands, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def max_over_ranks(value: float, device=None) -> float:
    """max of a per-rank scalar (timings) over the default process group; identity without one."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
