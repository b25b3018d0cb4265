"""Multi-GPU plumbing: walkers are independent, so the path shards by contiguous
walker ranges with the factor set replicated and NO data-path collective.  torch.distributed is used only for the
barrier and the max-over-ranks timing reduction of bench.py."""
from __future__ import annotations


def walker_shard(n_w: int, rank: int, world: int):
    """Contiguous walker range [lo, hi) of `rank` when n_w walkers are split over `world` ranks (strong scaling);
    sizes differ by at most one, lower ranks get the extra walker."""
    if not (0 <= rank < world) or n_w < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n_w, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar (e.g. the timed region's milliseconds); identity when not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
