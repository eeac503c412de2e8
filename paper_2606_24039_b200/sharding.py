"""Multi-GPU plumbing: the path shards by batch index with NO data-path collective (problems are
independent, PAPER.md:207-224 couples nothing across the batch).  One process per GPU; torch.distributed carries
only the barrier and the max-over-ranks reduction of the timings."""
from __future__ import annotations


def rank_problem_range(per_rank_batch: int, world: int, rank: int):
    """Weak scaling: rank r owns the global problem indices [r*B, (r+1)*B) of the seeded generator."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return rank * per_rank_batch, (rank + 1) * per_rank_batch


def split_batch(total: int, world: int, rank: int):
    """Strong scaling helper: contiguous near-equal split of `total` problems; returns (first, count)."""
    base, rem = divmod(total, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar (timings); identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
