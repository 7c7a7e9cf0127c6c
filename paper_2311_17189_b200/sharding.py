"""Host logic of the one-process-per-GPU layout: samples are independent
(PAPER.md:113, :291), so the path shards over sample ranges with no data-path collective.  Only
timings and tallies cross ranks, through torch.distributed (NCCL on GPUs, gloo in the CPU tests)."""
from __future__ import annotations


def shard_range(n_total: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous sample range [first, first + count) of ``rank``: ranges tile [0, n_total) in rank
    order and differ in size by at most one (strong scaling of a fixed batch)."""
    if world < 1 or not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(n_total, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def weak_range(n_per_rank: int, rank: int, world: int) -> tuple[int, int]:
    """Weak scaling: every rank evaluates ``n_per_rank`` samples; rank r owns the counter range
    starting at r * n_per_rank of the counter-based generator (reading P22), so the union over
    ranks is the same sample stream a single process would draw."""
    if world < 1 or not (0 <= rank < world) or n_per_rank < 0:
        raise ValueError("bad shard request")
    return rank * n_per_rank, n_per_rank


def max_over_ranks(value: float, dist=None) -> float:
    """Device-timed durations are combined as the max over ranks."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(values, dist=None):
    """Sums a list of floats over ranks (sample counts, Monte-Carlo tallies re/im)."""
    vals = [float(v) for v in values]
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return vals
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor(vals, dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.tolist()]
