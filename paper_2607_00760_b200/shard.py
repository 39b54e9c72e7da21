"""Host-side logic of the N > 1 path.

Units (layer, request, KV head) are independent, so the path shards by request with no data-path
collective: every rank owns a disjoint set of requests, runs the same kernels on them, and the
only exchange is the max-over-ranks of the timed region plus a sum of the units processed.
Holds none of the method's arithmetic; works on any torch.distributed backend (NCCL on the GPUs,
gloo in the CPU tests).
"""
from dataclasses import replace


def shard_requests(n_requests: int, rank: int, world: int):
    """strong scaling: contiguous, near-equal split of a fixed request list; returns range(lo, hi)"""
    base, rem = divmod(n_requests, world)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


def rank_workload(w, rank: int):
    """weak scaling: every rank holds its own batch of w.batch requests, drawn from its own seed"""
    return replace(w, seed=w.seed + rank) if rank else w


def max_over_ranks(x: float, world: int, device="cpu") -> float:
    """timing rule: a multi-GPU number is the max over ranks of the device-timed region"""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, world: int, device="cpu") -> float:
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_this_rank: float, seconds_this_rank: float, world: int, device="cpu") -> float:
    """whole-job units/s = units all ranks processed / max-over-ranks time"""
    return sum_over_ranks(units_this_rank, world, device) / max_over_ranks(seconds_this_rank, world, device)
