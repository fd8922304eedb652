"""Rank bookkeeping for `bench.py --gpus N`: the path has no exchange step, so N
GPUs run N independent replicas of the workload; the only communication is a barrier and the
max-over-ranks of the device time.  Works on any torch.distributed backend (nccl on GPUs, gloo in the CPU
tests); holds none of the method's arithmetic."""
from __future__ import annotations


def replica_seed(base_seed: int, rank: int) -> int:
    """Every rank draws its own data set of the same shape (independent problems, weak scaling)."""
    return int(base_seed) + int(rank)


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """The step time of the job is the slowest rank's."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, dist=None, device="cpu") -> float:
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_rate(units_this_rank: float, ms_this_rank: float, dist=None, device="cpu") -> float:
    """Units all ranks processed / the slowest rank's time (units per second)."""
    total = sum_over_ranks(units_this_rank, dist, device)
    ms = max_over_ranks(ms_this_rank, dist, device)
    return total / (ms / 1e3)
