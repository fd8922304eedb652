"""Rank bookkeeping.  The path has no exchange step: `bench.py --gpus N` runs N
independent replicas of the workload, the only communication a barrier and the max-over-ranks of the device
time; ONE problem can also be spread over GPUs by columns (`lambda_slice`, `gather_lambda_tables`; SURVEY.md
8(e)), the only communication the exchange of the fold-loss tables before lambda is selected.  Works on any
torch.distributed backend (nccl on GPUs, gloo in the CPU tests); holds none of the method's arithmetic."""
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


def lambda_slice(L: int, rank: int, world: int):
    """Indices of the lambda grid this rank fits: rank, rank + world, ... (interleaved, so that every rank gets
    its share of the small, slow lambdas).  May be empty only if world > L, which is refused."""
    import numpy as np
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    if world > L:
        raise ValueError("more ranks (%d) than lambda values (%d): shard bandwidths or data sets instead" % (world, L))
    return np.arange(rank, L, world)


def gather_lambda_tables(local, L: int, rank: int, world: int, dist=None, device="cpu"):
    """`local` [T, len(lambda_slice), V] of this rank -> the full [T, L, V] table on every rank (same dtype).
    Slices differ in length by at most one: they are padded to the longest for the all_gather."""
    import numpy as np
    local = np.ascontiguousarray(local)
    mine = lambda_slice(L, rank, world)
    T, Lr, V = local.shape
    if Lr != len(mine):
        raise ValueError("local table has %d lambda columns, this rank's slice has %d" % (Lr, len(mine)))
    full = np.empty((T, L, V), dtype=local.dtype)
    if world == 1:
        full[:] = local
        return full
    if dist is None or not dist.is_initialized() or dist.get_world_size() != world:
        raise RuntimeError("gather_lambda_tables: world > 1 needs an initialised process group of that size")
    import torch
    Lmax = (L + world - 1) // world
    pad = np.zeros((T, Lmax, V), dtype=local.dtype)
    pad[:, :Lr] = local
    send = torch.from_numpy(pad).to(device)
    recv = [torch.empty_like(send) for _ in range(world)]
    dist.all_gather(recv, send)
    for r in range(world):
        idx = lambda_slice(L, r, world)
        full[:, idx] = recv[r].cpu().numpy()[:, :len(idx)]
    return full
