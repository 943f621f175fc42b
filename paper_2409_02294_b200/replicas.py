"""Rank bookkeeping for multi-GPU runs: REPLICAS ONLY.

The path does not shard inside a solve (north_star: one GPU, no collectives); a batch of
independent fields is dealt round-robin to the ranks, each rank owning its own solver and its own
copy of the Green's-kernel spectrum.  There is no data-path collective: torch.distributed is used
only for the barrier around the timed region and the max-over-ranks of the device time.
Works with any backend (nccl on the GPUs, gloo in the CPU tests).  No arithmetic of the method here.
"""
from __future__ import annotations

import os


def dist_env():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)),
            int(os.environ.get("WORLD_SIZE", 1)))


def fields_of_rank(n_fields: int, rank: int, world: int) -> list:
    """Indices of the independent fields rank `rank` solves: round-robin, every field exactly once."""
    if world < 1 or not (0 <= rank < world) or n_fields < 0:
        raise ValueError(f"bad rank bookkeeping: n_fields={n_fields} rank={rank} world={world}")
    return list(range(rank, n_fields, world))


def barrier(world: int) -> None:
    if world > 1:
        import torch.distributed as dist
        dist.barrier()


def max_over_ranks(x: float, world: int, device="cpu") -> float:
    """MAX all-reduce of one float (the timing rule: a multi-GPU number is the slowest rank's)."""
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, world: int, device="cpu") -> float:
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(units_this_rank: float, ms_this_rank: float, world: int, device="cpu"):
    """Whole-job throughput: (units all ranks processed) / (slowest rank's time).
    Returns (units per second, ms of the slowest rank, total units)."""
    total = sum_over_ranks(units_this_rank, world, device)
    ms = max_over_ranks(ms_this_rank, world, device)
    return total * 1e3 / ms, ms, total
