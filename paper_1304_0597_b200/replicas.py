"""Multi-GPU harness for bench.py: N independent replicas of the GA problem, one per rank.

north_star fixes the hot path at one GPU, so there is no data-path collective:
each rank runs the same-shaped problem with its own seed and the only exchange is the max-over-ranks
of the timed region, as the bench contract requires.  Works on `nccl` (GPU box) and `gloo` (CPU tests).
"""
import os
from dataclasses import replace


def env_world():
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def replica_workload(w, rank):
    """Rank r evolves the same-shaped problem from a different seed (data and Philox key)."""
    return replace(w, seed=w.seed + 1000 * rank)


def max_over_ranks(value, world, device="cpu"):
    """MAX-reduce one float across ranks (the timed region's duration)."""
    if world == 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank, world, ms_local, device="cpu"):
    """Whole-job units/s: all ranks' units over the slowest rank's time."""
    ms = max_over_ranks(ms_local, world, device)
    return units_per_rank * world / (ms * 1e-3), ms
