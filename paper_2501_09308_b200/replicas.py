"""Host-side rank logic of a multi-GPU run (replicas only).

The path shards over independent sample-instances; north_star fixes one GPU per fit, so N GPUs run N
independent replicas (each rank fits its own restart of the same workload, own seeds) with NO data-path
collective.  The only communication is the timing barrier and the max-over-ranks of the device time,
through torch.distributed (NCCL on GPUs, gloo in the CPU tests).  No arithmetic of the method lives here.
"""
from __future__ import annotations


def replica_seeds(rank: int, base_seed: int = 1) -> dict:
    """What makes replica `rank` its own restart: `restart_offset` = rank shifts the restart index the R11 jitter is
    drawn for (xrdvi_reset_state_restart: rank > 0 starts from a jittered state even with one restart per handle),
    `state_seed` keys that jitter, `draw_seed` is the Philox key of the fit (xrdvi_fit).  Rank 0 with base_seed 1
    reproduces the single-GPU run (offset 0: no jitter)."""
    if rank < 0:
        raise ValueError("rank < 0")
    return {"state_seed": 0, "restart_offset": int(rank), "draw_seed": int(base_seed) + int(rank)}


def max_over_ranks(value: float, dist=None, device=None) -> float:
    """MAX all-reduce of one float64 (identity when not distributed)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, world: int, seconds_max: float) -> float:
    """Whole-job throughput: the units ALL ranks processed divided by the slowest rank's time."""
    if world < 1 or not seconds_max > 0:
        raise ValueError("world < 1 or non-positive time")
    return float(units_per_rank) * world / float(seconds_max)
