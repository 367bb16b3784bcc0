"""Replicas-only multi-GPU plumbing: the path does not shard, so N ranks run N independent copies
of the job and the only cross-rank traffic is the timing scalar.  No data-path collective exists on purpose.

Used by bench.py (backend nccl, one rank per GPU) and by tests/test_replicas_gloo.py (backend gloo, CPU).
"""
from __future__ import annotations

import os


def env_rank_world_local():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def max_over_ranks(x: float, device=None) -> float:
    """MAX of a host scalar over all ranks (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank_step: float, steps: int, total_ms_local: float, device=None):
    """(value, ms_per_step): units all ranks processed / max-over-ranks time.  Weak scaling: every rank does
    `units_per_rank_step` per step."""
    import torch.distributed as dist
    world = dist.get_world_size() if (dist.is_available() and dist.is_initialized()) else 1
    total_ms = max_over_ranks(total_ms_local, device)
    ms_per_step = total_ms / max(1, steps)
    return world * units_per_rank_step / (ms_per_step * 1e-3), ms_per_step
