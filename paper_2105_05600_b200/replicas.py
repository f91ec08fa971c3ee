"""Multi-GPU plumbing: REPLICAS ONLY.

The path does not shard across GPUs (the paper's system is single-GPU; a particle-sharded swarm would need one
all-reduce per iteration that costs as much as it saves at the paper's sizes), so N GPUs run N independent
sequences.  This module holds the host logic of that mode: which stretch of the seeded trajectory a rank tracks,
and how per-rank device times and unit counts combine into one whole-job number.  No data-path collective.
"""
from __future__ import annotations

from typing import Optional, Tuple


def shard_start(rank: int, n_frames: int, trajectory_len: int = 200, spacing: int = 23) -> int:
    """First frame of the stretch rank `rank` works on: ranks are spaced `spacing` frames apart along the seeded
    trajectory (wrapping so that a stretch of `n_frames` always fits)."""
    if n_frames > trajectory_len:
        raise ValueError("stretch longer than the trajectory")
    span = trajectory_len - n_frames
    return (rank * spacing) % span if span > 0 else 0


def aggregate(ms: float, units: float, group=None, device: Optional[str] = None) -> Tuple[float, float]:
    """Whole-job (time, units) from one rank's device time and unit count: MAX of the times, SUM of the units.
    Uses torch.distributed when a process group is initialised (nccl on GPUs, gloo in the CPU tests); a single
    process returns its own numbers."""
    import torch
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(ms), float(units)
    dev = device or ("cuda" if dist.get_backend(group) == "nccl" else "cpu")
    t = torch.tensor([float(ms)], dtype=torch.float64, device=dev)
    u = torch.tensor([float(units)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    dist.all_reduce(u, op=dist.ReduceOp.SUM, group=group)
    return float(t.item()), float(u.item())
