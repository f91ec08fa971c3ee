"""Multi-GPU plumbing.

Default mode: REPLICAS ONLY.  The paper's system is single-GPU; at its sizes a particle-sharded swarm pays one exchange per
iteration that costs as much as it saves, so N GPUs run N independent sequences: `shard_start` says which stretch of the
seeded trajectory a rank tracks and `aggregate` combines per-rank device times and unit counts into one whole-job
number.  No data-path collective.

Particle-sharded mode (for config-4-scale swarms): `particle_slices` splits a level's template into
contiguous per-rank slices for Volume.pfo_track_sharded, whose only exchange is one all-gather of a 128-byte row per rank
and iteration.  Host logic only; the arithmetic is in rf_track.cu.
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


def particle_slices(n_total: int, world: int):
    """Contiguous, balanced slices of a template of n_total particles: [(offset, count)] per rank, in rank order; the first
    n_total % world ranks hold one particle more.  Every rank must hold at least one particle."""
    if world < 1 or n_total < world:
        raise ValueError("need at least one particle per rank")
    base, extra = divmod(n_total, world)
    out, off = [], 0
    for r in range(world):
        cnt = base + (1 if r < extra else 0)
        out.append((off, cnt))
        off += cnt
    return out


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
