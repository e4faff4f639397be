"""Multi-GPU plumbing: the path has no exchange step, so ranks only split the frame stream and agree on time.

Every (WFS, frame, subaperture) spot is independent (PAPER.md:91 describes a per-sensor, per-subaperture
computation; PAPER.md:119 expects a factor 4 from 4 GPUs).  One process per GPU takes whole frame batches of
the stream; nothing crosses NVLink on the data path, and the only collective is the MAX of the elapsed time
(torch.distributed; NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations


def rank_batches(n_batches: int, rank: int, world: int) -> list[int]:
    """Round-robin ownership of the batches of a frame stream: rank r owns r, r+world, ..."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return list(range(rank, n_batches, world))


def rank_frames(total_frames: int, batch: int, rank: int, world: int, which: int = 0) -> range:
    """Frame indices of the `which`-th batch owned by `rank` (wrapping round the stream for weak scaling)."""
    n_batches = max(total_frames // batch, 1)
    b = (rank + which * world) % n_batches
    return range(b * batch, min((b + 1) * batch, max(total_frames, batch)))


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a host scalar (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank_per_step: int, steps: int, elapsed_ms_max: float, world: int) -> float:
    """Whole-job units per second: every rank did `units_per_rank_per_step * steps` in the slowest rank's time."""
    return world * units_per_rank_per_step * steps / (elapsed_ms_max * 1e-3)
