"""Multi-GPU plumbing: one process per GPU, frames partitioned across ranks.

The path shards over independent frames (steps x sensor instances): each rank
owns a sensor handle on its own GPU and a contiguous block of frames; no
data-path collective is needed (the paper's "multiple GPUs ...
in the same system").  torch.distributed is used only to agree
on timing (max over ranks) and, when a caller wants all results in one place,
to gather them.  Works with the nccl backend on GPUs and gloo on CPU (tests).
"""
from __future__ import annotations

from typing import List, Tuple

import torch
import torch.distributed as dist

from .workloads import shard_range


def my_frames(n_frames: int) -> Tuple[int, int]:
    """[lo, hi) of the frames this rank processes (whole batch if not distributed)."""
    if dist.is_available() and dist.is_initialized():
        return shard_range(n_frames, dist.get_rank(), dist.get_world_size())
    return 0, n_frames


def max_over_ranks(value: float, device: torch.device | str = "cpu") -> float:
    """Timing rule: a multi-GPU step takes as long as its slowest rank."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_frames(local: torch.Tensor, n_frames: int) -> List[torch.Tensor] | None:
    """Collect every rank's [hi-lo, ...] block on rank 0 in frame order (results
    normally stay where their inputs were; this is for callers that want one array)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [local]
    world, rank = dist.get_world_size(), dist.get_rank()
    sizes = [shard_range(n_frames, r, world) for r in range(world)]
    biggest = max(hi - lo for lo, hi in sizes)
    pad = torch.zeros((biggest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: local.shape[0]] = local
    bufs = [torch.empty_like(pad) for _ in range(world)] if rank == 0 else None
    dist.gather(pad, bufs, dst=0)
    if rank != 0:
        return None
    return [b[: hi - lo] for b, (lo, hi) in zip(bufs, sizes)]
