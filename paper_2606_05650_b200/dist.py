"""Replica-parallel plumbing for multi-GPU runs (the codec is intra-only: frames are independent,
so N GPUs = N independent frame streams; no collective touches the data path).  torch.distributed is used only to
line ranks up and to reduce timings: works with nccl (GPU) and gloo (CPU tests)."""
from __future__ import annotations

import torch
import torch.distributed as dist


def frame_shard(n_frames: int, rank: int, world: int) -> range:
    """Frames handled by `rank`: a contiguous block, sizes differing by at most one, covering every frame once."""
    base, rem = divmod(n_frames, world)
    lo = rank * base + min(rank, rem)
    return range(lo, lo + base + (1 if rank < rem else 0))


def max_over_ranks(value: float, device="cpu") -> float:
    """Slowest rank's time (the job takes as long as its slowest replica)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def job_throughput(units_this_rank: float, ms_this_rank: float, device="cpu") -> float:
    """Whole-job units per second = all ranks' units / slowest rank's time."""
    total = sum_over_ranks(units_this_rank, device)
    ms = max_over_ranks(ms_this_rank, device)
    return total / (ms * 1e-3)
