"""Multi-GPU plumbing: one process per GPU, frames sharded across ranks.

The render path has no exchange step: frames (camera, t) of a sweep are independent
(replicas only), so the scene is replicated, each rank renders its
own frames and no data-path collective exists. torch.distributed is used only for the
barrier around the timed region and the max-over-ranks of the measured time.
"""
from __future__ import annotations

import os
from typing import List, Sequence, Tuple


def world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process if absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str = "nccl") -> Tuple[int, int, int]:
    rank, local_rank, ws = world()
    if ws > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29500")
            dist.init_process_group(backend=backend, rank=rank, world_size=ws)
    return rank, local_rank, ws


def frame_schedule(rank: int, world_size: int, steps: int, frames: Sequence) -> List:
    """Weak scaling: every rank renders `steps` frames; global frame f = step * world_size + rank
    walks the sweep round-robin, so the ranks together cover consecutive frames of the clip."""
    n = len(frames)
    return [frames[(s * world_size + rank) % n] for s in range(steps)]


def barrier(device=None) -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        if device is not None and dist.get_backend() == "nccl":
            dist.barrier(device_ids=[device])
        else:
            dist.barrier()


def max_over_ranks(value: float, device="cpu") -> float:
    """Max of a per-rank scalar (the timed region's duration) over all ranks."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device="cpu") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def shutdown() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
