"""Multi-GPU plumbing: one process per GPU, frames sharded across ranks.

The render path has no exchange step: frames (camera, t) of a sweep are independent
(replicas only), so the scene is replicated, each rank renders its
own frames and no data-path collective exists. torch.distributed is used only for the
barrier around the timed region and the max-over-ranks of the measured time.

The optional within-frame split (`bench.py --split band`) is the one
place with an exchange: every rank renders a band of tile rows of the SAME frame
(Scene.set_tile_rows) and one all-gather of the bands assembles the image on every rank.
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


def band_rows(rank: int, world_size: int, tiles_y: int) -> Tuple[int, int]:
    """Tile rows [begin, end) of `rank`: contiguous bands whose heights differ by at most one row.
    With more ranks than rows the last ranks get an empty band (begin == end)."""
    base, extra = divmod(tiles_y, world_size)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def gather_bands(images, tiles_y: int, tile: int = 16):
    """All-gather of the image bands, in place: `images` are this rank's full-size tensors
    ([..., H, W], same device) of which only the pixel rows of its own band are valid; on return
    every rank holds the whole frame. One collective for all images: the bands are packed into
    one [C, rows, W] block per rank, padded to the tallest band."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return images
    rank, ws = dist.get_rank(), dist.get_world_size()
    H, W = images[0].shape[-2], images[0].shape[-1]
    planes = [im.reshape(-1, H, W) for im in images]          # views
    ch = sum(p.shape[0] for p in planes)
    bands = [band_rows(r, ws, tiles_y) for r in range(ws)]
    rows = [(min(b * tile, H), min(e * tile, H)) for b, e in bands]
    tallest = max(r1 - r0 for r0, r1 in rows)
    mine = torch.zeros((ch, tallest, W), dtype=images[0].dtype, device=images[0].device)
    r0, r1 = rows[rank]
    c = 0
    for p in planes:
        mine[c:c + p.shape[0], :r1 - r0] = p[:, r0:r1]
        c += p.shape[0]
    parts = [torch.empty_like(mine) for _ in range(ws)]
    dist.all_gather(parts, mine)
    for r, (q0, q1) in enumerate(rows):
        if r == rank or q1 <= q0:
            continue
        c = 0
        for p in planes:
            p[:, q0:q1] = parts[r][c:c + p.shape[0], :q1 - q0]
            c += p.shape[0]
    return images


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
