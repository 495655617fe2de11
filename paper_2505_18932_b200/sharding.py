"""Multi-GPU plan for the geometry-guidance path: rays / target views are independent, so ranks take
independent target frames of the same rig ("weak" scaling: per-GPU work fixed) and the data path has NO
collective.  The only communication is the bench's barrier and the max-over-ranks reduction of the timed
region (torch.distributed; NCCL on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

import os
from typing import Dict, List, Tuple


def env_rank() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def frames_for_rank(rank: int, world: int, n_frames: int, base_stride: int = 10) -> List[int]:
    """Frame indices rank `rank` generates its inputs from.

    Every rank gets `n_frames` consecutive frames starting at rank * base_stride, so that (for C3) ranks
    draw different held-out target cameras and the job as a whole covers `world` independent target
    streams; the per-rank work (views, resolution, bins) is identical."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world %d" % (rank, world))
    start = rank * base_stride
    return list(range(start, start + n_frames))


def assign_targets(n_targets: int, rank: int, world: int) -> List[int]:
    """Round-robin split of a frame's target views (C5: 8 targets) over ranks; each target's persistent
    volume lives on exactly one rank."""
    return [t for t in range(n_targets) if t % world == rank]


def reduce_timing(elapsed_ms: float, units: float, device=None) -> Dict[str, float]:
    """max over ranks of the timed region, sum over ranks of the units processed."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return {"ms": float(elapsed_ms), "units": float(units), "world": 1}
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=device)
    u = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return {"ms": float(t.item()), "units": float(u.item()), "world": dist.get_world_size()}
