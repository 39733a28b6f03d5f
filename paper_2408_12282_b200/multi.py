"""Multi-GPU plumbing of the benchmark: one process per GPU, no data-path collective.

Frames (view, light) of the render path are independent: every rank holds
a replica of the scene and renders its own frames; the only communication is the reduction of the
timing (max over ranks) and a barrier around the timed region.  "Replicas only": there is no
exchange step in the method, so no collective is invented.  Works with the nccl backend on GPUs
and with gloo on CPU (tests/test_multi_rank.py, world size 2).
"""
from __future__ import annotations

import os
from typing import List, Optional, Tuple


def env_ranks() -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) as torchrun exports them; (0, 1, 0) when run directly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def frames_of_rank(n_views: int, rank: int, world: int) -> List[int]:
    """Views of a multi-view sweep owned by `rank`: round-robin by view, so that a rank keeps the
    per-view geometry (projection, sort, tile lists) of its frames to itself."""
    return [v for v in range(n_views) if v % world == rank]


def max_over_ranks(value: float, device=None) -> float:
    """Max of a per-rank scalar (device time of the timed region) over all ranks."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier() -> None:
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def whole_job_mpix_per_s(world: int, steps: int, frames_per_step: int, npix: int, max_ms: float) -> float:
    """Whole-job throughput: every rank rendered steps x frames_per_step frames of npix pixels
    (weak scaling), in max_ms milliseconds (max over ranks)."""
    return world * steps * frames_per_step * npix / (max_ms * 1e-3) / 1e6
