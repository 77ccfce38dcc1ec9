"""Rank plumbing of the benchmark (torch.distributed only; no method arithmetic).

The hot path needs no data-path collective: every rank runs the same fused pass on its own, independently seeded
vectors (weak scaling, SURVEY.md §8(e) / DESIGN.md §10).  What the ranks exchange is the measurement itself: the job
time is the MAX over ranks of the device time, and the job throughput is the units all ranks processed over it.
"""
from __future__ import annotations

import os


def env_rank() -> tuple[int, int, int]:
    """(rank, local_rank, world_size) from the torchrun environment (1 process = 1 GPU)."""
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


def rank_streams(rank: int) -> tuple[int, int]:
    """Generator streams of rank r's x and y (config 1): (2r, 2r+1) — distinct data per rank, same distribution."""
    return 2 * rank, 2 * rank + 1


def max_over_ranks(values, dist=None, device="cpu"):
    """Element-wise max over ranks of a short list of floats (timings).  dist=None: single process."""
    import torch
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def job_throughput(units_per_rank: int, world: int, ms_max: float) -> float:
    """Whole-job units per second: all ranks' units over the slowest rank's time."""
    return world * units_per_rank / (ms_max * 1e-3)
