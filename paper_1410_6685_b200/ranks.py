"""Rank plumbing (torch.distributed only; no method arithmetic).

Replicas (the default of bench.py --gpus N): every rank runs the same fused pass on its own, independently seeded vectors
(weak scaling, SURVEY.md §8(e) / DESIGN.md §10); what the ranks exchange is the measurement itself: the job time is the MAX over
ranks of the device time, and the job throughput is the units all ranks processed over it.

Sharded collections (bench.py --shard): ONE collection split into contiguous index ranges, one per rank.
This module only says WHO owns WHAT and MOVES the per-rank partial results (at most 64 bytes per result and rank): index ranges,
the one-element overlap a neighbour predicate needs, an all-gather of small device tensors, the exclusive offsets of the filter
pieces.  Combining the gathered partials is arithmetic of the method and runs in the library (a pass over the W-element vector of
partials, workloads.cfg1_sharded) — or, in the CPU tests, in the oracle.
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


def shard_range(n: int, rank: int, world: int, overlap: int = 0) -> tuple[int, int]:
    """Rank `rank`'s contiguous index range [lo, hi) of an n-element collection: the first n % world ranks own one element more.
    overlap=1 extends the range by the first element of the next shard (clamped to n): the neighbour predicate x_i <= x_{i+1} of the
    pair that straddles the boundary is evaluated by the LEFT shard, so every pair is evaluated exactly once."""
    base, extra = divmod(n, world)
    lo = rank * base + min(rank, extra)
    hi = lo + base + (1 if rank < extra else 0)
    return lo, min(n, hi + overlap)


def all_gather_1d(t, dist=None):
    """All ranks' copies of a small 1-D tensor (the partial results of a sharded pass), concatenated in RANK ORDER on every rank —
    a fixed order, so the combine that follows is deterministic.  The tensor stays where it is (device tensors over NCCL, CPU tensors
    over gloo); nothing is reduced here."""
    import torch
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return t.clone()
    out = torch.empty(dist.get_world_size() * t.numel(), dtype=t.dtype, device=t.device)
    dist.all_gather_into_tensor(out, t.contiguous())
    return out


def exclusive_offsets(counts) -> list[int]:
    """Where each rank's piece of a sharded filter output starts in the concatenated result: the exclusive prefix sum of the kept
    counts (index bookkeeping, like shard_range)."""
    off, acc = [], 0
    for c in counts:
        off.append(acc)
        acc += int(c)
    return off
