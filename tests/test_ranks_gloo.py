"""The N>1 plumbing of bench.py on CPU: two processes, gloo backend, 127.0.0.1.  The hot path has no data-path collective
(independent problems per rank); what is exchanged is the timing (max over ranks) — DESIGN.md §10."""
from __future__ import annotations

import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1410_6685_b200 import inputs, ranks


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert ranks.env_rank() == (rank, rank, world)
        sx, sy = ranks.rank_streams(rank)
        x = inputs.normal_f32(2, sx, 1000)
        # each rank reports a different time; every rank must see the max
        mine = [10.0 + rank, 100.0 - rank]
        got = ranks.max_over_ranks(mine, dist, "cpu")
        dist.barrier()
        out.put((rank, got, float(x[:8].astype(np.float64).sum()), (sx, sy)))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_distinct_rank_data_world_size_2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [[11.0, 100.0], [11.0, 100.0]]        # max over ranks, on every rank
    assert res[0][3] == (0, 1) and res[1][3] == (2, 3)                    # distinct generator streams per rank
    assert res[0][2] != res[1][2]                                         # ... hence distinct data
    # whole-job throughput: all ranks' units over the slowest rank's time
    assert ranks.job_throughput(1 << 20, 2, 2.0) == 2 * (1 << 20) / 2e-3


def test_single_process_is_identity():
    assert ranks.max_over_ranks([1.5, 2.5], None) == [1.5, 2.5]
    assert ranks.rank_streams(0) == (0, 1)
