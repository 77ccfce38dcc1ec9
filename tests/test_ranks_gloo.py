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


# ----------------------------------------------------------------------------------------------------------
# ONE collection sharded over the ranks.  On CPU the per-shard pass and the combine are the oracle's primitives
# (the library needs a GPU); what is under test is the plumbing the GPU path uses unchanged: the ranges, the one-element overlap of the
# neighbour predicate, the rank-ordered all-gather of the partials, the offsets of the filter pieces.
# ----------------------------------------------------------------------------------------------------------
def _shard_worker(rank: int, world: int, port: int, out):
    import oracle as orc
    from oracle import configs as ocfg
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        res = {}
        # config 1: sum / max of the fused chain over a sharded collection
        n = 100003
        lo, hi = ranks.shard_range(n, rank, world)
        x, y = inputs.normal_f32(2, 0, hi - lo, start=lo), inputs.normal_f32(2, 1, hi - lo, start=lo)      # a rank generates only its range
        part = ocfg.cfg1(x, y)
        sums = ranks.all_gather_1d(torch.tensor([part["sum"]], dtype=torch.float64), dist).numpy()
        maxs = ranks.all_gather_1d(torch.tensor([float(part["max"])], dtype=torch.float32), dist).numpy()
        res["cfg1"] = (orc.sum(sums), float(orc.max(maxs)))                                                   # the combine: a pass over the W partials
        # config 3: the violated pair straddles the shard boundary; the LEFT shard's one-element overlap sees it
        n3 = 50001
        xs = inputs.sorted_cumsum_f32(4, 0, n3)
        b = ranks.shard_range(n3, 0, world)[1]                          # first index of rank 1's range
        xs[b] = np.float32(0.5) * xs[b - 1]                             # breaks exactly the pair (b-1, b)
        lo3, hi3 = ranks.shard_range(n3, rank, world, overlap=1)
        loc = ocfg.cfg3(xs[lo3:hi3].copy())
        flags = ranks.all_gather_1d(torch.tensor([int(loc["pre"]), int(loc["post"])], dtype=torch.uint8), dist).numpy().reshape(world, 2)
        res["cfg3"] = (bool(orc.all(flags[:, 0])), bool(orc.all(flags[:, 1])), bool(loc["post"]))
        # config 2: local stable filters, all-gather of the counts -> offsets of the pieces in the concatenated result
        n2 = 70001
        xi = inputs.uniform_i31(3, 0, n2)
        lo2, hi2 = ranks.shard_range(n2, rank, world)
        piece = ocfg.cfg2(xi[lo2:hi2])
        counts = ranks.all_gather_1d(torch.tensor([piece["count"]], dtype=torch.int64), dist).tolist()
        psums = ranks.all_gather_1d(torch.tensor([piece["sum"]], dtype=torch.int64), dist).numpy()
        off = ranks.exclusive_offsets(counts)
        res["cfg2"] = (off[rank], piece["kept"].tolist(), counts, orc.sum(psums))
        dist.barrier()
        out.put((rank, res))
    finally:
        dist.destroy_process_group()


def test_sharded_collection_combines_to_the_unsharded_result_world_size_2():
    import oracle as orc
    from oracle import configs as ocfg
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_shard_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # ranges: a partition of [0, n); overlap adds exactly the next shard's first element
    for n in (0, 1, 2, 7, 100003):
        rs = [ranks.shard_range(n, r, 3) for r in range(3)]
        assert rs[0][0] == 0 and rs[-1][1] == n and all(rs[i][1] == rs[i + 1][0] for i in range(2))
        assert max(h - l for l, h in rs) - min(h - l for l, h in rs) <= 1
        assert [ranks.shard_range(n, r, 3, overlap=1)[1] for r in range(3)] == [min(n, h + 1) for _, h in rs]
    # config 1: every rank holds the same global results, equal to the oracle on the whole collection
    n = 100003
    whole = ocfg.cfg1(inputs.normal_f32(2, 0, n), inputs.normal_f32(2, 1, n))
    assert res[0]["cfg1"] == res[1]["cfg1"]
    gsum, gmax = res[0]["cfg1"]
    assert abs(gsum - whole["sum"]) <= 1e-12 * float(np.abs(whole["w"].astype(np.float64)).sum()) and np.float32(gmax) == whole["max"]
    # config 3: globally not sorted although rank 1's own range is; only the overlapping left shard sees the broken pair
    assert res[0]["cfg3"][:2] == res[1]["cfg3"][:2] == (True, False)
    assert res[0]["cfg3"][2] is False and res[1]["cfg3"][2] is True
    # config 2: the pieces, placed at their offsets, are the unsharded stable filter
    n2 = 70001
    want = ocfg.cfg2(inputs.uniform_i31(3, 0, n2))
    cat = [None] * want["count"]
    for r in range(world):
        o, kept, counts, total = res[r]["cfg2"]
        cat[o:o + len(kept)] = kept
        assert sum(counts) == want["count"] and total == want["sum"]
    assert cat == want["kept"].tolist()
    assert ranks.exclusive_offsets([3, 0, 5]) == [0, 3, 3]


def test_single_process_is_identity():
    assert torch.equal(ranks.all_gather_1d(torch.tensor([1.0, 2.0]), None), torch.tensor([1.0, 2.0]))
    assert ranks.shard_range(10, 0, 1) == (0, 10)
    assert ranks.max_over_ranks([1.5, 2.5], None) == [1.5, 2.5]
    assert ranks.rank_streams(0) == (0, 1)
