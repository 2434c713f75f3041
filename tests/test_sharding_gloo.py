"""world_size-2 gloo test of the N>1 host logic (column sharding, max-over-ranks timing)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2208_07129_b200 import inputs, sharding


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        t = sharding.max_over_ranks(1.0 + rank, dist)
        lo, hi = sharding.column_block(rank, world, 4)
        off = sharding.generator_offset(rank, 10, 4)
        x = inputs.uniform_pm1(7, off, 40)
        # every rank's block must be the matching slice of the global stream
        ref = inputs.uniform_pm1(7, 0, 40 * world)[off:off + 40]
        gathered = [None] * world
        dist.all_gather_object(gathered, (lo, hi))
        q.put((rank, t, (lo, hi), bool((x == ref).all()), gathered))
    finally:
        dist.destroy_process_group()


def test_two_rank_sharding_and_timing():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs: p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs: p.join(timeout=60)
    assert all(p.exitcode == 0 for p in procs)
    for rank, t, blk, same, gathered in res:
        assert t == 2.0                                    # max over ranks of (1, 2)
        assert blk == (4 * rank, 4 * rank + 4) and same
        assert gathered == [(0, 4), (4, 8)]                # disjoint cover of the 8 global columns
    assert sharding.aggregate_throughput(100, 2, 2.0) == 100.0


def test_split_columns_cover():
    for n, w in ((1024, 8), (10, 4), (3, 5)):
        r = [sharding.split_columns(n, w, k) for k in range(w)]
        assert r[0][0] == 0 and r[-1][1] == n and all(r[k][1] == r[k + 1][0] for k in range(w - 1))
    with pytest.raises(ValueError):
        sharding.column_block(2, 2, 4)
