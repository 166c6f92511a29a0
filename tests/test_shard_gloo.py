"""-m "not gpu": the N > 1 host logic (snapshot sharding, max-over-ranks timing) on world_size 2
with the gloo backend."""
from __future__ import annotations

import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

from paper_2512_06254_b200 import shard  # noqa: E402


def test_shard_partition_is_exact():
    for n in (0, 1, 7, 1500):
        for w in (1, 2, 3, 8):
            seen = sorted(i for r in range(w) for i in shard.snapshot_shard(n, r, w))
            assert seen == list(range(n))
            sizes = [len(shard.snapshot_shard(n, r, w)) for r in range(w)]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.snapshot_shard(4, 2, 2)


def test_reduce_timing_single_process():
    assert shard.reduce_timing(3.5, 10) == (3.5, 10.0)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = shard.snapshot_shard(11, rank, world)
        shard.barrier()
        t, u = shard.reduce_timing(10.0 * (rank + 1), len(mine))
        q.put((rank, list(mine), t, u))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert out[0][1] == [0, 2, 4, 6, 8, 10] and out[1][1] == [1, 3, 5, 7, 9]
    for _, _, t, u in out:
        assert t == 20.0 and u == 11.0          # max over ranks, sum over ranks
