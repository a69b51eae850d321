"""Multi-rank host logic on CPU: world_size-2 gloo.  The per-rank compute is the
oracle here (tests may use it); on GPUs it is the CUDA path (paper_2106_12631_b200.shard.gpu_compute)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2106_12631_b200 import shard


def test_event_range_is_a_partition():
    for n_total in (0, 1, 7, 1000, 2**20 + 3):
        for world in (1, 2, 3, 8):
            pos = 5
            for r in range(world):
                first, count = shard.event_range(r, world, n_total, first_event=5)
                assert first == pos and count >= 0
                pos += count
            assert pos == 5 + n_total
    with pytest.raises(ValueError):
        shard.event_range(2, 2, 10)


def _oracle_compute(process, seed):
    def compute(first, count):
        me, w = oracle.pipeline(process, seed, first, count, nthreads=1)
        return me.sum(), (me * me).sum(), (me * w).sum()
    return compute


def _worker(rank, world, port, n_total, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        res = shard.sharded_sums(_oracle_compute(1, 7), n_total, first_event=11)
        q.put((rank, res))
    finally:
        dist.destroy_process_group()


def test_two_ranks_reproduce_the_single_rank_sums():
    n_total = 2001     # odd: ranks get 1001 and 1000 events
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n_total, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = dict(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    single = shard.sharded_sums(_oracle_compute(1, 7), n_total, first_event=11, rank=0, world=1)
    for r in (0, 1):
        assert out[r][3] == n_total
        assert out[r][0] == pytest.approx(single[0], rel=1e-13)
        assert out[r][1] == pytest.approx(single[1], rel=1e-9)
        assert out[r][2] == pytest.approx(single[2], rel=1e-13)
    assert out[0] == out[1]
