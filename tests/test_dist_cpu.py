"""N > 1 path of bench.py on CPU: world_size 2, gloo backend (rendezvous on 127.0.0.1)."""
import os
import socket

import pytest
import torch
import torch.multiprocessing as mp

from paper_2210_07912_b200 import dist_util


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    assert dist_util.env_world() == (rank, world, rank)
    dist_util.init("gloo")
    dist_util.barrier()
    ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slow one
    value, ms = dist_util.aggregate_throughput(1000, ms_local)
    ids = dist_util.shard_points(16, rank, world)
    out.put((rank, value, ms, ids[0], ids[-1]))
    dist_util.barrier()
    torch.distributed.destroy_process_group()


def test_world_size_two_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, ms, first, last in res:
        assert ms == 15.0                               # max over ranks
        assert abs(value - 2 * 1000 / 15e-3) < 1e-6     # whole-job units / max time
        assert (first, last) == (16 * rank, 16 * rank + 15)   # disjoint shards, no data-path collective


def test_single_process_defaults(monkeypatch):
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        monkeypatch.delenv(k, raising=False)
    assert dist_util.env_world() == (0, 1, 0)
    assert dist_util.max_over_ranks(3.5) == 3.5
    assert dist_util.aggregate_throughput(10, 2.0) == (5000.0, 2.0)
