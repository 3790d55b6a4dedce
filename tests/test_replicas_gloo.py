"""The N > 1 path of bench.py ("replicas only") on CPU: world_size 2, gloo backend."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1812_00525_b200 import replicas
    assert replicas.world() == (rank, world)
    replicas.barrier("cpu")
    # rank r processed (r+1)*1000 units in (r+1)*0.5 s: job = 3000 units in max(0.5, 1.0) s
    units, secs, rate = replicas.aggregate((rank + 1) * 1000.0, (rank + 1) * 0.5)
    q.put((rank, units, secs, rate))
    dist.destroy_process_group()


def test_aggregate_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, units, secs, rate in out:
        assert units == 3000.0 and secs == 1.0 and rate == 3000.0


def test_aggregate_single_process():
    from paper_1812_00525_b200 import replicas
    assert replicas.world() == (0, 1)
    assert replicas.aggregate(10.0, 2.0) == (10.0, 2.0, 5.0)
