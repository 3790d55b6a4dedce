"""NEXT-4 host logic on CPU: slab partition arithmetic and the ghost-row exchange (paper_1812_00525_b200/slab.py),
in-process and through torch.distributed (gloo, world_size 2 and 3).  No kernels run here: a tensor-backed stand-in
with the get_rows / set_rows interface of the CUDA context plays the sub-domain."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1812_00525_b200 import slab

NPHI, NR = 3, 5


class FakeSlab:
    """Three 8-field buffers on the rows of an Extent; owned rows hold the global truth, ghost rows hold garbage."""

    def __init__(self, ext, truth):
        self.ext = ext
        self.buf = {}
        for b in (0, 1, 2):
            t = truth(b)[:, :, ext.z0:ext.z1].clone()
            ghost = torch.ones(ext.nZ_local, dtype=torch.bool)
            ghost[ext.a - ext.z0:ext.b - ext.z0] = False
            if ext.rank == 0:
                ghost[:2] = False                  # frozen boundary rows are never exchanged and stay as they are
            if ext.rank == ext.world - 1:
                ghost[-2:] = False
            t[:, :, ghost] = -777.0
            self.buf[b] = t

    def get_rows(self, buffer, k0, n, out):
        out.copy_(self.buf[buffer][:, :, k0:k0 + n])
        return out

    def set_rows(self, buffer, k0, n, src):
        self.buf[buffer][:, :, k0:k0 + n] = src


class FakePushSlab(FakeSlab):
    """The same stand-in with the direct hand-over of clt_push_rows (rows of one buffer straight into another slab's)."""

    def push_rows(self, buffer, k0, n, dst, k0_dst):
        dst.buf[buffer][:, :, k0_dst:k0_dst + n] = self.buf[buffer][:, :, k0:k0 + n]


def _truth(nZ):
    def f(b):
        g = torch.arange(nZ, dtype=torch.float64).view(1, 1, nZ, 1)
        m = torch.arange(8, dtype=torch.float64).view(8, 1, 1, 1)
        j = torch.arange(NPHI, dtype=torch.float64).view(1, NPHI, 1, 1)
        i = torch.arange(NR, dtype=torch.float64).view(1, 1, 1, NR)
        return 1000.0 * b + 100.0 * m + 10.0 * j + g + 0.01 * i
    return f


def _mk(_slab, n):
    return torch.empty((8, NPHI, n, NR), dtype=torch.float64)


def _check(fake, truth, buffer):
    ex = fake.ext
    want = truth(buffer)[:, :, ex.z0:ex.z1]
    got = fake.buf[buffer]
    lo = 2 if ex.rank == 0 else 0
    hi = ex.nZ_local - 2 if ex.rank == ex.world - 1 else ex.nZ_local
    # after an exchange every row of the local grid (ghost rows included) holds the global values, except the rows
    # 2..3 next to a cut that the kernels recompute and nobody reads: here all ghost rows are exchanged, so all match
    assert torch.equal(got[:, :, lo:hi], want[:, :, lo:hi])


@pytest.mark.parametrize("nZ,world", [(20, 1), (20, 2), (21, 3), (64, 4), (37, 8)])
def test_partition_and_extents(nZ, world):
    parts = slab.partition(nZ, world)
    assert parts[0][0] == 2 and parts[-1][1] == nZ - 2
    assert all(b - a >= slab.GHOST for a, b in parts)
    assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))
    assert max(b - a for a, b in parts) - min(b - a for a, b in parts) <= 1
    deep = []
    for r in range(world):
        ex = slab.Extent(nZ, world, r)
        assert ex.nZ_local >= 9 or world == 1
        k0, k1 = ex.owned_local()
        assert (k0 + ex.z0, k1 + ex.z0 + 1) == parts[r] and k0 >= 2 and k1 <= ex.nZ_local - 3
        d0, d1 = ex.deep_local()
        deep += list(range(d0 + ex.z0, d1 + ex.z0 + 1))
        if ex.upper is not None:
            up = slab.Extent(nZ, world, r + 1)
            # what I send up lands exactly on the neighbour's lower ghost rows (same global rows), and vice versa
            assert ex.send_up()[0] + ex.z0 == up.recv_from_lower()[0] + up.z0
            assert up.send_down()[0] + up.z0 == ex.recv_from_upper()[0] + ex.z0
    assert deep == list(range(4, nZ - 4))          # the global deep interior, each row exactly once


def test_partition_rejects_thin_slabs():
    with pytest.raises(ValueError):
        slab.partition(16, 4)


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_in_process(world):
    nZ = 29
    truth = _truth(nZ)
    exts = [slab.Extent(nZ, world, r) for r in range(world)]
    fakes = [FakeSlab(e, truth) for e in exts]
    for buffer in (1, 2, 0):
        slab.exchange(fakes, exts, buffer, None, _mk)
        for f in fakes:
            _check(f, truth, buffer)
    assert slab.STAGE_BUFFER == {1: 1, 2: 2, 3: 1, 4: 0}


@pytest.mark.parametrize("world", [2, 3, 4])
def test_exchange_in_process_by_direct_push(world):
    """slab.exchange hands ghost rows over through push_rows when the backend has it (the CUDA context does): same
    row arithmetic, no staging buffers (make_buffer must not be called)."""
    nZ = 37
    truth = _truth(nZ)
    exts = [slab.Extent(nZ, world, r) for r in range(world)]
    fakes = [FakePushSlab(e, truth) for e in exts]

    def no_buffers(_slab, _n):
        raise AssertionError("the push_rows path allocates no staging buffer")

    for buffer in (1, 2, 0):
        slab.exchange(fakes, exts, buffer, None, no_buffers)
        for f in fakes:
            _check(f, truth, buffer)


def test_thin_slabs_send_all_their_rows_both_ways():
    nZ, world = 4 + 12, 3                      # 12 interior rows -> three slabs of exactly GHOST rows
    exts = [slab.Extent(nZ, world, r) for r in range(world)]
    assert [e.b - e.a for e in exts] == [slab.GHOST] * 3
    mid = exts[1]
    assert mid.send_down() == mid.send_up() == (slab.GHOST, slab.GHOST)      # the same four rows go to both neighbours
    truth = _truth(nZ)
    fakes = [FakePushSlab(e, truth) for e in exts]
    slab.exchange(fakes, exts, 1, None, _mk)
    for f in fakes:
        _check(f, truth, 1)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nZ = 33
    truth = _truth(nZ)
    ex = slab.Extent(nZ, world, rank)
    fake = FakeSlab(ex, truth)
    ok = True
    try:
        for buffer in (1, 2, 1, 0):
            slab.exchange([fake], [ex], buffer, dist, _mk)
            _check(fake, truth, buffer)
    except AssertionError:
        ok = False
    q.put((rank, ok))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_gloo(world):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert out == [(r, True) for r in range(world)]
