"""Host-side logic of the slab decomposition (paper_2508_08965_b200/slab.py): partition,
ring neighbours, periodic halo slices, and the message choreography of exchange_halos / global_min under torch.distributed
with the gloo backend, world sizes 2 and 3, on CPU.  The sub-domain here is a test double with the library's halo SEMANTICS
(pack = two outermost owned planes, unpack = two halo planes, a buffer of 80 * 2 * plane doubles); the order inside the buffer
is the double's own ([80][2][plane]) -- the library's is opaque and different (include/cgks.h), and slab.py never looks inside.
The kernels themselves are covered by tests/test_gpu_slab.py."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2508_08965_b200 import slab

NF = 80


class MockSub:
    """[80][nk_owned + 4][plane] on the CPU, same halo semantics as cgks_pack_halo / cgks_unpack_halo."""

    def __init__(self, k0, nk_owned, nk, plane):
        self.k0, self.nk_owned, self.plane = k0, nk_owned, plane
        kg = (torch.arange(k0 - 2, k0 + nk_owned + 2) % nk).double()
        f = torch.arange(NF).double()[:, None, None]; c = torch.arange(plane).double()[None, None, :]
        self.exact = 1000.0 * f + 10.0 * kg[None, :, None] + 0.001 * c          # value of (field, GLOBAL plane, cell)
        self.W = self.exact.clone()
        self.W[:, :2] = -1.0; self.W[:, -2:] = -1.0                               # halos unknown

    def halo_buffer(self):
        return torch.empty(NF * 2 * self.plane, dtype=torch.float64)

    def pack_halo(self, side, buf):
        k = self.nk_owned if side else 2                                         # nkl - 4 = nk_owned
        buf.copy_(self.W[:, k:k + 2].reshape(-1))

    def unpack_halo(self, side, buf):
        k = self.nk_owned + 2 if side else 0
        self.W[:, k:k + 2] = buf.view(NF, 2, self.plane)


def test_partition_and_neighbours():
    assert slab.partition(384, 8) == [(48 * r, 48) for r in range(8)]
    p = slab.partition(13, 3)
    assert p == [(0, 5), (5, 4), (9, 4)] and sum(c for _, c in p) == 13
    assert slab.partition(7, 1) == [(0, 7)]
    with pytest.raises(ValueError):
        slab.partition(5, 3)
    assert slab.neighbours(0, 4) == (3, 1) and slab.neighbours(3, 4) == (2, 0) and slab.neighbours(0, 1) == (0, 0)
    assert slab.neighbours(1, 2) == (0, 0)


def test_extended_wraps_periodically():
    a = torch.arange(2 * 7 * 3).double().view(2, 7, 3)
    e = slab.extended(a, 0, 3, 1)
    assert e.shape == (2, 7, 3)
    assert torch.equal(e[:, 0], a[:, 5]) and torch.equal(e[:, 1], a[:, 6]) and torch.equal(e[:, 2], a[:, 0]) and torch.equal(e[:, 6], a[:, 4])
    e = slab.extended(a, 5, 2, 1)
    assert torch.equal(e[:, 4], a[:, 0]) and torch.equal(e[:, 5], a[:, 1]) and torch.equal(e[:, 0], a[:, 3])


def test_local_exchange_fills_every_halo():
    nk, plane = 11, 6
    subs = [MockSub(k0, cnt, nk, plane) for k0, cnt in slab.partition(nk, 3)]
    slab.exchange_halos_local(subs)
    for s in subs:
        assert torch.equal(s.W, s.exact)
    one = MockSub(0, nk, nk, plane)
    slab.exchange_halos(one, 0, 1)                       # world of one: the slab is its own neighbour on both sides
    assert torch.equal(one.W, one.exact)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, nk, plane, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        k0, cnt = slab.partition(nk, world)[rank]
        s = MockSub(k0, cnt, nk, plane)
        # NCCL matches point-to-point messages between a pair of ranks by posting order and ignores tags (gloo honours them, so
        # this test cannot see a tag dependence directly): check instead that no exchange ever posts two messages in the same
        # direction to the same peer, and that every tag is overwritten with one value before posting
        posted = []
        real_batch = dist.batch_isend_irecv

        def spy(ops):
            posted.append(sorted((op.op.__name__, op.peer) for op in ops))
            for op in ops:
                op.tag = 7
            return real_batch(ops)
        dist.batch_isend_irecv = spy
        for _ in range(2):                               # twice: the exchange must be repeatable (stage 1, stage 2)
            s.W[:, :2] = -1.0; s.W[:, -2:] = -1.0
            slab.exchange_halos(s, rank, world)
            ok = torch.equal(s.W, s.exact)
        dist.batch_isend_irecv = real_batch
        unambiguous = all(len(set(p)) == len(p) for p in posted) and len(posted) == 2
        dt = slab.global_min(0.5 + 0.25 * ((rank + 1) % world), torch.device("cpu"))
        out[rank] = (bool(ok) and unambiguous, dt)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_exchange_and_dt_allreduce_gloo(world):
    mgr = mp.Manager(); out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), 13, 5, out), nprocs=world, join=True)
    assert len(out) == world
    for r in range(world):
        ok, dt = out[r]
        assert ok, "rank %d: halos wrong" % r
        assert dt == 0.5                                  # the minimum over ranks, identical on every rank
