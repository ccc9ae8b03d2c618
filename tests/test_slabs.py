"""Host logic of the eta_s-slab decomposition (paper_1802_04449_b200/slabs.py) on CPU: the halo
bookkeeping, and the point-to-point exchange itself between two gloo ranks on a stand-in context whose "planes" carry
their global plane number (the GPU arithmetic is covered by tests/test_gpu_slabs.py)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1802_04449_b200 import slabs


@pytest.mark.parametrize("nslab,nz,periodic", [(1, 9, False), (1, 9, True), (2, 7, True), (2, 8, False), (3, 24, False),
                                               (3, 25, True), (4, 201, False), (8, 201, True)])
def test_halo_plan_covers_the_grid_and_messages_land_on_their_planes(nslab, nz, periodic):
    plans = [slabs.halo_plan(r, nslab, nz, periodic) for r in range(nslab)]
    # interiors tile [0, nz) in order; sizes differ by at most one plane
    assert plans[0].k0 == 0 and plans[-1].k1 == nz
    for a, b in zip(plans[:-1], plans[1:]):
        assert a.k1 == b.k0
    sizes = [p.nint for p in plans]
    assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 2
    # ghosts exist exactly where there is a neighbour; neighbours are mutual
    for r, p in enumerate(plans):
        assert (p.g_lo == 2) == (p.lo >= 0) and (p.g_hi == 2) == (p.hi >= 0)
        if p.lo >= 0:
            assert plans[p.lo].hi == r
        if p.hi >= 0:
            assert plans[p.hi].lo == r
        if not periodic or nslab == 1:
            assert (p.lo >= 0) == (r > 0) and (p.hi >= 0) == (r < nslab - 1)
    # every message: the global planes the sender reads are the global planes of the ghosts the receiver writes
    glob = [slabs.slab_planes(p, nz) for p in plans]
    for r, p in enumerate(plans):
        for peer, send_k0, recv_k0 in slabs.exchange_ops(p):
            down = send_k0 == p.g_lo
            peer_ops = {(k0 == plans[peer].g_lo): (pr, k0, r0) for pr, k0, r0 in slabs.exchange_ops(plans[peer])}
            pr, _, peer_recv = peer_ops[not down]          # the peer receives my message where IT talks the other way
            assert pr == r
            assert list(glob[r][send_k0:send_k0 + 2]) == list(glob[peer][peer_recv:peer_recv + 2])
            # and the planes I send are interior planes of mine
            assert p.g_lo <= send_k0 and send_k0 + 2 <= p.g_lo + p.nint
    with pytest.raises(ValueError):
        slabs.halo_plan(0, nz, nz, periodic)              # fewer than two interior planes per slab


class _FakeHydro:
    """Stand-in for a Hydro context: plane k of buffer `which` holds (1000 * which + global plane number)."""

    def __init__(self, planes):
        self.data = {w: np.array([1000.0 * w + g for g in planes]) for w in (0, 1)}

    def planes_get(self, which, k0, nk, host=False):
        return torch.from_numpy(self.data[which][k0:k0 + nk].copy()).view(torch.uint8)

    def planes_put(self, which, k0, buf):
        v = buf.view(torch.float64).numpy()
        self.data[which][k0:k0 + len(v)] = v


class _FakeSlab:
    def __init__(self, rank, nslab, nz, periodic):
        self.rank, self.plan = rank, slabs.halo_plan(rank, nslab, nz, periodic)
        self.planes = slabs.slab_planes(self.plan, nz)
        self.h = _FakeHydro(self.planes)
        # spoil the ghosts: the exchange must restore them
        for w in (0, 1):
            self.h.data[w][:self.plan.g_lo] = -1.0
            if self.plan.g_hi:
                self.h.data[w][-self.plan.g_hi:] = -1.0


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, nz, periodic, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    s = _FakeSlab(rank, world, nz, periodic)
    for which in (1, 0):
        slabs.exchange_dist(s, which, host=True)
    dist.barrier()
    out.put((rank, s.planes.tolist(), s.h.data[0].tolist(), s.h.data[1].tolist()))
    dist.destroy_process_group()


@pytest.mark.parametrize("periodic", [False, True])
def test_two_rank_exchange_restores_the_ghost_planes(periodic):
    """world_size 2 over gloo.  periodic = True is the case where both neighbours are the SAME peer and the two messages
    of a pair must not be swapped."""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, 11, periodic, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, planes, d0, d1 in res:
        assert d0 == [float(g) for g in planes], (rank, planes, d0)
        assert d1 == [1000.0 + g for g in planes], (rank, planes, d1)
