"""eta_s-slab decomposition of ONE event over several contexts / GPUs.

The stencil of a stage reaches two planes along eta_s (KT reconstruction), so a slab that carries two
ghost planes per interior side reproduces the undivided grid on its interior planes exactly, provided the ghost planes
hold the neighbours' data whenever a stage reads them: one point-to-point exchange of 2 planes x 19 words per neighbour
after EACH stage (stage 1 writes the state ' that stage 2 differentiates; stage 2 writes the state the next stage 1
differentiates).  The slab's own eta_s boundary is zero-gradient: what a stage computes IN the ghost planes is wrong and
is overwritten by the next exchange.  Host logic only -- every arithmetic step still runs in the library's kernels
(hydro_stage), the planes travel as opaque bytes (hydro_planes).

    plan = halo_plan(rank, nslab, nz, periodic)     pure bookkeeping (tested on CPU)
    s = Slab(cfg, eos, rank, nslab); s.load(T); s.step(n, exchange)   with exchange = exchange_dist (torch.distributed
        point-to-point, one process per GPU) or the closure made by exchange_local (several slabs in one process, used
        by the single-GPU test: the slabs run one after the other, no kernel ever waits on another)
"""
from __future__ import annotations

import dataclasses

import numpy as np

GHOST = 2


@dataclasses.dataclass(frozen=True)
class HaloPlan:
    k0: int            # first interior plane of this slab in the global grid
    k1: int            # one past the last
    g_lo: int          # ghost planes below / above the interior (0 or 2)
    g_hi: int
    lo: int            # neighbour ranks (-1: none)
    hi: int

    @property
    def nint(self):
        return self.k1 - self.k0

    @property
    def nz_local(self):
        return self.nint + self.g_lo + self.g_hi


def halo_plan(rank: int, nslab: int, nz: int, periodic: bool) -> HaloPlan:
    """Planes [k0, k1) of slab `rank` (sizes differ by at most one plane) and its neighbours."""
    if not (0 <= rank < nslab) or nslab < 1 or nz < GHOST * nslab:
        raise ValueError("need at least 2 interior planes per slab")
    base, rem = divmod(nz, nslab)
    k0 = rank * base + min(rank, rem)
    k1 = k0 + base + (1 if rank < rem else 0)
    wrap = periodic and nslab > 1
    lo = rank - 1 if rank > 0 else (nslab - 1 if wrap else -1)
    hi = rank + 1 if rank < nslab - 1 else (0 if wrap else -1)
    return HaloPlan(k0, k1, GHOST if lo >= 0 else 0, GHOST if hi >= 0 else 0, lo, hi)


def slab_planes(plan: HaloPlan, nz: int) -> np.ndarray:
    """Global plane index of every local plane (ghosts wrap around a periodic grid)."""
    return np.arange(plan.k0 - plan.g_lo, plan.k1 + plan.g_hi) % nz


def exchange_ops(plan: HaloPlan):
    """[(peer, send_k0, recv_k0)] in local plane indices, 2 planes each: to the lower neighbour go the two lowest interior
    planes and its two highest interior planes come back into the lower ghosts; likewise upwards."""
    ops = []
    if plan.lo >= 0:
        ops.append((plan.lo, plan.g_lo, 0))
    if plan.hi >= 0:
        ops.append((plan.hi, plan.g_lo + plan.nint - GHOST, plan.g_lo + plan.nint))
    return ops


class Slab:
    """One slab: a Hydro context on the local grid (nz_local planes, zero-gradient in eta_s)."""

    def __init__(self, cfg, eos, rank, nslab, **hydro_kw):
        from .hydro import from_config
        self.cfg, self.rank, self.nslab = cfg, rank, nslab
        periodic = cfg.bc[2] == 1
        self.plan = halo_plan(rank, nslab, cfg.nz, periodic)
        bc_eta = 1 if (periodic and nslab == 1) else 0
        self.local_cfg = dataclasses.replace(cfg, nz=self.plan.nz_local, bc=(cfg.bc[0], cfg.bc[1], bc_eta))
        self.h = from_config(self.local_cfg, eos, **hydro_kw)
        self.planes = slab_planes(self.plan, cfg.nz)

    def load(self, T, pi=None):
        """T [4, nz, ny, nx], pi [10, nz, ny, nx] of the WHOLE event (host arrays): the slab takes its planes and ghosts."""
        dt = self.h.np_dtype
        Tl = np.ascontiguousarray(np.asarray(T)[:, self.planes], dtype=dt)
        pl = None if pi is None else np.ascontiguousarray(np.asarray(pi)[:, self.planes], dtype=dt)
        self.h.load(Tl, pl)

    def step(self, n, exchange):
        """n RK2 steps; exchange(slab, which) fills the ghost planes of buffer `which` (1: state ', 0: the new state)."""
        for _ in range(n):
            self.h.stage(1)
            exchange(self, 1)
            self.h.stage(2)
            exchange(self, 0)

    def read_interior(self):
        e, u, pi = self.h.read()
        a, b = self.plan.g_lo, self.plan.g_lo + self.plan.nint
        return e[a:b], u[:, a:b], pi[:, a:b]


def exchange_dist(slab: Slab, which: int, host: bool = False):
    """Ghost-plane exchange between processes (one slab each) with torch.distributed point-to-point operations: NCCL on
    device tensors (host=False) or gloo on host tensors (host=True).  Both neighbours are served in one batch."""
    import torch
    import torch.distributed as dist
    # Posting order: [send towards lower, recv from upper, send towards upper, recv from lower].  With two slabs on a
    # periodic grid both neighbours are the same peer and messages between a pair are matched in posting order: the peer's
    # first message (its lowest interior planes, sent "towards lower") must meet my first receive (my UPPER ghosts).
    plan = slab.plan
    sends, recvs = {}, {}
    for peer, send_k0, recv_k0 in exchange_ops(plan):
        down = send_k0 == plan.g_lo                      # this pair of planes travels to the lower neighbour
        out = slab.h.planes_get(which, send_k0, GHOST, host=host)
        sends[down] = (peer, out)
        recvs[down] = (peer, recv_k0, torch.empty_like(out))      # ... and the lower neighbour's planes come back
    ops = []
    for down_send, down_recv in ((True, False), (False, True)):
        if down_send in sends:
            ops.append(dist.P2POp(dist.isend, sends[down_send][1], sends[down_send][0]))
        if down_recv in recvs:
            ops.append(dist.P2POp(dist.irecv, recvs[down_recv][2], recvs[down_recv][0]))
    if ops:
        for r in dist.batch_isend_irecv(ops):
            r.wait()
    for peer, recv_k0, inc in recvs.values():
        slab.h.planes_put(which, recv_k0, inc)


def exchange_local(slabs):
    """Several slabs in ONE process (the single-GPU test): returns exchange(slab, which) that, once every slab has
    finished the stage, copies the planes between the contexts.  The caller steps the slabs stage by stage through
    step_local below."""
    def run(which):
        boxes = {}
        for s in slabs:
            for peer, send_k0, _ in exchange_ops(s.plan):
                boxes[(s.rank, peer, send_k0 == s.plan.g_lo)] = s.h.planes_get(which, send_k0, GHOST)
        for s in slabs:
            for peer, send_k0, recv_k0 in exchange_ops(s.plan):
                # what the peer sent towards me: its message whose "towards lower" flag is the opposite of mine
                towards_lower = send_k0 == s.plan.g_lo          # I talk to my lower neighbour
                s.h.planes_put(which, recv_k0, boxes[(peer, s.rank, not towards_lower)])
    return run


def step_local(slabs, n):
    """n RK2 steps of all slabs in one process, stage by stage."""
    run = exchange_local(slabs)
    for _ in range(n):
        for s in slabs:
            s.h.stage(1)
        run(1)
        for s in slabs:
            s.h.stage(2)
        run(0)
