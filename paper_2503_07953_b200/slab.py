"""Slab decomposition of the hot path along the last grid direction: one slab per process / GPU.

The paper populates its buffer regions across processes by message passing.  Here a slab is
an ordinary handle of the C-ABI library whose last direction has MFC_BC_HALO on the ends that touch a neighbour:
before every RHS evaluation the three layers next to each such end are packed (mfc_pack_halo, one strided
device copy per end), exchanged with the neighbours (NCCL send/recv through torch.distributed; a device copy when the
neighbour is the slab itself) and read by the sweep of that direction as its ghost cells; the sweeps of the other
directions run while the transfer is in flight (mfc_rk3_stage_parts).  Per RK3 step: three
exchanges of neq*3*plane doubles per end and one scalar MIN all-reduce for dt.  Everything else is the single-GPU path.

This module is host plumbing only (partition, neighbours, buffers, the exchange); all arithmetic runs in the kernels.
"""
import os
from dataclasses import replace

from . import BC_EXTRAP, BC_HALO, BC_PERIODIC, Grid

# MFC_SLAB_SYNC=1: host-synchronise behind the packing and behind the transfers instead of relying on stream events alone.
# The event ordering of the NCCL branch has been read, not run (no two-GPU box so far): this is the safe way out if a
# two-process run shows halos read before they have landed.
SYNC_FALLBACK = os.environ.get("MFC_SLAB_SYNC", "0") == "1"


def partition(n_last, world):
    """balanced split of n_last cells over `world` slabs: list of (start, count); every slab needs >= 3 cells"""
    base, rem = divmod(n_last, world)
    out, start = [], 0
    for r in range(world):
        cnt = base + (1 if r < rem else 0)
        out.append((start, cnt))
        start += cnt
    if min(c for _, c in out) < 3:
        raise ValueError(f"{n_last} cells over {world} slabs leaves a slab with fewer than 3 cells (the halo depth)")
    return out


def neighbours(rank, world, periodic):
    """(below, above) ranks along the last direction; None at a non-periodic end of the domain"""
    below = rank - 1 if rank > 0 else (world - 1 if periodic else None)
    above = rank + 1 if rank < world - 1 else (0 if periodic else None)
    return below, above


def local_case(case, rank, world):
    """the Case of slab `rank` of the global `case`: its share of the last direction, MFC_BC_HALO towards neighbours"""
    d = case.ndim - 1
    if case.ndim < 2:
        raise ValueError("slab decomposition needs a 2-D or 3-D grid")
    periodic = case.bc_lo[d] == BC_PERIODIC
    if periodic != (case.bc_hi[d] == BC_PERIODIC):
        raise ValueError("periodic must be set on both ends")
    start, cnt = partition(case.n[d], world)[rank]
    below, above = neighbours(rank, world, periodic)
    n = list(case.n)
    n[d] = cnt
    lo, hi = list(case.bc_lo), list(case.bc_hi)
    lo[d] = BC_HALO if below is not None else case.bc_lo[d]
    hi[d] = BC_HALO if above is not None else case.bc_hi[d]
    return replace(case, n=tuple(n), bc_lo=tuple(lo), bc_hi=tuple(hi)), start, cnt


def exchange(send_lo, send_hi, halo_lo, halo_hi, rank, below, above, dist=None, group=None, wait=True):
    """send_lo -> below's halo_hi, send_hi -> above's halo_lo; receive halo_lo <- below's send_hi, halo_hi <- above's send_lo.
    A neighbour equal to `rank` (one slab, periodic) is a local copy.  Posting order: with two slabs on a periodic domain both
    messages go to the same peer; it sends (send_lo, send_hi) in that order, so the receives are posted (halo_hi, halo_lo).
    wait=False returns the pending work handles (the caller waits on them before the sweep that reads the halos)."""
    ops = []
    if below == rank and above == rank:
        halo_lo.copy_(send_hi)
        halo_hi.copy_(send_lo)
        return []
    if below is not None:
        ops.append(dist.P2POp(dist.isend, send_lo, below, group))
    if above is not None:
        ops.append(dist.P2POp(dist.isend, send_hi, above, group))
    if above is not None:
        ops.append(dist.P2POp(dist.irecv, halo_hi, above, group))
    if below is not None:
        ops.append(dist.P2POp(dist.irecv, halo_lo, below, group))
    works = dist.batch_isend_irecv(ops) if ops else []
    if wait:
        for w in works:
            w.wait()
        return []
    return works


class Slab:
    """One process's slab: Grid + halo / send buffers + the exchange.  `case` is the GLOBAL case."""

    def __init__(self, case, rank=0, world=1, device=0, dist=None, group=None):
        import torch
        self.rank, self.world, self.dist, self.group = rank, world, dist, group
        self.case, self.start, self.count = local_case(case, rank, world)
        d = case.ndim - 1
        self.below, self.above = neighbours(rank, world, case.bc_lo[d] == BC_PERIODIC)
        # the stream the kernels of the handle run on (Grid takes torch's current stream of the device at construction)
        self.stream = torch.cuda.current_stream(device)
        self.grid = Grid.from_case(self.case, device=device, stream=self.stream.cuda_stream)
        plane = self.case.cells // self.case.n[d]
        n = self.case.neq * 3 * plane
        mk = lambda: torch.empty(n, dtype=torch.float64, device=f"cuda:{device}")
        self.halo_lo = mk() if self.below is not None else None
        self.halo_hi = mk() if self.above is not None else None
        self.send_lo = mk() if self.below is not None else None
        self.send_hi = mk() if self.above is not None else None
        self.grid.set_halo(self.halo_lo, self.halo_hi)
        self.exchanges = 0

    def pack(self, q, stage=1):
        """fills send_lo / send_hi from the state that stage `stage` sweeps"""
        if self.send_lo is not None or self.send_hi is not None:
            self.grid.pack_halo(q, stage, self.send_lo, self.send_hi)

    def refresh(self, q, stage=1, wait=True):
        """ghost layers of the state that stage `stage` sweeps (stage 1: q).  wait=False: returns the pending transfers"""
        if self.below is None and self.above is None:
            return []
        import torch
        cur = torch.cuda.current_stream(self.stream.device)
        if cur != self.stream:
            # whatever produced q was enqueued on the caller's current stream: the handle's stream (packing, sweeps) follows it
            ev = torch.cuda.Event()
            ev.record(cur)
            self.stream.wait_event(ev)
        self.pack(q, stage)
        if SYNC_FALLBACK:
            self.stream.synchronize()
        if self.below == self.rank and self.above == self.rank:
            # one periodic slab, its own neighbour: the two local copies run on the handle's stream, between the packing and
            # the sweep that reads the halos — ordered by the stream itself, whatever the caller's current stream is
            with torch.cuda.stream(self.stream):
                exchange(self.send_lo, self.send_hi, self.halo_lo, self.halo_hi, self.rank, self.below, self.above,
                         self.dist, self.group, wait=False)
            self.exchanges += 1
            return []
        # the packed buffers must be complete before NCCL reads them: NCCL's stream waits for the CURRENT stream when the
        # transfers are posted, so the current stream is made to wait for an event recorded behind the packing — the
        # host is not stalled (no synchronize; three per step in round 1)
        if cur != self.stream:
            ev = torch.cuda.Event()
            ev.record(self.stream)
            cur.wait_event(ev)
        works = exchange(self.send_lo, self.send_hi, self.halo_lo, self.halo_hi, self.rank, self.below, self.above,
                         self.dist, self.group, wait=False)
        self.exchanges += 1
        if wait:
            self._wait(works)
            return []
        return works

    def rhs(self, q, out):
        self.refresh(q, 1)
        self.grid.rhs(q, out)

    def rk3_step(self, q, dt):
        """per stage: start the halo exchange, run the sweeps that need no halo while it is in flight, wait, run the last
        sweep (which reads the halos and applies the RK stage)"""
        for stage in (1, 2, 3):
            works = self.refresh(q, stage, wait=False)
            self.grid.rk3_stage(q, dt, stage, parts=1)
            self._wait(works)
            self.grid.rk3_stage(q, dt, stage, parts=2)

    def _wait(self, works):
        """NCCL work.wait() makes the current stream wait for the transfer (no host stall); the handle's stream follows it"""
        if not works:
            return
        import torch
        for w in works:
            w.wait()
        cur = torch.cuda.current_stream(self.stream.device)
        if SYNC_FALLBACK:
            cur.synchronize()
        if cur != self.stream:
            ev = torch.cuda.Event()
            ev.record(cur)
            self.stream.wait_event(ev)

    def cfl_dt(self, q, cfl):
        """global dt: the minimum over slabs of the local one (one scalar all-reduce)"""
        dt = self.grid.cfl_dt(q, cfl)
        if self.world > 1:
            import torch
            t = torch.tensor([dt], dtype=torch.float64, device=q.device)
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MIN, group=self.group)
            dt = float(t.item())
        return dt

    def advance(self, q, cfl, nsteps):
        t = 0.0
        for _ in range(nsteps):
            dt = self.cfl_dt(q, cfl)
            self.rk3_step(q, dt)
            t += dt
        return t

    def close(self):
        self.grid.close()
