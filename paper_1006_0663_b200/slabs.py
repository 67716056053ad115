"""NEXT-4: r*-slab decomposition of one problem over several GPUs, one process per GPU.

The paper parallelises by domain decomposition.  Here every rank owns a contiguous range of r*
columns (all theta rows) and runs the ordinary step kernels on a WINDOW = owned columns + a halo of `halo` columns on
each cut side (a `teuk_create_slab` handle: same tables, bit for bit, as the full grid has there).  One iteration of
Eqs. (13)-(14) reaches one column in r*, and the window's edge columns are Dirichlet rows, so t
iterations after a refresh the columns within t of a cut edge are invalid while everything further in is exact.  With
halo = exchange_every + 2 the owned columns (and the observer's node column just beyond them) stay exact for
`exchange_every` iterations, after which each rank sends the `halo` owned columns next to each cut to that neighbour and
overwrites its own halos with what it receives - ONE neighbour exchange per `exchange_every` iterations (default 32 =
one CUDA-graph replay) instead of one or two per iteration: the messages are tiny (4 L n_theta halo doubles), so the
exchange is latency bound and is amortised over a whole graph; the price is 2 halo / owned redundant columns.

The only collective is point-to-point (`torch.distributed.batch_isend_irecv`: NCCL over NVLink between GPUs, gloo in
the CPU test); there is no all-reduce.  This module holds the index logic and the exchange; the stepping itself is
behind a three-method `stepper` (step, read_columns, write_columns) - `TeukStepper` wraps a slab handle of the CUDA
library.  It contains none of the method's arithmetic."""
from __future__ import annotations

from dataclasses import dataclass


@dataclass(frozen=True)
class Slab:
    rank: int
    world: int
    n_r: int          # global number of r* nodes
    lo: int           # owned global columns [lo, hi)
    hi: int
    wlo: int          # window (handle) global columns [wlo, whi)
    whi: int
    halo: int

    @property
    def n_win(self) -> int:
        return self.whi - self.wlo

    @property
    def owned_local(self) -> tuple:
        """(first local column, count) of the owned range inside the window"""
        return self.lo - self.wlo, self.hi - self.lo

    def outgoing(self) -> dict:
        """peer rank -> (first LOCAL column, count) of the owned strip that peer needs as its halo"""
        out = {}
        if self.rank > 0:
            out[self.rank - 1] = (self.lo - self.wlo, self.halo)
        if self.rank < self.world - 1:
            out[self.rank + 1] = (self.hi - self.halo - self.wlo, self.halo)
        return out

    def incoming(self) -> dict:
        """peer rank -> (first LOCAL column, count) of this window's halo that peer's strip overwrites"""
        inc = {}
        if self.rank > 0:
            inc[self.rank - 1] = (0, self.lo - self.wlo)
        if self.rank < self.world - 1:
            inc[self.rank + 1] = (self.hi - self.wlo, self.whi - self.hi)
        return inc


def plan(n_r: int, world: int, exchange_every: int = 32) -> list:
    """Balanced owned ranges (sizes differ by at most one), halo = exchange_every + 2 columns on each cut side."""
    if world < 1 or exchange_every < 1:
        raise ValueError("world >= 1 and exchange_every >= 1")
    halo = exchange_every + 2
    base, extra = divmod(n_r, world)
    if world > 1 and base < halo:
        raise ValueError(f"{n_r} columns over {world} ranks leaves {base} owned columns < halo {halo}: "
                         "lower exchange_every or use fewer ranks")
    slabs, lo = [], 0
    for r in range(world):
        hi = lo + base + (1 if r < extra else 0)
        slabs.append(Slab(r, world, n_r, lo, hi, max(0, lo - halo) if r > 0 else 0,
                          min(n_r, hi + halo) if r < world - 1 else n_r, halo))
        lo = hi
    return slabs


def owner_of_observer(slabs: list, w) -> int:
    """rank whose OWNED columns contain the lower observer node (its upper node is then inside that rank's valid halo)"""
    ro, _ = w.observer
    x = (ro - w.rstar_min) / w.dr
    i0 = min(int(x), w.n_r - 2)
    for s in slabs:
        if s.lo <= i0 < s.hi:
            return s.rank
    raise ValueError("observer outside the grid")


class TeukStepper:
    """slab handle of the CUDA library behind the stepper protocol"""

    def __init__(self, w, slab: Slab, options=None, obs_capacity=0, **kw):
        from . import teuk
        self.g = teuk.Teuk.from_workload(w, obs_capacity=obs_capacity, slab=(slab.wlo, slab.n_win), **kw)
        for k, v in (options or {}).items():
            self.g.set_option(k, v)

    def step(self, n):
        self.g.step(n)

    def read_columns(self, i_first, n_cols):
        return self.g.read_columns(i_first, n_cols)

    def write_columns(self, i_first, t):
        self.g.write_columns(i_first, t)


class SlabRun:
    """One rank's part of the run: step in chunks of at most `exchange_every`, exchange halos after every chunk."""

    def __init__(self, slab: Slab, stepper, dist=None, exchange_every: int = 32):
        if exchange_every + 2 > slab.halo:
            raise ValueError("exchange_every exceeds what the slab's halo allows")
        self.slab, self.stepper, self.dist, self.every = slab, stepper, dist, exchange_every
        self.exchanges = 0

    def step(self, n: int):
        while n > 0:
            k = min(n, self.every)
            self.stepper.step(k)
            self.exchange()
            n -= k

    def exchange(self):
        if self.slab.world == 1:
            return
        d = self.dist
        send = {p: self.stepper.read_columns(a, c) for p, (a, c) in self.slab.outgoing().items()}
        inc = self.slab.incoming()
        recv = {p: send[p].new_empty(send[p].shape[:3] + (c,)) for p, (a, c) in inc.items()}
        ops = [d.P2POp(d.isend, t, p) for p, t in sorted(send.items())] + \
              [d.P2POp(d.irecv, t, p) for p, t in sorted(recv.items())]
        for req in d.batch_isend_irecv(ops):
            req.wait()
        for p, (a, c) in inc.items():
            self.stepper.write_columns(a, recv[p])
        self.exchanges += 1

    def owned(self):
        a, c = self.slab.owned_local
        return self.stepper.read_columns(a, c)


def exchange_local(runs: list):
    """All slabs in ONE process (single-GPU test of the sharded path, no ranks waiting on one another): the same
    strips as SlabRun.exchange, moved by direct copies."""
    strips = {r.slab.rank: {p: r.stepper.read_columns(a, c) for p, (a, c) in r.slab.outgoing().items()} for r in runs}
    for r in runs:
        for p, (a, c) in r.slab.incoming().items():
            r.stepper.write_columns(a, strips[p][r.slab.rank])
        r.exchanges += 1


def step_local(runs: list, n: int):
    every = runs[0].every
    while n > 0:
        k = min(n, every)
        for r in runs:
            r.stepper.step(k)
        if len(runs) > 1:
            exchange_local(runs)
        n -= k
