"""NEXT-4 (r*-slab decomposition, paper_1006_0663_b200/slabs.py).

CPU: the index logic, and world_size-2 and -3 gloo runs whose per-rank stepper is an oracle window - the sharded run with
one halo exchange per `exchange_every` iterations must equal the full-grid oracle BIT FOR BIT on every owned column
(domain of dependence: r* reach of Eqs. 13-14 is one column per iteration).
GPU (one device, one process, slabs stepped one after another - no ranks waiting on one another): slab handles of the
CUDA library (teuk_create_slab + the column calls) against the full-grid handle, bit for bit, and against the oracle."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle import oracle
from paper_1006_0663_b200 import inputs, slabs


# ------------------------------------------------------------------------------------------------ index logic
@pytest.mark.parametrize("n_r,world,every", [(1000, 1, 32), (1000, 2, 32), (1001, 3, 16), (16384, 8, 32), (257, 4, 8)])
def test_plan_covers_the_grid_and_strips_match(n_r, world, every):
    pl = slabs.plan(n_r, world, every)
    assert [s.rank for s in pl] == list(range(world))
    assert pl[0].lo == 0 and pl[-1].hi == n_r and pl[0].wlo == 0 and pl[-1].whi == n_r
    for a, b in zip(pl, pl[1:]):
        assert a.hi == b.lo
    sizes = [s.hi - s.lo for s in pl]
    assert max(sizes) - min(sizes) <= 1
    for s in pl:
        assert s.halo == every + 2
        assert s.wlo == (0 if s.rank == 0 else s.lo - s.halo) and s.whi == (n_r if s.rank == world - 1 else s.hi + s.halo)
        for peer, (a, c) in s.outgoing().items():
            # what I send is exactly what the peer overwrites, in GLOBAL columns, and it lies in my owned range
            pa, pc = pl[peer].incoming()[s.rank]
            assert c == pc and s.wlo + a == pl[peer].wlo + pa
            assert s.lo <= s.wlo + a and s.wlo + a + c <= s.hi
        for peer, (a, c) in s.incoming().items():
            g0 = s.wlo + a
            assert g0 + c <= s.lo or g0 >= s.hi          # halos never overlap owned columns


def test_plan_rejects_slabs_thinner_than_the_halo():
    with pytest.raises(ValueError):
        slabs.plan(100, 4, 32)
    with pytest.raises(ValueError):
        slabs.SlabRun(slabs.plan(1000, 2, 8)[0], None, None, exchange_every=16)


# ------------------------------------------------------------------------------------------------ oracle stepper
class OracleStepper:
    """an oracle WINDOW behind the stepper protocol (tests only)"""

    def __init__(self, w, slab, L):
        self.o = oracle.Oracle.from_workload(w, precision=L, i_lo=slab.wlo, n_win=slab.n_win)

    def set_initial(self, u):
        self.o.set_initial(u)

    def step(self, n):
        self.o.step(n)

    def read_columns(self, a, c):
        return torch.from_numpy(np.ascontiguousarray(self.o.read()[..., a:a + c]))

    def write_columns(self, a, t):
        u = self.o.read()
        u[..., a:a + t.shape[-1]] = t.numpy()
        self.o.set_initial(u)


def _workload(n_r=220, n_t=10):
    w = inputs.config(2).scaled(n_r=n_r, n_theta=n_t, rstar_min=-30.0, rstar_max=60.0)
    return w.scaled(dt_override=inputs.stable_dt(w))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out, L, steps, every):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    oracle.set_threads(1)
    w = _workload()
    u0 = inputs.random_state(w.n_r, w.n_theta, L, seed=5)
    slab = slabs.plan(w.n_r, world, every)[rank]
    st = OracleStepper(w, slab, L)
    st.set_initial(np.ascontiguousarray(u0[..., slab.wlo:slab.whi]))
    run = slabs.SlabRun(slab, st, dist, exchange_every=every)
    for n in steps:
        run.step(n)
    torch.save({"lo": slab.lo, "hi": slab.hi, "u": run.owned(), "exchanges": run.exchanges}, f"{out}.{rank}")
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world,L,steps,every", [(2, 1, (40, 7), 16), (2, 2, (21,), 8), (3, 1, (25, 6), 8)])
def test_slab_run_equals_full_grid_oracle_gloo(tmp_path, world, L, steps, every):
    """world_size 2 and 3 (an interior rank exchanges with both neighbours), fp64 and dd, chunked step calls"""
    out = str(tmp_path / "slab")
    mp.spawn(_worker, args=(world, _free_port(), out, L, steps, every), nprocs=world, join=True)
    w = _workload()
    u0 = inputs.random_state(w.n_r, w.n_theta, L, seed=5)
    o = oracle.Oracle.from_workload(w, precision=L)
    o.set_initial(u0)
    o.step(sum(steps))
    ref = o.read()
    got = np.zeros_like(ref)
    for r in range(world):
        d = torch.load(f"{out}.{r}")
        got[..., d["lo"]:d["hi"]] = d["u"].numpy()
        assert d["exchanges"] == sum(-(-n // every) for n in steps)
    assert np.array_equal(got, ref)


def test_stale_halo_is_detected():
    """negative control: without the exchange the owned columns next to the cut go wrong after halo iterations"""
    w, L, every = _workload(), 1, 8
    u0 = inputs.random_state(w.n_r, w.n_theta, L, seed=5)
    pl = slabs.plan(w.n_r, 2, every)
    st = OracleStepper(w, pl[0], L)
    st.set_initial(np.ascontiguousarray(u0[..., pl[0].wlo:pl[0].whi]))
    o = oracle.Oracle.from_workload(w, precision=L)
    o.set_initial(u0)
    a, c = pl[0].owned_local
    st.step(every)
    o.step(every)
    assert np.array_equal(st.read_columns(a, c).numpy(), o.read()[..., pl[0].lo:pl[0].hi])
    st.step(every)
    o.step(every)
    assert not np.array_equal(st.read_columns(a, c).numpy(), o.read()[..., pl[0].lo:pl[0].hi])


# ------------------------------------------------------------------------------------------------ CUDA library
@pytest.mark.gpu
@pytest.mark.parametrize("L,world,steps,every,opts", [(1, 3, (64, 9), 32, {}), (1, 2, (33,), 16, {"time_block": 2}),
                                                      (2, 2, (24,), 8, {}), (4, 2, (10,), 4, {}),
                                                      (1, 2, (20,), 8, {"coef_variant": 1})])
def test_gpu_slabs_equal_full_grid_handle(L, world, steps, every, opts):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1006_0663_b200 import teuk
    w = _workload(n_r=400, n_t=20)
    total = sum(steps)
    u0 = inputs.random_state(w.n_r, w.n_theta, L, seed=11)
    obs = (12.3, 1.0)
    full = teuk.Teuk.from_workload(w, precision=L, obs_capacity=total)
    for k, v in opts.items():
        full.set_option(k, v)
    full.set_observer(obs[0], obs[1], total)
    full.set_initial(u0)
    full.step(total)
    ref = full.read()
    wo = w.scaled(rstar_obs=obs[0], theta_obs=obs[1], precision=L)
    pl = slabs.plan(w.n_r, world, every)
    owner = slabs.owner_of_observer(pl, wo)
    runs = []
    for s in pl:
        st = slabs.TeukStepper(wo, s, options=opts, obs_capacity=total if s.rank == owner else 0)
        if s.rank == owner:
            st.g.set_observer(obs[0], obs[1], total)
        st.g.set_initial(np.ascontiguousarray(u0[..., s.wlo:s.whi]))
        runs.append(slabs.SlabRun(s, st, None, exchange_every=every))
    for n in steps:
        slabs.step_local(runs, n)
    got = np.zeros_like(ref)
    for r in runs:
        got[..., r.slab.lo:r.slab.hi] = r.owned().cpu().numpy()
    assert np.array_equal(got, ref)
    assert np.array_equal(runs[owner].stepper.g.observe(total), full.observe(total))
    o = oracle.Oracle.from_workload(w, precision=L)
    o.set_initial(u0)
    o.step(total)
    assert max(oracle.rel_linf(got, o.read()).values()) <= {1: 1e-12, 2: 1e-27, 4: 1e-55}[L]


@pytest.mark.gpu
def test_gpu_slab_tables_and_argument_checks():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1006_0663_b200 import teuk
    w = _workload(n_r=300, n_t=12)
    full = teuk.Teuk.from_workload(w)
    part = teuk.Teuk.from_workload(w, slab=(37, 101))
    assert np.array_equal(part.tables(False), full.tables(False)[..., 37:138])
    assert np.array_equal(part.tables(True), full.tables(True)[..., 37:137])
    assert np.array_equal(part.radial()[0], full.radial()[0][74:275])
    with pytest.raises(teuk.TeukError):
        teuk.Teuk.from_workload(w, slab=(250, 101))
    with pytest.raises(teuk.TeukError):
        part.read_columns(0, 4)                      # before set_initial
    part.set_initial(inputs.random_state(101, w.n_theta, 1, seed=1))
    with pytest.raises(teuk.TeukError):
        part.read_columns(99, 4)
    with pytest.raises(teuk.TeukError):
        part.set_observer(-29.0, 1.0, 0)             # physical location outside this slab
    t = part.read_columns(5, 7)
    part.write_columns(20, t)
    assert torch.equal(part.read_columns(20, 7), t)
