"""GPU parity tests (pin P10): the CUDA path through the C ABI (paper_1006_0663_b200.teuk) against the
oracle (oracle/) element by element on the same seeded inputs.  Tolerances are BASELINE.json's relative
L-infinity bounds (reading A17): 1e-12 fp64, 1e-27 dd, 1e-55 qd."""
import math
import os

import numpy as np
import pytest

from oracle import mp_ref, oracle
from paper_1006_0663_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = {1: 1e-12, 2: 1e-27, 4: 1e-55}


@pytest.fixture(scope="module")
def teuk():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1006_0663_b200 import teuk as t
    return t


def run_gpu(teuk, w, u0, steps, precision=None, observer=None, options=None):
    L = precision or w.precision
    g = teuk.Teuk.from_workload(w, precision=L, obs_capacity=steps if observer else 0)
    for k, v in (options or {}).items():
        g.set_option(k, v)
    if observer:
        g.set_observer(observer[0], observer[1], steps)
    g.set_initial(u0)
    g.step(steps)
    return g


def run_oracle(w, u0, steps, precision=None, observer=None, i_lo=0, n_win=None):
    o = oracle.Oracle.from_workload(w, precision=precision or w.precision, i_lo=i_lo, n_win=n_win)
    if observer:
        o.set_observer(observer[0], observer[1], steps)
    o.set_initial(u0)
    o.step(steps)
    return o


def series_err(a, b):
    """observer series [n][4][L]: max over samples of |F_gpu - F_ref| / max |F_ref| per complex field"""
    a4 = np.ascontiguousarray(np.transpose(a, (1, 2, 0)))
    b4 = np.ascontiguousarray(np.transpose(b, (1, 2, 0)))
    return oracle.rel_linf(a4, b4)


# ------------------------------------------------------------------------------- arithmetic layer on device
@pytest.mark.parametrize("L", [2, 4])
@pytest.mark.parametrize("op", ["add", "sub", "mul", "div", "sqrt", "mul_d"])
def test_device_arithmetic_bitwise_equals_host_build(teuk, L, op):
    rng = np.random.default_rng(7 + L)
    n = 4096
    a = rng.uniform(0.5, 2.0, size=(n, L)) * (2.0 ** (-54.0 * np.arange(L)))[None, :] * rng.choice([-1, 1], size=(n, L))
    b = rng.uniform(0.5, 2.0, size=(n, L)) * (2.0 ** (-54.0 * np.arange(L)))[None, :] * rng.choice([-1, 1], size=(n, L))
    if op == "sqrt":
        a[:, 0] = np.abs(a[:, 0])
    b[::3] = -a[::3] * (1 + 2.0 ** -70)                       # cancellation rows
    host = teuk.test_mp_op(op, L, a, b, on_device=False)
    dev = teuk.test_mp_op(op, L, a, b, on_device=True)
    assert np.array_equal(host, dev)


# ------------------------------------------------------------------------------- setup: r(r*) and tables
@pytest.mark.parametrize("cfg", [1, 2, 4])
def test_radial_inversion_matches_mpmath(teuk, cfg):
    import mpmath as mp
    w = inputs.config(cfg).scaled(n_r=257)
    g = teuk.Teuk.from_workload(w)
    r, d = g.radial()
    with mp.workdps(110):
        lo = mp.mpf(w.rstar_min)
        dr = (mp.mpf(w.rstar_max) - lo) / (w.n_r - 1)
        for k in (0, 1, 2, 17, 128, 255, 400, 512):
            rr, dd = mp_ref.r_of_rstar(lo + k * dr / 2, w.M, w.a)
            assert abs(mp_ref.from_limbs(r[k]) - rr) / rr < mp.mpf(10) ** -58
            assert abs(mp_ref.from_limbs(d[k]) - dd) / dd < mp.mpf(10) ** -58, (k, mp.nstr(dd, 5))


@pytest.mark.parametrize("cfg,L", [(1, 1), (2, 1), (2, 2), (4, 4)])
def test_coefficient_tables_match_oracle(teuk, cfg, L):
    w = inputs.config(cfg).scaled(n_r=129)
    g = teuk.Teuk.from_workload(w, precision=L)
    o = oracle.Oracle.from_workload(w, precision=L)
    eps = {1: 2.0 ** -52, 2: 2.0 ** -102, 4: 2.0 ** -198}[L]
    for half in (False, True):
        tg, to = g.tables(half), o.tables(half)
        for q in range(8):
            diff, _ = oracle._limb_diff(tg[q], to[q])
            scale = np.maximum(np.abs(to[q, 0]).ravel(), np.abs(to[:, 0]).max(axis=0).ravel() / 64)
            assert np.all(np.abs(diff) <= 8 * eps * scale), (half, q, float(np.max(np.abs(diff) / scale)))


# ------------------------------------------------------------------------------- full runs on small / ragged grids
def test_config1_full_run_fp64(teuk):
    w = inputs.config(1)
    u0 = inputs.initial_state(w)
    g = run_gpu(teuk, w, u0, w.steps, observer=w.observer)
    o = run_oracle(w, u0, w.steps, observer=w.observer)
    err = oracle.rel_linf(g.read(), o.read())
    print("cfg1 final-state error", err)
    assert max(err.values()) <= TOL[1]
    serr = series_err(g.observe(w.steps), o.observe(w.steps))
    print("cfg1 observer error", serr)
    assert max(serr.values()) <= TOL[1]
    assert g.steps_done() == w.steps


@pytest.mark.parametrize("L,n_r,n_t,steps,base", [(1, 203, 13, 300, 2), (2, 203, 13, 200, 2), (4, 131, 11, 80, 2),
                                                  (2, 300, 40, 60, 4), (4, 150, 32, 40, 4), (1, 1000, 70, 100, 2)])
def test_ragged_grids_all_precisions(teuk, L, n_r, n_t, steps, base):
    """sizes that span several tiles with ragged tails in both directions; generic complex state with
    every field and limb populated; Kerr coefficients (cfg 2 physics) or cfg 4 physics"""
    w0 = inputs.config(base)
    lo, hi = -30.0, 60.0
    w = w0.scaled(n_r=n_r, n_theta=n_t, rstar_min=lo, rstar_max=hi, precision=L)
    w = w.scaled(dt_override=inputs.stable_dt(w))
    u0 = inputs.random_state(n_r, n_t, L, seed=100 + L)
    obs = (10.3, 1.1)
    g = run_gpu(teuk, w, u0, steps, observer=obs)
    o = run_oracle(w, u0, steps, observer=obs)
    err = oracle.rel_linf(g.read(), o.read())
    serr = series_err(g.observe(steps), o.observe(steps))
    print(L, n_r, n_t, "state", err, "observer", serr)
    assert max(err.values()) <= TOL[L]
    assert max(serr.values()) <= TOL[L]


@pytest.mark.parametrize("ti,tj", [(8, 4), (32, 16), (64, 8), (16, 64)])
def test_tile_shapes_give_identical_results(teuk, ti, tj):
    w = inputs.config(2).scaled(n_r=150, n_theta=24, rstar_min=-30.0, rstar_max=60.0, precision=2)
    w = w.scaled(dt_override=inputs.stable_dt(w))
    u0 = inputs.random_state(w.n_r, w.n_theta, 2, seed=9)
    ref = run_gpu(teuk, w, u0, 30).read()
    got = run_gpu(teuk, w, u0, 30, options={"tile_i": ti, "tile_j": tj}).read()
    assert np.array_equal(ref, got)


@pytest.mark.parametrize("n_r,n_t", [(203, 13), (512, 16), (1000, 70), (40, 3)])
def test_tma_kernel_matches_generic_kernel_fp64(teuk, n_r, n_t):
    """the fp64 TMA kernel (default) and the generic kernel run the same arithmetic; compiler FMA contraction
    may differ between the two instantiations, so compare to a few ulps, and both against the oracle"""
    w = inputs.config(2).scaled(n_r=n_r, n_theta=n_t, rstar_min=-30.0, rstar_max=60.0)
    w = w.scaled(dt_override=inputs.stable_dt(w))
    u0 = inputs.random_state(n_r, n_t, 1, seed=21)
    outs = {}
    for name, opts in (("tma16", {}), ("tma8", {"tile_j": 8}), ("generic", {"use_tma": 0})):
        g = run_gpu(teuk, w, u0, 64, options=opts, observer=(10.3, 1.1))
        outs[name] = (g.read(), g.observe(64), g.step_geometry())
    assert outs["tma16"][2]["tile_j"] == 16 and outs["tma8"][2]["tile_j"] == 8
    o = run_oracle(w, u0, 64, observer=(10.3, 1.1))
    ref, sref = o.read(), o.observe(64)
    for name, (u, ser, _) in outs.items():
        assert max(oracle.rel_linf(u, ref).values()) <= TOL[1], name
        assert max(series_err(ser, sref).values()) <= TOL[1], name
    assert max(oracle.rel_linf(outs["tma16"][0], outs["generic"][0]).values()) <= 1e-14
    assert np.array_equal(outs["tma16"][0], outs["tma8"][0])


# ------------------------------------------------------------------------------- NEXT-3: two iterations per launch (fp64)
@pytest.mark.parametrize("n_r,n_t,steps", [(203, 13, 64), (512, 16, 65), (1000, 70, 37), (40, 3, 8), (33, 17, 21), (97, 64, 50)])
@pytest.mark.parametrize("m,s", [(2, -2), (1, -1)])
def test_time_blocked_kernel_fp64(teuk, n_r, n_t, steps, m, s):
    """time_block=2 (step2_kernel_f64_tma: two iterations of Eqs. 13-14 per launch, u^{n+1} only in shared memory)
    against the oracle and against the single-step kernel, on ragged grids, odd step counts (the last iteration falls to
    the single-step kernel), both tile heights, even and odd |m| (ghost sign), with the observer sampled every step"""
    w = inputs.config(2).scaled(n_r=n_r, n_theta=n_t, rstar_min=-30.0, rstar_max=60.0, m=m, s=s)
    w = w.scaled(dt_override=inputs.stable_dt(w))
    u0 = inputs.random_state(n_r, n_t, 1, seed=33)
    obs = (10.3, 1.1)
    one = run_gpu(teuk, w, u0, steps, observer=obs)
    outs = {}
    for name, opts in (("tb16", {"time_block": 2}), ("tb8", {"time_block": 2, "tile_j": 8}),
                       ("tb16_nograph", {"time_block": 2, "graph_steps": 0}), ("tb16_g2", {"time_block": 2, "graph_steps": 2})):
        g = run_gpu(teuk, w, u0, steps, options=opts, observer=obs)
        outs[name] = (g.read(), g.observe(steps))
        assert g.steps_done() == steps
    o = run_oracle(w, u0, steps, observer=obs)
    ref, sref = o.read(), o.observe(steps)
    for name, (u, ser) in outs.items():
        assert ser.shape[0] == steps, name
        assert max(oracle.rel_linf(u, ref).values()) <= TOL[1], name
        assert max(series_err(ser, sref).values()) <= TOL[1], name
        # same arithmetic as the single-step kernel (FMA contraction may differ between instantiations: a few ulps)
        assert max(oracle.rel_linf(u, one.read()).values()) <= 1e-14, name
    assert np.array_equal(outs["tb16"][0], outs["tb8"][0])
    assert np.array_equal(outs["tb16"][0], outs["tb16_nograph"][0])
    assert np.array_equal(outs["tb16"][0], outs["tb16_g2"][0])
    assert np.array_equal(outs["tb16"][1], outs["tb16_g2"][1])


def test_time_blocked_kernel_split_calls_and_invariants(teuk):
    """teuk_step called in odd pieces equals one call; Dirichlet rows stay exactly zero; a = 0, s = m = 0 reflection
    symmetry stays bit-exact; time_block=2 is refused where it does not exist (dd, theta_order 10, recompute supply)"""
    w = inputs.config(1).scaled(n_r=600, n_theta=24)      # omega dt = 0.5: inside the stability bound (reading A15b)
    u0 = inputs.initial_state(w)
    a = run_gpu(teuk, w, u0, 101, options={"time_block": 2})
    b = teuk.Teuk.from_workload(w)
    b.set_option("time_block", 2)
    b.set_initial(u0)
    for n in (1, 2, 33, 64, 1):
        b.step(n)
    ua, ub = a.read(), b.read()
    assert np.array_equal(ua, ub)
    assert not ua[:, :, :, 0].any() and not ua[:, :, :, -1].any()
    assert np.array_equal(ua, ua[:, :, ::-1, :])
    o = run_oracle(w, u0, 101)
    assert max(oracle.rel_linf(ua, o.read()).values()) <= TOL[1]
    g = teuk.Teuk.from_workload(w, precision=2)
    with pytest.raises(teuk.TeukError):
        g.set_option("time_block", 2)
    for bad in ({"theta_order": 10}, {"coef_variant": 1}, {"use_tma": 0}):
        g = teuk.Teuk.from_workload(w)
        g.set_option("time_block", 2)
        for k, v in bad.items():
            g.set_option(k, v)
        with pytest.raises(teuk.TeukError):
            g.set_initial(u0)


def test_time_blocked_config2_prefix_full_grid(teuk):
    """config 2 at full size in the bench launch geometry, time_block=2, 1000-step prefix vs the full-grid oracle"""
    w = inputs.config(2)
    u0 = inputs.initial_state(w)
    steps = 1000
    g = run_gpu(teuk, w, u0, steps, observer=w.observer, options={"time_block": 2})
    o = run_oracle(w, u0, steps, observer=w.observer)
    err = oracle.rel_linf(g.read(), o.read())
    print("cfg2 prefix, time_block=2", err)
    assert max(err.values()) <= TOL[1]
    serr = series_err(g.observe(steps), o.observe(steps))
    assert max(serr.values()) <= TOL[1] or np.abs(o.observe(steps)).max() < 1e-300


# ------------------------------------------------------------------------------- semi-recompute coefficient supply (H1b)
@pytest.mark.parametrize("cfg", [1, 2])
def test_recomputed_coefficients_match_stored_planes(teuk, cfg):
    """coef_variant 1 rebuilds the folded coefficients from one 1/Sigma plane + 1-D tables; they must agree with
    the stored planes (rounded from quad-double) to a few ulps of the largest coefficient at the point"""
    w = inputs.config(cfg).scaled(n_r=257)
    g = teuk.Teuk.from_workload(w)
    for half in (False, True):
        a, b = g.folded(half, 0), g.folded(half, 1)
        scale = np.abs(a).max(axis=0, keepdims=True)
        rel = np.abs(a - b) / np.maximum(np.abs(a), scale / 16)
        assert rel.max() <= 16 * 2.0 ** -52, (half, float(rel.max()), np.unravel_index(rel.argmax(), rel.shape))
        # variant (c), full recompute: 1/Sigma = rsqrt(R^2 - a^2 Delta sin^2 theta) in fp64 enters up to the third power
        c = g.folded(half, 2)
        relc = np.abs(a - c) / np.maximum(np.abs(a), scale / 16)
        print("cfg", cfg, "half", half, "max ulps (b)", float(rel.max()) * 2.0 ** 52, "(c)", float(relc.max()) * 2.0 ** 52)
        assert relc.max() <= 32 * 2.0 ** -52, (half, float(relc.max()), np.unravel_index(relc.argmax(), relc.shape))


@pytest.mark.parametrize("n_r,n_t,base,m", [(203, 13, 2, 2), (512, 16, 1, 0), (1000, 70, 2, 2), (40, 3, 2, 2), (3, 2, 2, 1),
                                             (31, 2, 2, 2), (61, 5, 2, 1), (32, 9, 2, 2), (30, 4, 2, 1)])
def test_recompute_kernel_parity_fp64(teuk, n_r, n_t, base, m):
    """semi-recompute supply on the column-march kernel (whole columns, automatic and odd work-unit lengths) and on the TMA
    tile kernel, full recompute on the tile kernel; ragged and degenerate grids (3 columns, 2 rows, strips of exactly 30
    and 30 + 1 + 1 columns), even and odd |m|"""
    w = inputs.config(base).scaled(n_r=n_r, n_theta=n_t, rstar_min=-30.0, rstar_max=60.0, m=m)
    w = w.scaled(dt_override=inputs.stable_dt(w))
    u0 = inputs.random_state(n_r, n_t, 1, seed=33)
    o = run_oracle(w, u0, 200, observer=(10.3, 1.1))
    ref, sref = o.read(), o.observe(200)
    for opts in ({"coef_variant": 1}, {"coef_variant": 1, "march_chunk": n_t}, {"coef_variant": 1, "march_chunk": min(3, n_t)},
                 {"coef_variant": 1, "march": 0}, {"coef_variant": 1, "march": 0, "tile_j": 8},
                 {"coef_variant": 2}, {"coef_variant": 2, "tile_j": 8}):
        g = run_gpu(teuk, w, u0, 200, options=opts, observer=(10.3, 1.1))
        err = oracle.rel_linf(g.read(), ref)
        serr = series_err(g.observe(200), sref)
        print(n_r, n_t, opts, err, serr)
        assert max(err.values()) <= TOL[1] and max(serr.values()) <= TOL[1]


def test_recompute_kernel_config2_prefix(teuk):
    w = inputs.config(2)
    u0 = inputs.initial_state(w)
    steps = 1000
    o = run_oracle(w, u0, steps)
    for cv in (1, 2):
        g = run_gpu(teuk, w, u0, steps, options={"coef_variant": cv})
        err = oracle.rel_linf(g.read(), o.read())
        print("cfg2 1000-step prefix, recompute supply", cv, ":", err)
        assert max(err.values()) <= TOL[1]
    with pytest.raises(teuk.TeukError):
        teuk.Teuk.from_workload(inputs.config(3).scaled(n_r=64)).set_option("coef_variant", 1)   # fp64 only


# ------------------------------------------------------------------------------- NEXT-1: 10th-order theta operator
@pytest.mark.parametrize("L,n_r,n_t,steps,base", [(1, 203, 13, 200, 2), (2, 203, 13, 100, 2), (4, 131, 11, 40, 2),
                                                  (1, 300, 64, 100, 2), (2, 150, 32, 40, 4), (4, 90, 32, 20, 4),
                                                  (1, 64, 5, 50, 2)])
def test_theta10_parity_all_precisions(teuk, L, n_r, n_t, steps, base):
    """10th-order angular operator, rest of the scheme unchanged; column kernel vs oracle"""
    w = inputs.config(base).scaled(n_r=n_r, n_theta=n_t, rstar_min=-30.0, rstar_max=60.0, precision=L)
    w = w.scaled(dt_override=0.5 * inputs.stable_dt(w))       # the wide stencil's largest eigenvalue is ~1.7x larger
    u0 = inputs.random_state(n_r, n_t, L, seed=200 + L)
    obs = (10.3, 1.1)
    g = run_gpu(teuk, w, u0, steps, observer=obs, options={"theta_order": 10})
    o = oracle.Oracle.from_workload(w, theta_order=10)
    o.set_observer(obs[0], obs[1], steps)
    o.set_initial(u0)
    o.step(steps)
    err = oracle.rel_linf(g.read(), o.read())
    serr = series_err(g.observe(steps), o.observe(steps))
    print("theta10", L, n_r, n_t, err, serr)
    assert max(err.values()) <= TOL[L] and max(serr.values()) <= TOL[L]
    # the option is live: the 2nd-order kernel gives a different answer
    g2 = run_gpu(teuk, w, u0, steps)
    assert not np.array_equal(g2.read(), g.read())


@pytest.mark.parametrize("n_r,n_t,m", [(203, 13, 2), (300, 64, 2), (64, 5, 1), (1000, 70, 2), (2100, 30, 1), (40, 6, 2), (17, 9, 1)])
def test_theta10_fp64_tma_column_kernel(teuk, n_r, n_t, m):
    """fp64 theta_order=10 defaults to the TMA column kernels (semi-recompute supply): the row-run kernel (8- and 16-column
    tiles; N_theta not a multiple of the run length, runs that straddle both poles, odd |m|), the point-per-thread kernel
    at all its tile widths and the generic column kernel must agree with the oracle"""
    w = inputs.config(2).scaled(n_r=n_r, n_theta=n_t, rstar_min=-30.0, rstar_max=60.0, m=m)
    w = w.scaled(dt_override=0.5 * inputs.stable_dt(w))
    u0 = inputs.random_state(n_r, n_t, 1, seed=77)
    o = oracle.Oracle.from_workload(w, theta_order=10)
    o.set_observer(10.3, 1.1, 80)
    o.set_initial(u0)
    o.step(80)
    ref, sref = o.read(), o.observe(80)
    for opts in ({}, {"tile_i": 8}, {"tile_i": 16}, {"col_run": 0}, {"col_run": 0, "tile_i": 8}, {"tile_i": 12},
                 {"col_run": 0, "tile_i": 16}, {"use_tma": 0}):
        g = run_gpu(teuk, w, u0, 80, observer=(10.3, 1.1), options={"theta_order": 10, **opts})
        geom = g.step_geometry()
        assert geom["tile_j"] == n_t
        err = oracle.rel_linf(g.read(), ref)
        serr = series_err(g.observe(80), sref)
        assert max(err.values()) <= TOL[1] and max(serr.values()) <= TOL[1], (opts, err, serr)


def test_theta10_invariants_and_tiles(teuk):
    w = inputs.config(1).scaled(n_r=96, precision=2)
    u0 = inputs.initial_state(w)
    u = run_gpu(teuk, w, u0, 40, options={"theta_order": 10}).read()
    assert np.array_equal(u, u[:, :, ::-1, :])
    assert not u[..., 0].any() and not u[..., -1].any() and not u[1].any()
    for ti in (2, 5, 16):
        v = run_gpu(teuk, w, u0, 40, options={"theta_order": 10, "tile_i": ti}).read()
        assert np.array_equal(u, v)
    h = teuk.Teuk.from_workload(w.scaled(n_theta=4))
    with pytest.raises(teuk.TeukError):
        h.set_option("theta_order", 10)          # needs n_theta >= 5


@pytest.mark.parametrize("cfg,steps_gpu,k", [(2, 100, 8), (3, 60, 6), (4, 60, 4)])
def test_theta10_full_size_configs_windowed(teuk, cfg, steps_gpu, k):
    w = inputs.config(cfg)
    w = w.scaled(dt_override=0.5 * w.dt)
    L = w.precision
    u0 = inputs.initial_state(w)
    g = run_gpu(teuk, w, u0, steps_gpu, options={"theta_order": 10})
    mid = g.read()
    assert np.isfinite(mid).all()
    g.step(k)
    fin = g.read()
    i_c = int((inputs.pulse_parameters(w)[0] - w.rstar_min) / w.dr)
    n_win = 64
    for i_lo in (0, i_c - n_win // 2, w.n_r - n_win):
        o = oracle.Oracle.from_workload(w, i_lo=i_lo, n_win=n_win, theta_order=10)
        o.set_initial(np.ascontiguousarray(mid[..., i_lo:i_lo + n_win]))
        o.step(k)
        ref = o.read()
        a, b = (0 if i_lo == 0 else k + 1), (n_win if i_lo + n_win == w.n_r else n_win - k - 1)
        got = np.ascontiguousarray(fin[..., i_lo:i_lo + n_win][..., a:b])
        want = np.ascontiguousarray(ref[..., a:b])
        for re, im in ((0, 1), (2, 3)):
            dre, _ = oracle._limb_diff(got[re], want[re])
            dim, _ = oracle._limb_diff(got[im], want[im])
            den = np.hypot(fin[re, 0], fin[im, 0]).max()
            assert float(np.hypot(dre, dim).max() / den) <= TOL[L], (cfg, i_lo, re)


# ------------------------------------------------------------------------------- NEXT-2: multipole-projection observer
def _mp_err(a, b):
    """series [n][n_ell][2][L]: max |a - b| over everything / max |b| (complex), differences formed exactly"""
    n, ne, _, L = b.shape
    A = np.ascontiguousarray(np.transpose(a, (2, 3, 0, 1)))      # [2][L][n][n_ell]
    B = np.ascontiguousarray(np.transpose(b, (2, 3, 0, 1)))
    dre, _ = oracle._limb_diff(A[0], B[0])
    dim, _ = oracle._limb_diff(A[1], B[1])
    return float(np.hypot(dre, dim).max() / np.hypot(B[0, 0], B[1, 0]).max())


@pytest.mark.parametrize("L,base,n_r,n_t,steps,order", [(1, 2, 203, 24, 120, 2), (2, 2, 150, 16, 60, 2), (4, 2, 90, 12, 30, 2),
                                                        (1, 4, 300, 40, 100, 2), (2, 4, 120, 32, 40, 10), (4, 4, 80, 32, 20, 10)])
def test_multipole_observer_parity(teuk, L, base, n_r, n_t, steps, order):
    w = inputs.config(base).scaled(n_r=n_r, n_theta=n_t, rstar_min=-30.0, rstar_max=60.0, precision=L)
    w = w.scaled(dt_override=0.5 * inputs.stable_dt(w))
    u0 = inputs.random_state(n_r, n_t, L, seed=300 + L)
    n_ell = 9
    g = teuk.Teuk.from_workload(w, obs_capacity=steps)
    g.set_option("theta_order", order)
    g.set_option("graph_steps", 8)
    g.set_observer(10.3, 1.1, steps)
    g.set_multipole_observer(12.7, n_ell, steps)
    g.set_initial(u0)
    g.step(steps)
    o = oracle.Oracle.from_workload(w, theta_order=order)
    o.set_observer(10.3, 1.1, steps)
    o.set_multipole_observer(12.7, n_ell, steps)
    o.set_initial(u0)
    o.step(steps)
    got, ref = g.observe_multipoles(steps), o.observe_multipoles(steps)
    assert got.shape == ref.shape == (steps, n_ell, 2, L)
    err = _mp_err(got, ref)
    print("multipoles", L, base, order, err)
    assert err <= TOL[L]
    assert max(series_err(g.observe(steps), o.observe(steps)).values()) <= TOL[L]      # the point observer still works beside it
    assert max(oracle.rel_linf(g.read(), o.read()).values()) <= TOL[L]


def test_multipole_observer_config4_full_size(teuk):
    """config 4 (qd, 8192 x 32, a = 0.5, pure l = 0 data: the Fig. 1 setting) at full size: the oracle advances a radial
    window around the observer from the GPU's state and must reproduce the projected series"""
    w = inputs.config(4)
    u0 = inputs.initial_state(w)
    k, pre = 5, 40
    g = teuk.Teuk.from_workload(w, obs_capacity=pre + k)
    g.set_multipole_observer(w.rstar_obs, 9, pre + k)
    g.set_initial(u0)
    g.step(pre)
    mid = g.read()
    g.step(k)
    got = g.observe_multipoles(pre + k)[pre:]
    i_c = int((w.rstar_obs - w.rstar_min) / w.dr)
    n_win = 48
    i_lo = i_c - n_win // 2
    o = oracle.Oracle.from_workload(w, i_lo=i_lo, n_win=n_win)
    o.set_multipole_observer(w.rstar_obs, 9, k)
    o.set_initial(np.ascontiguousarray(mid[..., i_lo:i_lo + n_win]))
    o.step(k)
    err = _mp_err(got, o.observe_multipoles(k))
    print("cfg4 multipoles, full size:", err)
    assert err <= TOL[4]
    with pytest.raises(teuk.TeukError):
        g.set_multipole_observer(w.rstar_obs, 10, 1)          # at most 9 multipoles (l' = 0..8 of Fig. 1)


# ------------------------------------------------------------------------------- full-size configs (bench launch geometry)
@pytest.mark.parametrize("cfg,steps_gpu,k", [(2, 300, 12), (3, 120, 8), (4, 100, 6)])
def test_full_size_configs_windowed(teuk, cfg, steps_gpu, k):
    """BASELINE.json configs 2-4 at full grid size in the launch configuration bench.py times: the GPU
    runs steps_gpu iterations, then k more; the oracle advances sampled radial windows of the GPU's
    state by the same k iterations (domain of dependence: interior of the window is exact)."""
    w = inputs.config(cfg)
    L = w.precision
    u0 = inputs.initial_state(w)
    g = run_gpu(teuk, w, u0, steps_gpu)
    mid = g.read()
    assert np.isfinite(mid).all() and np.abs(mid[0, 0]).max() > 1e-3
    g.step(k)
    fin = g.read()
    c = inputs.pulse_parameters(w)[0]
    i_c = int((c - w.rstar_min) / w.dr)
    n_win = 96
    worst = {}
    for i_lo in (0, i_c - n_win // 2, i_c + 3 * n_win, w.n_r - n_win):
        o = oracle.Oracle.from_workload(w, i_lo=i_lo, n_win=n_win)
        o.set_initial(np.ascontiguousarray(mid[..., i_lo:i_lo + n_win]))
        o.step(k)
        ref = o.read()
        a, b = k + 1, n_win - k - 1
        if i_lo == 0:
            a = 0                                   # true Dirichlet wall: the window edge IS the boundary
        if i_lo + n_win == w.n_r:
            b = n_win
        sl = slice(a, b)
        scale_ref = np.zeros_like(fin)              # normalise by the global field maximum (A17)
        got = np.ascontiguousarray(fin[..., i_lo:i_lo + n_win][..., sl])
        want = np.ascontiguousarray(ref[..., sl])
        diffs = {}
        for name, (re, im) in {"Phi": (0, 1), "Pi": (2, 3)}.items():
            dre, _ = oracle._limb_diff(got[re], want[re])
            dim, _ = oracle._limb_diff(got[im], want[im])
            den = np.hypot(fin[re, 0], fin[im, 0]).max()
            diffs[name] = float(np.hypot(dre, dim).max() / den)
        worst[i_lo] = diffs
        assert max(diffs.values()) <= TOL[L], (i_lo, diffs)
    print(cfg, worst)


@pytest.mark.parametrize("n_r,n_t,L", [(4096, 32, 1), (4096, 256, 1), (16384, 64, 2), (4096, 256, 2), (4096, 64, 4), (65536, 32, 1)])
def test_sweep_cells_prefix_windowed(teuk, n_r, n_t, L):
    """BASELINE.json config 5 (a = 0.99, s = -2, m = 2) cells in the launch geometry bench.py --sweep times: 60-step GPU
    prefix, then k more steps checked against oracle windows (inner wall, pulse, outer wall)"""
    w = inputs.sweep_cell(n_r, n_t, L)
    u0 = inputs.initial_state(w)
    pre, k = 60, 6
    g = run_gpu(teuk, w, u0, pre)
    mid = g.read()
    assert np.isfinite(mid).all()
    g.step(k)
    fin = g.read()
    i_c = int((inputs.pulse_parameters(w)[0] - w.rstar_min) / w.dr)
    n_win = 40
    for i_lo in (0, i_c - n_win // 2, n_r - n_win):
        o = oracle.Oracle.from_workload(w, i_lo=i_lo, n_win=n_win)
        o.set_initial(np.ascontiguousarray(mid[..., i_lo:i_lo + n_win]))
        o.step(k)
        ref = o.read()
        a, b = (0 if i_lo == 0 else k + 1), (n_win if i_lo + n_win == n_r else n_win - k - 1)
        got = np.ascontiguousarray(fin[..., i_lo:i_lo + n_win][..., a:b])
        want = np.ascontiguousarray(ref[..., a:b])
        for re, im in ((0, 1), (2, 3)):
            dre, _ = oracle._limb_diff(got[re], want[re])
            dim, _ = oracle._limb_diff(got[im], want[im])
            den = np.hypot(fin[re, 0], fin[im, 0]).max()
            assert float(np.hypot(dre, dim).max() / den) <= TOL[L], (n_r, n_t, L, i_lo, re)


def test_config2_prefix_full_grid_fp64(teuk):
    """config 2 at full size against the full-grid oracle for a 1000-step prefix (observer included)."""
    w = inputs.config(2)
    u0 = inputs.initial_state(w)
    steps = 1000
    g = run_gpu(teuk, w, u0, steps, observer=w.observer)
    o = run_oracle(w, u0, steps, observer=w.observer)
    err = oracle.rel_linf(g.read(), o.read())
    print("cfg2 prefix", err)
    assert max(err.values()) <= TOL[1]
    serr = series_err(g.observe(steps), o.observe(steps))
    assert max(serr.values()) <= TOL[1] or np.abs(o.observe(steps)).max() < 1e-300


# Config 2 at full size and FULL length against the oracle, for every fp64 kernel family at the same 1e-12: see
# tests/test_gpu_golden.py (un-gated; the oracle side is cached in tests/golden/cfg2_full.npz).


@pytest.mark.parametrize("cfg", [3, 4])
def test_full_length_precision_ladder_on_gpu(teuk, cfg):
    """SMOKE, NOT PARITY (it compares the CUDA path with itself; parity at full length is tests/test_gpu_golden.py):
    configs 3 and 4 at full size and full length at the three precisions must form a ladder -- fp64 agrees with dd to
    fp64 accuracy, dd with qd to dd accuracy -- and stay finite.  Observer series included."""
    w = inputs.config(cfg)
    u0 = inputs.initial_state(w)
    out = {}
    for L in (1, 2, 4):
        g = run_gpu(teuk, w, u0, w.steps, precision=L, observer=w.observer)
        u, ser = g.read(), g.observe(w.steps)
        assert np.isfinite(u).all() and ser.shape[0] == w.steps
        pad = np.zeros((4, 4) + u.shape[2:])
        pad[:, :L] = u
        sp = np.zeros((w.steps, 4, 4))
        sp[:, :, :L] = ser
        out[L] = (pad, sp)
        g.close()
    e12 = oracle.rel_linf(out[1][0], out[2][0])
    e24 = oracle.rel_linf(out[2][0], out[4][0])
    s12 = series_err(out[1][1], out[2][1])
    s24 = series_err(out[2][1], out[4][1])
    print("cfg", cfg, "full length ladder: fp64-dd", e12, s12, "dd-qd", e24, s24)
    assert max(e12.values()) <= 1e-11 and max(s12.values()) <= 1e-11
    assert max(e24.values()) <= 1e-26 and max(s24.values()) <= 1e-26
    assert max(e24.values()) > 0 and max(e12.values()) > 1e-18          # the rungs are distinct


@pytest.mark.skipif(os.environ.get("TEUK_FULL_LENGTH") != "1",
                    reason="15 minutes of host time for the full-grid dd / qd oracle; set TEUK_FULL_LENGTH=1 "
                           "(TEUK_FULL_STEPS_CFG3 / TEUK_FULL_STEPS_CFG4 change the prefix; results: DESIGN.md section 5)")
@pytest.mark.parametrize("cfg", [3, 4])
def test_config3_config4_full_grid_long_runs(teuk, cfg):
    """BASELINE.json configs 3 (dd) and 4 (qd) at FULL size against the FULL-GRID oracle (no windows) in its ARBITRATION
    tier (exact-then-round arithmetic, about 3.5e5 updates/s on 16 cores), observer series included, over a prefix.
    The full-length comparison (fast oracle tier, cached) is tests/test_gpu_golden.py."""
    w = inputs.config(cfg)
    steps = int(os.environ.get(f"TEUK_FULL_STEPS_CFG{cfg}", {3: 200, 4: 400}[cfg]))
    u0 = inputs.initial_state(w)
    g = run_gpu(teuk, w, u0, steps, observer=w.observer)
    got, ser = g.read(), g.observe(steps)
    g.close()
    o = run_oracle(w, u0, steps, observer=w.observer)
    err = oracle.rel_linf(got, o.read())
    serr = series_err(ser, o.observe(steps))
    print("cfg", cfg, "full grid,", steps, "steps: state", err, "observer", serr)
    assert max(err.values()) <= TOL[w.precision]
    assert max(serr.values()) <= TOL[w.precision]


def test_fig1_tail_rule_on_gpu(teuk):
    """The paper's Fig. 1 experiment on the product path (quad-double, 10th-order theta operator, multipole observer;
    BASELINE.json config 4 = Kerr a = 0.5, pure l = 0 data): the multipoles l' = 0 and 2 decay as t^-(l + l' + 3), the
    rule the caption of Fig. 1 states (expected exponents from tests/golden/tail_exponents.txt), while the
    SAME run in fp64 loses l' = 2 in rounding noise - the paper's case for high precision."""
    from paper_1006_0663_b200 import fig1_tails
    rows = [ln.split() for ln in open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "tail_exponents.txt"))
            if ln.strip() and not ln.startswith("#")]
    n = {int(r[2]): int(r[3]) for r in rows if r[0] == "kerr" and r[1] == "0"}
    t, amp, wall, w = fig1_tails.run(4, 10, t_end=1060.0, n_ell=3)
    i0 = fig1_tails.power_index(t, amp[:, 0], 700, 1050)
    i2 = fig1_tails.power_index(t, amp[:, 2], 700, 1050)
    print("fig. 1 run, qd:", wall, "s; indices l'=0:", i0, "l'=2:", i2)
    assert i0 is not None and abs(i0 + n[0]) < 0.1                 # -3
    assert i2 is not None and abs(i2 + n[2]) < 0.4                 # -5 (still approaching the asymptote at t ~ 1000 M)
    k = int(np.searchsorted(t, 1000.0))
    assert 1e-13 < abs(amp[k, 2]) < 1e-9 and abs(amp[k, 1]) < 1e-40 * abs(amp[k, 0])     # odd l' stays at rounding level
    t1, amp1, _, _ = fig1_tails.run(1, 10, t_end=1060.0, n_ell=3)
    assert abs(amp1[k, 2]) > 100 * abs(amp[k, 2])                  # fp64: l' = 2 drowned in rounding noise


# ------------------------------------------------------------------------------- invariants and edge cases
@pytest.mark.parametrize("L", [1, 2, 4])
def test_gpu_exact_invariants(teuk, L):
    w = inputs.config(1).scaled(n_r=96, precision=L)
    u0 = inputs.initial_state(w)
    g = run_gpu(teuk, w, u0, 50)
    u = g.read()
    assert np.array_equal(u, u[:, :, ::-1, :])                      # reflection symmetry (A12), bitwise
    assert not u[..., 0].any() and not u[..., -1].any()             # Dirichlet rows
    assert not u[1].any() and not u[3].any()                        # real data stay real for a = 0
    # power-of-two linearity, bitwise
    g2 = run_gpu(teuk, w, u0 * 2.0 ** 7, 50)
    assert np.array_equal(g2.read(), u * 2.0 ** 7)
    # checkpoint / restart and graph / no-graph equivalence, bitwise
    g3 = run_gpu(teuk, w, u0, 21, options={"graph_steps": 0})
    mid = g3.read()
    g4 = run_gpu(teuk, w, mid, 29, options={"graph_steps": 4})
    assert np.array_equal(g4.read(), u)


def test_observer_reset_mid_run(teuk):
    """teuk_set_observer between teuk_step calls restarts the series at the current step"""
    w = inputs.config(1).scaled(n_r=96)
    u0 = inputs.initial_state(w)
    g = teuk.Teuk.from_workload(w, obs_capacity=50)
    g.set_observer(40.0, 1.2, 50)
    g.set_initial(u0)
    g.step(20)
    assert g.observe(50).shape[0] == 20
    g.set_observer(30.0, 1.0, 50)
    assert g.observe(50).shape[0] == 0
    g.step(7)
    got = g.observe(50)
    assert got.shape[0] == 7
    o = run_oracle(w, u0, 20)
    o.set_observer(30.0, 1.0, 50)
    o.step(7)
    assert max(series_err(got, o.observe(50)).values()) <= TOL[1]


def test_multipole_observer_enabled_mid_run(teuk):
    """teuk_set_multipole_observer between teuk_step calls restarts BOTH series at the current step: no stale or zero
    leading samples, and the multipole samples are those of the oracle run from the same state"""
    w = inputs.config(4).scaled(n_r=96, n_theta=12, rstar_min=-20.0, rstar_max=75.0, precision=1)
    u0 = inputs.initial_state(w)
    g = teuk.Teuk.from_workload(w, obs_capacity=40)
    g.set_observer(40.0, 1.2, 40)
    g.set_initial(u0)
    g.step(13)
    assert g.observe(40).shape[0] == 13
    g.set_multipole_observer(30.0, 3, 40)
    assert g.observe_multipoles(40).shape[0] == 0 and g.observe(40).shape[0] == 0
    g.step(9)
    got = g.observe_multipoles(40)
    assert got.shape[0] == 9 and g.observe(40).shape[0] == 9
    o = run_oracle(w, u0, 13)
    o.set_multipole_observer(30.0, 3, 40)
    o.step(9)
    ref = o.observe_multipoles(40)
    assert ref.shape == got.shape
    scale = np.abs(ref).max()
    assert scale > 0 and np.abs(got - ref).max() <= TOL[1] * scale


def test_edge_cases_and_errors(teuk):
    import ctypes
    # smallest legal grid, odd m, zero steps
    w = inputs.config(1).scaled(n_r=3, n_theta=2, m=1)
    u0 = inputs.random_state(3, 2, 1, seed=1)
    g = run_gpu(teuk, w, u0, 0)
    assert g.steps_done() == 0
    g.step(5)
    o = run_oracle(w, u0, 5)
    assert max(oracle.rel_linf(g.read(), o.read()).values()) <= TOL[1] or not o.read().any()
    # odd m on a real grid
    w = inputs.config(2).scaled(n_r=90, n_theta=10, m=1, s=-1, rstar_min=-20.0, rstar_max=40.0)
    w = w.scaled(dt_override=inputs.stable_dt(w))
    u0 = inputs.random_state(90, 10, 1, seed=2)
    g = run_gpu(teuk, w, u0, 40)
    o = run_oracle(w, u0, 40)
    assert max(oracle.rel_linf(g.read(), o.read()).values()) <= TOL[1]
    # state errors
    h = teuk.Teuk.from_workload(w)
    with pytest.raises(teuk.TeukError) as e:
        h.step(1)
    assert e.value.code == teuk.ESTATE
    with pytest.raises(teuk.TeukError) as e:
        h.set_observer(1e9, 1.0, 0)
    assert e.value.code == teuk.EINVAL
    h.set_initial(u0)
    with pytest.raises(teuk.TeukError) as e:
        h.set_option("graph_steps", 8)
    assert e.value.code == teuk.ESTATE
    with pytest.raises(teuk.TeukError):
        teuk.Teuk(1.0, 1.5, 0, 0, 64, 8, -10.0, 10.0, 0.1, 1)
    # non-finite detection is sticky and reported
    bad = u0.copy()
    bad[0, 0, 5, 40] = np.inf
    hb = teuk.Teuk.from_workload(w, obs_capacity=8)
    hb.set_observer(w.rstar_min + 40.2 * w.dr, (5.5) * math.pi / w.n_theta, 8)
    hb.set_initial(bad)
    hb.step(3)
    hb.observe(8, allow_nonfinite=True)
    assert hb.last_observe_status == teuk.ENONFINITE
