"""Own memory-safety and race checks of every kernel family (compute-sanitizer is closed on the GPU pool this project
is measured on, see profiles/r02_sanitizer.md): on small ragged grids, each family runs inside a workspace surrounded by
guard bands (no kernel may write outside the memory it was given), must leave the row padding of the state planes
untouched, must be bit-for-bit reproducible run after run and across launch decompositions (a shared-memory or
halo race shows up as a run-to-run difference), and the fp64 families must agree with one another to rounding."""
import numpy as np
import pytest

from paper_1006_0663_b200 import inputs

pytestmark = pytest.mark.gpu

FAMILIES = [
    ("f64_tma", 1, {}),
    ("f64_generic", 1, {"use_tma": 0}),
    ("f64_march", 1, {"coef_variant": 1}),
    ("f64_march_chunk7", 1, {"coef_variant": 1, "march_chunk": 7}),
    ("f64_rc", 1, {"coef_variant": 1, "march": 0}),
    ("f64_rc_full", 1, {"coef_variant": 2}),
    ("f64_tb2", 1, {"time_block": 2}),
    ("dd", 2, {}),
    ("dd_pair", 2, {"variant": 3, "tile_i": 32, "tile_j": 16}),
    ("qd", 4, {}),
    ("qd_pair_32x8", 4, {"variant": 3, "tile_i": 32, "tile_j": 8}),
    ("qd_pair_16x8", 4, {"variant": 3, "tile_i": 16, "tile_j": 8}),
    ("qd_one_thread_per_point", 4, {"variant": 4}),
    ("f64_col_run", 1, {"theta_order": 10}),
    ("f64_col_run8", 1, {"theta_order": 10, "tile_i": 8}),
    ("f64_col_tma", 1, {"theta_order": 10, "col_run": 0}),
    ("f64_col", 1, {"theta_order": 10, "use_tma": 0}),
    ("dd_col", 2, {"theta_order": 10}),
    ("qd_col", 4, {"theta_order": 10}),
    ("qd_col_one_thread_per_point", 4, {"theta_order": 10, "variant": 4}),
]


@pytest.fixture(scope="module")
def teuk():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1006_0663_b200 import teuk as t
    return t


def _run(teuk, L, opts, n_r, n_theta, m, steps):
    w = inputs.config(2).scaled(n_r=n_r, n_theta=n_theta, rstar_min=-30.0, rstar_max=60.0, precision=L, m=m)
    w = w.scaled(dt_override=0.5 * inputs.stable_dt(w))
    u0 = inputs.random_state(n_r, n_theta, L, seed=11)
    g = teuk.Teuk.from_workload(w, obs_capacity=steps, guard_bytes=1 << 16)
    for k, v in opts.items():
        g.set_option(k, v)
    g.set_observer(7.0, 1.3, steps)
    g.set_initial(u0)
    g.step(steps)
    u, ser = g.read(), g.observe(steps)
    intact = g.guards_intact()
    g.close()
    return u, ser, intact


@pytest.mark.parametrize("name,L,opts", FAMILIES, ids=[f[0] for f in FAMILIES])
@pytest.mark.parametrize("n_r,n_theta,m", [(131, 22, 2), (67, 12, 1)])
def test_guard_bands_and_reproducibility(teuk, name, L, opts, n_r, n_theta, m):
    steps = 9
    u1, s1, ok1 = _run(teuk, L, opts, n_r, n_theta, m, steps)
    u2, s2, ok2 = _run(teuk, L, opts, n_r, n_theta, m, steps)
    assert ok1 and ok2, "a kernel wrote outside its workspace"
    assert np.isfinite(u1).all() and np.isfinite(s1).all() and np.abs(u1[0, 0]).max() > 0
    assert np.array_equal(u1, u2) and np.array_equal(s1, s2), "run-to-run difference"
    assert np.all(u1[:, :, :, 0] == 0.0) and np.all(u1[:, :, :, -1] == 0.0)      # radial Dirichlet rows


@pytest.mark.parametrize("L", [2, 4])
@pytest.mark.parametrize("n_r,n_theta,m", [(131, 22, 2), (67, 12, 1), (40, 37, 2)])
def test_pair_kernel_is_bitwise_the_one_thread_per_point_kernel(teuk, L, n_r, n_theta, m):
    """step_kernel_pair (two lanes per point, partner values by shuffle) performs step_kernel's operations in
    step_kernel's order: same bits in state and observer series, on ragged grids, for every pair tile shape"""
    steps = 9
    ref_opts = {"variant": 4} if L == 4 else {}
    ref, sref, ok = _run(teuk, L, ref_opts, n_r, n_theta, m, steps)
    assert ok
    shapes = ([{}, {"variant": 3, "tile_i": 32, "tile_j": 8}, {"variant": 3, "tile_i": 16, "tile_j": 8}] if L == 4
              else [{"variant": 3, "tile_i": 32, "tile_j": 16}])
    for opts in shapes:
        u, s, ok = _run(teuk, L, opts, n_r, n_theta, m, steps)
        assert ok
        assert np.array_equal(u, ref) and np.array_equal(s, sref), opts
    if L == 4:      # theta order 10: step_kernel_col_pair against step_kernel_col
        ref, sref, ok = _run(teuk, 4, {"theta_order": 10, "variant": 4}, n_r, n_theta, m, steps)
        for opts in ({"theta_order": 10}, {"theta_order": 10, "tile_i": 3}, {"theta_order": 10, "tile_i": 8}):
            u, s, ok2 = _run(teuk, 4, opts, n_r, n_theta, m, steps)
            assert ok and ok2
            assert np.array_equal(u, ref) and np.array_equal(s, sref), opts


def test_march_kernel_is_independent_of_its_work_decomposition(teuk):
    """the column-march kernel cut into work units of different lengths (and the tile kernel of the same supply) gives
    the same bits: no dependence on which warp handled which rows, no stale ring slots between units; nor on whether the
    steps are launched programmatically dependent (default) or fully serialised ("pdl" = 0)"""
    ref = None
    for opts in ({"coef_variant": 1}, {"coef_variant": 1, "march_chunk": 5}, {"coef_variant": 1, "march_chunk": 8},
                 {"coef_variant": 1, "march_chunk": 23}, {"coef_variant": 1, "march_chunk": 37},
                 {"coef_variant": 1, "pdl": 0}, {"coef_variant": 1, "pdl": 0, "march_chunk": 8}):
        u, ser, ok = _run(teuk, 1, opts, 333, 37, 2, 33)
        assert ok
        if ref is None:
            ref = (u, ser)
        assert np.array_equal(u, ref[0]) and np.array_equal(ser, ref[1]), opts
    tiles, _, _ = _run(teuk, 1, {"coef_variant": 1, "march": 0}, 333, 37, 2, 33)
    assert np.abs(tiles - ref[0]).max() <= 1e-13 * np.abs(ref[0]).max()


def test_handle_created_for_one_supply_only(teuk):
    """teuk_create(coef_variant = 1): no stored planes in the workspace (H1b); same bits as the all-supplies
    handle stepping with that variant; the supplies that are not resident are refused"""
    n_r, n_theta, steps = 300, 24, 21
    w = inputs.config(2).scaled(n_r=n_r, n_theta=n_theta, rstar_min=-30.0, rstar_max=60.0, precision=1)
    w = w.scaled(dt_override=inputs.stable_dt(w))
    u0 = inputs.random_state(n_r, n_theta, 1, seed=3)
    out = {}
    for cv in (-1, 1, 2, 0):
        g = teuk.Teuk.from_workload(w, obs_capacity=steps, guard_bytes=1 << 16, coef_variant=cv)
        if cv == -1:
            g.set_option("coef_variant", 1)
            full_bytes = g.workspace_nbytes
        else:
            plane = n_theta * ((n_r + 15) // 16 * 16) * 8
            assert full_bytes - g.workspace_nbytes >= (16 if cv else 2) * plane - 4096
            for other in ({0, 1, 2} - {cv} if cv == 0 else {0}):
                with pytest.raises(teuk.TeukError) as e:
                    g.set_option("coef_variant", other)
                assert e.value.code == teuk.EINVAL
            with pytest.raises(teuk.TeukError):
                g.folded(False, 0 if cv else 1)
        g.set_observer(7.0, 1.3, steps)
        g.set_initial(u0)
        g.step(steps)
        out[cv] = (g.read(), g.observe(steps))
        assert g.guards_intact()
        g.close()
    assert np.array_equal(out[1][0], out[-1][0]) and np.array_equal(out[1][1], out[-1][1])
    for cv in (2, 0):
        assert np.abs(out[cv][0] - out[1][0]).max() <= 1e-13 * np.abs(out[1][0]).max()
    # theta_order 10 on a recompute-only handle uses the TMA column kernel (it reads that supply); without TMA it needs planes
    g = teuk.Teuk.from_workload(w.scaled(dt_override=0.5 * w.dt), coef_variant=1)
    g.set_option("theta_order", 10)
    g.set_initial(u0)
    g.step(3)
    assert np.isfinite(g.read()).all()
    g = teuk.Teuk.from_workload(w, coef_variant=1)
    g.set_option("theta_order", 10)
    g.set_option("use_tma", 0)
    with pytest.raises(teuk.TeukError):
        g.set_initial(u0)
