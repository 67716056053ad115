"""`python -m paper_1006_0663_b200.selfcheck` — run every kernel family of libteuk.so once on a small problem.

A quick installation check for users and the command the sanitizer runs in profiles/sanitizer.md execute
(`compute-sanitizer --tool memcheck|racecheck|initcheck python -m paper_1006_0663_b200.selfcheck`): small grids with a
ragged tail in both directions, odd |m| among them, a handful of iterations per family.  No oracle is involved: each
family must stay finite and the fp64 families must agree with one another to rounding (they compute the same
iteration, Eqs. (13)-(14), with different data movement).
"""
from __future__ import annotations

import sys

import numpy as np

from . import inputs, teuk

N_R, N_THETA, STEPS = 150, 20, 7


def _run(w, u0, options, steps=STEPS, multipole=False):
    g = teuk.Teuk.from_workload(w, obs_capacity=steps)
    for k, v in options.items():
        g.set_option(k, v)
    g.set_observer(11.0, 1.2, steps)
    if multipole:
        g.set_multipole_observer(9.0, 3, steps)
    g.set_initial(u0)
    g.step(steps)
    u, ser = g.read(), g.observe(steps)
    mp = g.observe_multipoles(steps) if multipole else None
    geom = g.step_geometry()
    g.close()
    return u, ser, mp, geom


def main() -> int:
    ok = True
    families = [
        ("stored planes, TMA tiles (step_kernel_f64_tma)", 1, {}),
        ("stored planes, generic tiles (step_kernel<1>)", 1, {"use_tma": 0}),
        ("semi-recompute, column march (step_kernel_f64_march)", 1, {"coef_variant": 1}),
        ("semi-recompute, TMA tiles (step_kernel_f64_rc)", 1, {"coef_variant": 1, "march": 0}),
        ("full recompute, TMA tiles (step_kernel_f64_rc<full>)", 1, {"coef_variant": 2}),
        ("two iterations per launch (step2_kernel_f64_tma)", 1, {"time_block": 2}),
        ("double-double (step_kernel<2>)", 2, {}),
        ("double-double, two threads per point (step_kernel_pair<2>)", 2, {"variant": 3, "tile_i": 32, "tile_j": 16}),
        ("quad-double, two threads per point (step_kernel_pair<4>)", 4, {}),
        ("quad-double, one thread per point (step_kernel<4>)", 4, {"variant": 4}),
        ("theta order 10, fp64 TMA columns, row runs (step_kernel_f64_col_run)", 1, {"theta_order": 10}),
        ("theta order 10, fp64 TMA columns, point per thread (step_kernel_f64_col_tma)", 1, {"theta_order": 10, "col_run": 0}),
        ("theta order 10, fp64 generic columns (step_kernel_col<1>)", 1, {"theta_order": 10, "use_tma": 0}),
        ("theta order 10, double-double (step_kernel_col<2>)", 2, {"theta_order": 10}),
        ("theta order 10, quad-double, two threads per point (step_kernel_col_pair<4>)", 4, {"theta_order": 10}),
        ("theta order 10, quad-double, one thread per point (step_kernel_col<4>)", 4, {"theta_order": 10, "variant": 4}),
    ]
    for m in (2, 1):                                      # even and odd |m| (polar ghost sign)
        ref = {}
        for name, L, opts in families:
            w = inputs.config(2).scaled(n_r=N_R, n_theta=N_THETA, rstar_min=-30.0, rstar_max=60.0, precision=L, m=m)
            w = w.scaled(dt_override=0.5 * inputs.stable_dt(w))
            u0 = inputs.random_state(w.n_r, w.n_theta, L, seed=42)
            u, ser, mp, geom = _run(w, u0, opts, multipole=(L != 1 or not opts))
            fine = bool(np.isfinite(u).all() and np.isfinite(ser).all() and np.abs(u[0, 0]).max() > 0)
            fine = fine and bool(np.all(u[:, :, :, 0] == 0.0) and np.all(u[:, :, :, -1] == 0.0))
            if mp is not None:
                fine = fine and bool(np.isfinite(mp).all())
            order = opts.get("theta_order", 2)
            note = ""
            if L == 1:
                if order in ref:
                    d = float(np.abs(u - ref[order]).max() / np.abs(ref[order]).max())
                    fine = fine and d < 1e-12
                    note = f"  vs first fp64 family: {d:.1e}"
                else:
                    ref[order] = u
            else:
                # the dd / qd kernels of one precision and theta order perform the same operations in the same order: bitwise equal
                if (L, order) in ref:
                    same = bool(np.array_equal(u, ref[(L, order)]))
                    fine = fine and same
                    note = f"  bitwise == first {'dd' if L == 2 else 'qd'} family: {same}"
                else:
                    ref[(L, order)] = u
            print(f"m={m}  {'ok  ' if fine else 'FAIL'} {name}  tile {geom['tile_i']}x{geom['tile_j']}{note}", flush=True)
            ok = ok and fine
    # the allocation-free hook and the device build of the arithmetic layer
    w = inputs.config(2).scaled(n_r=N_R, n_theta=N_THETA, rstar_min=-30.0, rstar_max=60.0, precision=1)
    g = teuk.Teuk.from_workload(w.scaled(dt_override=inputs.stable_dt(w)))
    same = bool(np.array_equal(g.folded_static(True, 1), g.folded(True, 1)))
    print(f"     {'ok  ' if same else 'FAIL'} teuk_get_folded_static == teuk_get_folded", flush=True)
    rng = np.random.default_rng(3)
    a = rng.uniform(0.5, 2.0, size=(256, 4)) * (2.0 ** (-54.0 * np.arange(4)))[None, :]
    b = rng.uniform(0.5, 2.0, size=(256, 4)) * (2.0 ** (-54.0 * np.arange(4)))[None, :]
    arith = all(np.array_equal(teuk.test_mp_op(op, 4, a, b, on_device=True), teuk.test_mp_op(op, 4, a, b, on_device=False))
                for op in ("add", "mul", "div"))
    print(f"     {'ok  ' if arith else 'FAIL'} device quad-double arithmetic == host build", flush=True)
    return 0 if (ok and same and arith) else 1


if __name__ == "__main__":
    sys.exit(main())
