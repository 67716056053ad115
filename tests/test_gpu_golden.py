"""Full-length parity of configs 2, 3 and 4 (BASELINE.json `north_star`: "GPU results must match the oracle ...
after the run"; the tails appear only long after the ringing has died away, so the long run IS the
workload).  The oracle side is cached: tests/golden/cfg{2,3,4}_full.npz, written by `python -m oracle.make_golden`
(which calls only oracle/ and the seeded input recipe) on the FULL grid at FULL length -- fp64 with the plain double
stepper, dd/qd with the oracle's fast arithmetic tier (pinned against the exact-then-round tier in
tests/test_oracle_fast_tier.py).  The CUDA path runs the same seeded inputs through the C ABI in bench.py's launch
configuration and is compared ELEMENT BY ELEMENT on every stored r* column (all theta rows, all limbs) at every
stored checkpoint, and on the whole observer series, at 1e-12 / 1e-27 / 1e-55 (reading A17).
Not env-gated: about 1 s / 3 s / 17 s of device time."""
import json
import os

import numpy as np
import pytest

from oracle import oracle
from paper_1006_0663_b200 import inputs

pytestmark = pytest.mark.gpu
TOL = {1: 1e-12, 2: 1e-27, 4: 1e-55}
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


@pytest.fixture(scope="module")
def teuk():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1006_0663_b200 import teuk as t
    return t


def _load(k):
    path = os.path.join(GOLDEN, f"cfg{k}_full.npz")
    if not os.path.exists(path):
        pytest.skip(f"{path} is missing: run `python -m oracle.make_golden --cfg {k}`")
    z = np.load(path)
    return z, json.loads(str(z["meta"]))


def _series_err(a, b):
    a4 = np.ascontiguousarray(np.transpose(a, (1, 2, 0)))
    b4 = np.ascontiguousarray(np.transpose(b, (1, 2, 0)))
    return oracle.rel_linf(a4, b4)


def _run_against_golden(teuk, k, options=None):
    z, meta = _load(k)
    w = inputs.config(k)
    assert meta["dt_hex"] == float(w.dt).hex() and meta["n_r"] == w.n_r and meta["n_theta"] == w.n_theta
    assert meta["precision"] == w.precision and meta["seed"] == w.seed and meta["steps_full"] == w.steps
    done = meta["steps_done"]
    ro, to = w.observer
    g = teuk.Teuk.from_workload(w, obs_capacity=done)
    for key, v in (options or {}).items():
        g.set_option(key, v)
    g.set_observer(ro, to, done)
    g.set_initial(inputs.initial_state(w))
    report, at = {}, 0
    for n in [int(c) for c in z["checkpoints"]]:
        g.step(n - at)
        at = n
        ref = z[f"state_{n}"]
        stride = meta["final_stride"] if n == meta["steps_full"] else meta["mid_stride"]
        got = np.ascontiguousarray(g.read()[:, :, :, ::stride])
        assert got.shape == ref.shape
        assert np.abs(ref[0, 0]).max() > 0
        err = oracle.rel_linf(got, ref)
        report[n] = err
        assert max(err.values()) <= TOL[w.precision], (k, n, err)
    ser = g.observe(done)
    assert ser.shape == z["observer"].shape
    serr = _series_err(ser, z["observer"])
    report["observer"] = serr
    print(f"cfg{k} {options or ''}: steps {done}/{w.steps}: {report}")
    assert max(serr.values()) <= TOL[w.precision], (k, serr)
    return done, w.steps


@pytest.mark.parametrize("k", [2, 3, 4])
def test_full_length_against_cached_oracle(teuk, k):
    done, full = _run_against_golden(teuk, k)
    if done < full:
        # only when a golden file was written with --max-steps (the committed ones cover every step)
        pytest.xfail(f"cfg{k}: parity verified on the first {done} of {full} steps only")


@pytest.mark.parametrize("options", [{"coef_variant": 1}, {"coef_variant": 1, "march": 0}, {"coef_variant": 0},
                                     {"coef_variant": 2}, {"time_block": 2}],
                         ids=["semi_recompute_march", "semi_recompute_tiles", "stored_planes", "full_recompute", "time_block_2"])
def test_config2_full_length_every_fp64_path(teuk, options):
    """H1b / NEXT-3: every fp64 kernel family meets the SAME 1e-12 at full length (no per-variant tolerance)"""
    done, full = _run_against_golden(teuk, 2, options)
    assert done == full
