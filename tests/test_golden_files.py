"""The cached full-length oracle results (tests/golden/cfg{2,3,4}_full.npz, written by `python -m oracle.make_golden`)
are what the `-m gpu` full-length parity tests compare with, so they are checked here, on the CPU, against the oracle
as it stands: the recorded parameters are BASELINE.json's configs as `inputs.config` builds them, and the first
observer samples are reproduced BIT FOR BIT by a fresh oracle run on a radial window around the observer (window
interior = full grid by the domain of dependence, pinned in tests/test_oracle_invariants.py).  A golden file written
by different oracle arithmetic, different inputs or a different dt fails here."""
import json
import math
import os

import numpy as np
import pytest

from oracle import oracle
from paper_1006_0663_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
N_CHECK = 24


@pytest.mark.parametrize("k", [2, 3, 4])
def test_golden_file_is_reproduced_by_the_current_oracle(k):
    path = os.path.join(GOLDEN, f"cfg{k}_full.npz")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated yet")
    z = np.load(path)
    meta = json.loads(str(z["meta"]))
    w = inputs.config(k)
    for key in ("M", "a", "s", "m", "n_r", "n_theta", "rstar_min", "rstar_max", "precision", "seed"):
        assert meta[key] == getattr(w, key), key
    assert meta["dt_hex"] == float(w.dt).hex() and meta["steps_full"] == w.steps
    assert meta["tier"] == ("exact" if w.precision == 1 else "fast")
    done = meta["steps_done"]
    assert z["observer"].shape == (done, 4, w.precision) and int(z["checkpoints"][-1]) == done
    for n in z["checkpoints"]:
        stride = meta["final_stride"] if n == w.steps else meta["mid_stride"]
        assert z[f"state_{n}"].shape == (4, w.precision, w.n_theta, len(range(0, w.n_r, stride)))
        assert np.all(z[f"state_{n}"][:, :, :, 0] == 0.0)                    # radial Dirichlet row
    # first samples of the observer series, re-derived on a window around the observer
    ro, to = w.observer
    oi = int(math.floor((ro - w.rstar_min) / w.dr))
    i_lo, n_win = oi - (N_CHECK + 4), 2 * (N_CHECK + 4) + 2
    o = oracle.Oracle.from_workload(w, i_lo=i_lo, n_win=n_win, tier=meta["tier"])
    o.set_observer(ro, to, N_CHECK)
    o.set_initial(np.ascontiguousarray(inputs.initial_state(w)[:, :, i_lo:i_lo + n_win]))
    o.step(N_CHECK)
    assert np.array_equal(o.observe(N_CHECK), z["observer"][:N_CHECK])
    assert np.abs(z["observer"][:, 0, 0]).max() > 0
