"""Pin for reading A15b: why configs 2, 3 and 5 do NOT run at BASELINE.json's dt = 0.5 dr*.

Eqs. (13)-(14) are a two-step (midpoint) rule for the source terms: a mode with
Phi_tt = -omega^2 Phi is advanced with amplification |G| = sqrt(1 + (omega dt)^4/4) ~ 1 + (omega dt)^4/8 per step
(no damping for radially smooth modes).  For (s, m) != (0, 0) the pole rows of the theta grid carry
omega^2 ~ kappa_max [4/dtheta^2 + (|m|+|s|)^2/sin^2(dtheta/2)] (`inputs.omega_max`), so at config 2's dr*, dtheta
the literal dt = 0.5 dr* has omega dt ~ 1.05 and the run blows up; `inputs.stable_dt` replaces it.  The oracle
shows all three facts on a 1201-column strip of config 2's grid (same dr*, dtheta, a, s, m):
  (a) at 0.5 dr* the field grows by > 1e20 in 500 steps at the per-step rate (omega dt)^4/8 (within 20 %),
  (b) at `stable_dt` it stays bounded over the same steps,
  (c) (s, m) = (0, 0) -- configs 1 and 4, which keep BASELINE's dt -- is bounded at 0.5 dr*.
"""
import math

import numpy as np

from oracle import oracle
from paper_1006_0663_b200 import inputs

N_STRIP = 1201


def _strip(w):
    """config-2-like strip centred on the peak of kappa (r* ~ 2): same dr*, dtheta and physics, 1201 columns"""
    dr = w.dr
    i0 = int(round((2.0 - w.rstar_min) / dr)) - N_STRIP // 2
    lo = w.rstar_min + i0 * dr
    return w.scaled(n_r=N_STRIP, rstar_min=lo, rstar_max=lo + (N_STRIP - 1) * dr, centre=(2.0, 0.0), width=(3.0, 0.0))


def _max_history(w, steps, every):
    o = oracle.Oracle.from_workload(w, precision=1)
    o.set_initial(inputs.initial_state(w))
    out = []
    for _ in range(steps // every):
        o.step(every)
        u = o.read()
        out.append(float(np.abs(u).max()))
    return np.array(out)


def test_literal_dt_blows_up_at_the_midpoint_rule_rate():
    w = _strip(inputs.config(2))
    w_lit = w.scaled(dt_override=0.5 * w.dr)                      # BASELINE.json: "dt = 0.5 dr*"
    hist = _max_history(w_lit, 500, 50)
    assert hist[-1] > 1e20 * max(hist[0], 1.0), hist
    rate = math.log(hist[-1] / hist[-5]) / (4 * 50)               # per-step log growth once the stiffest mode dominates
    z = inputs.omega_max(w_lit) * w_lit.dt
    predicted = 0.5 * math.log1p(z ** 4 / 4.0)                    # ln|G|, = z^4/8 to leading order
    print(f"omega dt = {z:.3f}: measured growth {rate:.4f}/step, predicted {predicted:.4f} (z^4/8 = {z ** 4 / 8:.4f})")
    assert abs(rate - predicted) <= 0.2 * predicted


def test_stable_dt_stays_bounded_and_rule_is_the_e_fold_rule():
    w = _strip(inputs.config(2))
    assert w.dt == inputs.config(2).dt                            # the strip keeps config 2's own reduced dt
    z = inputs.omega_max(w) * w.dt
    assert abs(z - (8.0 / w.steps) ** 0.25) < 1e-12               # z = (8/N)^(1/4) ...
    assert abs((1 + z ** 4 / 8) ** w.steps - math.e) < 0.01       # ... i.e. at most one e-fold over the whole run
    hist = _max_history(w, 500, 50)
    # the pulse itself evolves (max|u| drifts by a factor of a few as it moves inward); what must not happen is the
    # exponential runaway of the first test (> 1e20 over the same 500 steps)
    assert hist.max() < 20.0 * max(hist[0], 0.05), hist
    assert hist[-1] / hist[-2] < 1.5, hist


def test_s0_m0_is_bounded_at_the_literal_dt():
    """configs 1 and 4 have no pole term and keep dt = 0.5 dr*"""
    w4 = inputs.config(4)
    assert w4.dt == 0.5 * w4.dr and inputs.config(1).dt == 0.5 * inputs.config(1).dr
    w = _strip(inputs.config(2)).scaled(s=0, m=0, profile="P2", dt_override=None)
    assert w.dt == 0.5 * w.dr
    hist = _max_history(w, 500, 50)
    # the pulse itself evolves (max|u| drifts by a factor of a few as it moves inward); what must not happen is the
    # exponential runaway of the first test (> 1e20 over the same 500 steps)
    assert hist.max() < 20.0 * max(hist[0], 0.05), hist
    assert hist[-1] / hist[-2] < 1.5, hist
