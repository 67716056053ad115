"""Fig. 1 workload of the paper on the GPU path: pure l = 0 data in Kerr (BASELINE.json config 4:
a = 0.5, s = m = 0, 8192 x 32), 10th-order theta operator, multipole-projection observer l' = 0..8, run up
to the first echo of the radial Dirichlet walls (t ~ 1100 M, reading A13), and print the amplitudes and local
power-law indices of every multipole.  Usage:  python -m paper_1006_0663_b200.fig1_tails [precision 1|2|4] [theta_order 2|10]
"""
from __future__ import annotations

import sys
import time

import numpy as np


def run(prec: int = 4, order: int = 10, t_end: float = 1080.0, n_ell: int = 9):
    """-> (t[steps], a[steps][n_ell]) : leading limb of Re a_l'(t) at the config-4 observer, and the wall time of the run"""
    import torch
    from . import inputs, teuk
    w = inputs.config(4).scaled(precision=prec)
    if order == 10:
        w = w.scaled(dt_override=0.5 * w.dt)
    steps = int(t_end / w.dt)
    g = teuk.Teuk.from_workload(w, obs_capacity=steps)
    g.set_option("theta_order", order)
    g.set_multipole_observer(w.rstar_obs, n_ell, steps)
    g.set_initial(inputs.initial_state(w))
    t0 = time.time()
    g.step(steps)
    torch.cuda.synchronize()
    wall = time.time() - t0
    amp = g.observe_multipoles(steps)[:, :, 0, 0].copy()
    g.close()
    return (np.arange(steps) + 1) * w.dt, amp, wall, w


def power_index(t, y, lo, hi):
    """local power-law index d ln|y| / d ln t over lo < t < hi (None if y changes sign or vanishes there)"""
    sel = (t > lo) & (t < hi)
    a = np.abs(y[sel])
    if a.min() <= 0 or np.any(np.sign(y[sel]) != np.sign(y[sel][0])):
        return None
    return float(np.polyfit(np.log(t[sel]), np.log(a), 1)[0])


def main(argv):
    prec = int(argv[1]) if len(argv) > 1 else 4
    order = int(argv[2]) if len(argv) > 2 else 10
    t, amp, wall, w = run(prec, order)
    steps = len(t)
    print(f"precision limbs {prec}, theta_order {order}: {steps} steps of {w.n_r} x {w.n_theta} in {wall:.2f} s")
    for lo, hi in ((400, 700), (700, 1050)):
        sel = (t > lo) & (t < hi)
        idx = []
        for l in range(9):
            y = np.abs(amp[sel, l])
            idx.append(None if y.min() <= 0 else round(float(np.polyfit(np.log(t[sel]), np.log(y), 1)[0]), 3))
        print(f"local power index d ln|a_l'| / d ln t for t in [{lo}, {hi}], l' = 0..8: {idx}")
    k = int(np.searchsorted(t, 1000.0))
    print("a_l'(t = 1000), l' = 0..8:", ["%.3e" % v for v in amp[k]])


if __name__ == "__main__":
    main(sys.argv)
