"""Fig. 1 workload of the paper on the GPU path: pure l = 0 data in Kerr (BASELINE.json config 4:
a = 0.5, s = m = 0, 8192 x 32), 10th-order theta operator, multipole-projection observer l' = 0..8, run up
to the first echo of the radial Dirichlet walls (t ~ 1100 M, reading A13), and print the amplitudes and local
power-law indices of every multipole.  Usage:  python -m paper_1006_0663_b200.fig1_tails [precision 1|2|4] [theta_order 2|10]
"""
from __future__ import annotations

import sys
import time

import numpy as np


def main(argv):
    import torch
    from . import inputs, teuk
    prec = int(argv[1]) if len(argv) > 1 else 4
    order = int(argv[2]) if len(argv) > 2 else 10
    w = inputs.config(4).scaled(precision=prec)
    if order == 10:
        w = w.scaled(dt_override=0.5 * w.dt)
    steps = int(1080.0 / w.dt)
    g = teuk.Teuk.from_workload(w, obs_capacity=steps)
    g.set_option("theta_order", order)
    g.set_multipole_observer(w.rstar_obs, 9, steps)
    g.set_initial(inputs.initial_state(w))
    t0 = time.time()
    g.step(steps)
    torch.cuda.synchronize()
    print(f"precision limbs {prec}, theta_order {order}: {steps} steps of {w.n_r} x {w.n_theta} in {time.time() - t0:.2f} s")
    amp = g.observe_multipoles(steps)[:, :, 0, 0]
    t = (np.arange(steps) + 1) * w.dt
    for lo, hi in ((400, 700), (700, 1050)):
        sel = (t > lo) & (t < hi)
        idx = []
        for l in range(9):
            y = np.abs(amp[sel, l])
            idx.append(None if y.min() <= 0 else round(float(np.polyfit(np.log(t[sel]), np.log(y), 1)[0]), 3))
        print(f"local power index d ln|a_l'| / d ln t for t in [{lo}, {hi}], l' = 0..8: {idx}")
    k = int(np.searchsorted(t, 1000.0))
    print("a_l'(t = 1000), l' = 0..8:", ["%.3e" % v for v in amp[k]])
    g.close()


if __name__ == "__main__":
    main(sys.argv)
