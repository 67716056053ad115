"""Pins P4-P7 for the oracle: what the paper and textbook black-hole perturbation theory fix.

P4  second-order convergence of the whole Lax-Wendroff scheme.
P5  a = 0, s = 0 reduces to the textbook 1+1D Regge-Wheeler equation for psi = r^4 Phi; an
    independent leapfrog solver (own r(r*) through the Lambert-W closed form) must agree.
P6  quasinormal ringing: Schwarzschild l=2 fundamental modes,
    s=0: M omega = 0.4836 - 0.0968i, |s|=2: 0.3737 - 0.0890i (north_star; reading A23).
P7  late-time tail t^-(2l+3) for a = 0, l = 0.
"""
import math
import os

import numpy as np
import pytest
from scipy.special import lambertw

from oracle import oracle
from paper_1006_0663_b200 import inputs


def _lambda_matrix(n):
    """even-|m| discrete angular operator as a dense matrix, typed from PAPER.md:110-112."""
    dth = math.pi / n
    th = (np.arange(n) + 0.5) * dth
    A = np.zeros((n, n))
    for j in range(n):
        jm, jp = (j - 1 if j > 0 else 0), (j + 1 if j < n - 1 else n - 1)
        A[j, jp] += 1 / dth ** 2 + 1 / math.tan(th[j]) / (2 * dth)
        A[j, jm] += 1 / dth ** 2 - 1 / math.tan(th[j]) / (2 * dth)
        A[j, j] += -2 / dth ** 2
    return A, th


def _rw_leapfrog(rs, r, psi0, psit0, lam, dt, n_steps, rec_index):
    """psi_tt = psi_** - f (lam/r^2 + 2M/r^3) psi, M = 1, standard 3-level leapfrog, psi = 0 at the ends."""
    f = 1 - 2 / r
    V = f * (lam / r ** 2 + 2 / r ** 3)
    dr = rs[1] - rs[0]

    def rhs(p):
        out = np.zeros_like(p)
        out[1:-1] = (p[2:] - 2 * p[1:-1] + p[:-2]) / dr ** 2 - V[1:-1] * p[1:-1]
        return out
    prev = psi0.copy()
    cur = psi0 + dt * psit0 + 0.5 * dt ** 2 * rhs(psi0)
    cur[0] = cur[-1] = 0
    series = [cur[rec_index]]
    for _ in range(n_steps - 1):
        nxt = 2 * cur - prev + dt ** 2 * rhs(cur)
        nxt[0] = nxt[-1] = 0
        prev, cur = cur, nxt
        series.append(cur[rec_index])
    return np.array(series)


# ----------------------------------------------------------------------------------------- P5
def test_schwarzschild_scalar_reduces_to_regge_wheeler():
    n_t = 8
    A, th = _lambda_matrix(n_t)
    evals, evecs = np.linalg.eig(A)
    k = int(np.argmin(np.abs(evals.real + 6)))           # the discrete l = 2 mode
    lam = -evals[k].real
    vec = evecs[:, k].real
    vec /= vec[np.argmax(np.abs(vec))]
    assert abs(lam - 6) < 0.5                            # N_theta = 8: discrete l(l+1) = 5.6
    diffs = []
    for n_r in (401, 801):
        lo, hi = -40.0, 60.0
        dr = (hi - lo) / (n_r - 1)
        dt = 0.5 * dr
        rs = lo + np.arange(n_r) * dr
        r = 2 * (1 + np.real(lambertw(np.exp(rs / 2 - 1))))      # r* = r + 2 ln(r/2 - 1) inverted
        g = np.exp(-(rs - 15.0) ** 2 / (2 * 3.0 ** 2))
        u0 = np.zeros((4, n_t, n_r))
        u0[0] = vec[:, None] * g[None, :]
        o = oracle.Oracle(1.0, 0.0, 0, 0, n_r, n_t, lo, hi, dt, 1)
        steps = int(round(60.0 / dt))
        i_obs = int(round((30.0 - lo) / dr))
        o.set_initial(u0)
        prof_err = 0.0
        series = []
        for _ in range(steps // 20):
            o.step(20)
            u = o.read()[:, 0]
            series.append(u[0, :, i_obs] @ vec / (vec @ vec))
            col = u[0, :, i_obs]
            prof_err = max(prof_err, np.abs(col - series[-1] * vec).max() / np.abs(u[0]).max())
        assert prof_err < 1e-12                                   # theta-profile stays the eigenvector
        # Pi = 0 means Phi_t = -b Phi_* = -Phi_* (a = 0): psi_t = -r^4 Phi_*
        psi0 = r ** 4 * g
        dg = -(rs - 15.0) / 9.0 * g
        ref = _rw_leapfrog(rs, r, psi0, -r ** 4 * dg, lam, dt, steps, i_obs)
        ref = ref[19::20] / r[i_obs] ** 4
        series = np.array(series)
        diffs.append(np.abs(series - ref).max() / np.abs(ref).max())
    print("RW agreement:", diffs)
    assert diffs[1] < 2e-3 and 3.0 < diffs[0] / diffs[1] < 5.0


# ----------------------------------------------------------------------------------------- P6
def _fit_qnm(t, x):
    """x(t) ~ Re(A exp(-i w t)): two-term linear prediction x_{k+2} = c1 x_{k+1} + c2 x_k."""
    Amat = np.stack([x[1:-1], x[:-2]], axis=1)
    c1, c2 = np.linalg.lstsq(Amat, x[2:], rcond=None)[0]
    z = np.roots([1, -c1, -c2])
    z = z[np.argmax(z.imag)]
    dt = t[1] - t[0]
    w = 1j * np.log(z) / dt                # z = exp(-i w dt)
    return complex(abs(w.real), w.imag)


def _golden(name):
    """rows of a tests/golden/ fixture (whitespace-separated, '#' comments); every file cites where its values come from"""
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    return [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")]


def _qnm(abs_s):
    row = [r for r in _golden("qnm_frequencies.txt") if int(r[0]) == abs_s and int(r[1]) == 2][0]
    return complex(float(row[2]), float(row[3]))


@pytest.mark.parametrize("s,m,profile", [(0, 0, "P2"), (-2, 2, "Y22m2")])
def test_quasinormal_ringing(s, m, profile):
    """BASELINE.json config-1 grid and data; the second case is the |s| = 2 companion run of reading A23.
    Expected frequencies: tests/golden/qnm_frequencies.txt."""
    expect = _qnm(abs(s))
    w = inputs.config(1).scaled(s=s, m=m, profile=profile)
    w = w.scaled(dt_override=inputs.stable_dt(w))              # reading A15b: s=-2 needs the reduced dt
    o = oracle.Oracle.from_workload(w)
    o.set_observer(40.0, 0.5 * math.pi, w.steps)
    o.set_initial(inputs.initial_state(w))
    steps = int(176.0 / w.dt)                               # t = 176 < first wall echo at t ~ 180 (A13)
    o.set_observer(40.0, 0.5 * math.pi, steps)
    o.step(steps)
    ser = o.observe(steps)[:, 0, 0]
    t = (np.arange(len(ser)) + 1) * w.dt
    sel = (t > 95) & (t < 150)
    stride = max(1, int(round(1.5 / w.dt)))
    omega = _fit_qnm(t[sel][::stride], ser[sel][::stride])
    print("fitted M omega =", omega)
    assert abs(omega.real - expect.real) / expect.real < 0.02
    assert abs(omega.imag - expect.imag) / abs(expect.imag) < 0.05


# ----------------------------------------------------------------------------------------- P4
def test_second_order_convergence_kerr():
    vals = []
    for k in (2, 4, 8):
        n_r, n_t = 60 * k + 1, 6 * k
        lo, hi = -20.0, 40.0
        dr = (hi - lo) / (n_r - 1)
        w = inputs.config(2).scaled(n_r=n_r, n_theta=n_t, rstar_min=lo, rstar_max=hi, centre=(8.0, 0.0),
                                    width=(4.0, 0.0), dt_override=0.1 * dr)
        o = oracle.Oracle.from_workload(w)
        steps = int(round(12.0 / w.dt))
        o.set_observer(10.0, 0.5 * math.pi, steps)
        o.set_initial(inputs.initial_state(w))
        o.step(steps)
        s_ = o.observe(steps)[:, :, 0]
        pick = [steps // 2 - 1, 3 * steps // 4 - 1, steps - 1]
        vals.append(s_[pick, 0] + 1j * s_[pick, 1])
    e1 = np.abs(vals[0] - vals[1])
    e2 = np.abs(vals[1] - vals[2])
    ratio = e1 / e2
    print("Richardson ratios:", ratio)
    assert np.all(ratio > 3.4) and np.all(ratio < 4.6)


# ----------------------------------------------------------------------------------------- P7
def test_late_time_tail_l0():
    """a = 0, l = 0 data: local power index -> -(2l+3) = -3.  Sanity pin (slow approach)."""
    lo, hi = -480.0, 600.0
    n_r, n_t = 4321, 4
    dr = (hi - lo) / (n_r - 1)
    w = inputs.config(4).scaled(a=0.0, n_r=n_r, n_theta=n_t, rstar_min=lo, rstar_max=hi, precision=1,
                                centre=(20.0, 0.0), width=(4.0, 0.0))
    o = oracle.Oracle.from_workload(w)
    steps = int(round(1000.0 / w.dt))
    o.set_observer(40.0, 0.5 * math.pi, steps)
    o.set_initial(inputs.initial_state(w))
    o.step(steps)
    ser = o.observe(steps)[:, 0, 0]
    t = (np.arange(steps) + 1) * w.dt
    sel = (t > 600) & (t < 1000)
    idx = np.polyfit(np.log(t[sel]), np.log(np.abs(ser[sel])), 1)[0]
    print("tail index", idx)
    n = [int(r[3]) for r in _golden("tail_exponents.txt") if r[0] == "0.0" and r[1] == "0" and r[2] == "0"][0]   # 2l+3 = 3
    assert n == 3 and -n - 0.3 < idx < -n + 0.3
    assert np.all(np.sign(ser[sel]) == np.sign(ser[sel][0]))    # no oscillation left: a pure power law
