"""Pins P3, P8, P9 for the oracle stepper (oracle/teuk_oracle.cpp): the discrete angular operator
on known eigenfunctions, exact invariants of the iteration (Eqs. 13-14), and the
precision ladder double -> dd -> qd -> mpmath (brute force on a tiny grid)."""
import math

import numpy as np
import pytest

from oracle import mp_ref, oracle
from paper_1006_0663_b200 import inputs


def _theta(n):
    return (np.arange(n) + 0.5) * math.pi / n


# ----------------------------------------------------------------------------------------- P3
@pytest.mark.parametrize("ell", [0, 1, 2, 3, 4])
def test_lambda_on_legendre_second_order(ell):
    """Lambda_j[P_l(cos theta)] -> -l(l+1) P_l, error falling x4 per doubling of N_theta
    (second-order centred differences; even-|m| ghosts)."""
    errs = []
    for n in (16, 32, 64):
        o = oracle.Oracle(1.0, 0.0, 0, 0, 8, n, -10.0, 10.0, 0.1, 1)
        th = _theta(n)
        f = np.polynomial.legendre.Legendre.basis(ell)(np.cos(th))
        lam = o.apply_lambda(f[None, :])[0]
        errs.append(np.abs(lam + ell * (ell + 1) * f).max())
    if ell == 0:
        assert max(errs) == 0.0          # constants are annihilated exactly
    else:
        assert 3.5 < errs[0] / errs[1] < 4.5 and 3.7 < errs[1] / errs[2] < 4.3, errs


def test_lambda_spin_weighted_eigenfunction():
    """(Lambda - [(m + s cos)^2/sin^2 - s]) f = -(l-s)(l+s+1) f = -4 f for f = (1+cos)^2, s=-2, m=2."""
    errs = []
    for n in (32, 64, 128):
        o = oracle.Oracle(1.0, 0.0, -2, 2, 8, n, -10.0, 10.0, 0.1, 1)
        th = _theta(n)
        f = (1 + np.cos(th)) ** 2
        lam = o.apply_lambda(f[None, :])[0]
        pot = ((2 - 2 * np.cos(th)) ** 2 / np.sin(th) ** 2 + 2) * f
        errs.append(np.abs(lam - pot + 4 * f).max())
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.7 < errs[1] / errs[2] < 4.3, errs


def test_lambda_odd_m_ghost_sign():
    """odd |m|: Phi = 0 on the axis -> ghost f_{-1} = -f_0.  For f = sin(theta)
    (l=1, |m|=1): Lambda f - f/sin^2 = -2 f.  Away from the axis the error is second order; in the
    axis rows the 1/theta terms make it first order in max norm, but the ghost sign decides whether it
    is small at all."""
    errs, axis = [], []
    for n in (32, 64):
        o = oracle.Oracle(1.0, 0.0, 0, 1, 8, n, -10.0, 10.0, 0.1, 1)
        th = _theta(n)
        f = np.sin(th)
        res = o.apply_lambda(f[None, :])[0] - f / np.sin(th) ** 2 + 2 * f
        errs.append(np.abs(res[n // 4: 3 * n // 4]).max())
        axis.append(abs(res[0]))
    assert 3.5 < errs[0] / errs[1] < 4.5, errs
    assert axis[0] < 0.05 and axis[1] < 0.6 * axis[0]
    # the two ghost rules differ exactly by 2 f_0 (1/dtheta^2 - cot_0/(2 dtheta)) in row 0 and nowhere else
    n = 32
    th = _theta(n)
    f = np.sin(th) + 0.3
    odd = oracle.Oracle(1.0, 0.0, 0, 1, 8, n, -10.0, 10.0, 0.1, 1).apply_lambda(f[None, :])[0]
    even = oracle.Oracle(1.0, 0.0, 0, 0, 8, n, -10.0, 10.0, 0.1, 1).apply_lambda(f[None, :])[0]
    dth = math.pi / n
    assert np.array_equal(odd[1:-1], even[1:-1])
    assert abs((even[0] - odd[0]) - 2 * f[0] * (1 / dth ** 2 - 1 / math.tan(th[0]) / (2 * dth))) < 1e-9 * abs(even[0])


# ----------------------------------------------------------------------------------------- P8
def _small(w, n_r=96, steps=60, **kw):
    return w.scaled(n_r=n_r, steps=steps, **kw)


@pytest.mark.parametrize("precision", [1, 2, 4])
def test_reflection_symmetry_bitwise_cfg1(precision):
    """a = 0, s = 0: theta -> pi - theta is an exact symmetry of the discrete scheme (reading A12)."""
    w = _small(inputs.config(1), n_r=64, steps=40)
    o = oracle.Oracle.from_workload(w, precision=precision)
    o.set_initial(inputs.initial_state(w))
    o.step(w.steps)
    u = o.read()
    assert np.abs(u[0]).max() > 0.1
    assert np.array_equal(u, u[:, :, ::-1, :])
    # boundary rows exactly zero; imaginary parts exactly zero (all coefficients real)
    assert not u[:, :, :, 0].any() and not u[:, :, :, -1].any()
    assert not u[1].any() and not u[3].any()


def test_kerr_spin2_is_not_reflection_symmetric():
    """negative control for the previous test: (m + s cos)^2 breaks the symmetry."""
    w = _small(inputs.config(2), n_r=64, n_theta=8, rstar_min=-20.0, rstar_max=40.0, steps=20,
               centre=(10.0, 0.0), width=(3.0, 0.0))
    o = oracle.Oracle.from_workload(w)
    o.set_initial(inputs.initial_state(w))
    o.step(w.steps)
    u = o.read()
    assert not np.array_equal(u, u[:, :, ::-1, :])
    assert np.abs(u[1]).max() > 1e-6           # Kerr couples real and imaginary parts


@pytest.mark.parametrize("precision", [1, 2])
def test_power_of_two_linearity_and_restart(precision):
    w = _small(inputs.config(2), n_r=48, n_theta=8, rstar_min=-20.0, rstar_max=40.0, steps=30,
               centre=(10.0, 0.0), width=(3.0, 0.0))
    u0 = inputs.random_state(w.n_r, w.n_theta, precision, seed=11)
    a = oracle.Oracle.from_workload(w, precision=precision)
    a.set_initial(u0)
    a.step(30)
    ua = a.read()
    b = oracle.Oracle.from_workload(w, precision=precision)
    b.set_initial(u0 * 2.0 ** 9)
    b.step(30)
    assert np.array_equal(b.read(), ua * 2.0 ** 9)
    # checkpoint / restart: step(30) == step(12); read; set; step(18)
    c = oracle.Oracle.from_workload(w, precision=precision)
    c.set_initial(u0)
    c.step(12)
    mid = c.read()
    d = oracle.Oracle.from_workload(w, precision=precision)
    d.set_initial(mid)
    d.step(18)
    assert np.array_equal(d.read(), ua)


def test_window_interior_equals_full_grid():
    """domain of dependence i-1..i+1 per step: a window stepped alone agrees in its interior."""
    w = _small(inputs.config(2), n_r=80, n_theta=8, rstar_min=-20.0, rstar_max=40.0)
    u0 = inputs.random_state(w.n_r, w.n_theta, 1, seed=3)
    full = oracle.Oracle.from_workload(w)
    full.set_initial(u0)
    full.step(7)
    uf = full.read()
    i_lo, n_win = 20, 30
    win = oracle.Oracle.from_workload(w, i_lo=i_lo, n_win=n_win)
    win.set_initial(np.ascontiguousarray(u0[:, :, :, i_lo:i_lo + n_win]))
    win.step(7)
    uw = win.read()
    # window edge rows are zeroed at set_initial, so after k steps rows 0..k and n_win-1-k.. are off
    assert np.array_equal(uw[..., 8:n_win - 8], uf[..., i_lo + 8:i_lo + n_win - 8])
    assert not np.array_equal(uw[..., 7:n_win - 7], uf[..., i_lo + 7:i_lo + n_win - 7])


def test_observer_bilinear_matches_state():
    w = _small(inputs.config(1), n_r=64, steps=10)
    o = oracle.Oracle.from_workload(w)
    o.set_observer(40.0, 0.5 * math.pi, 10)
    o.set_initial(inputs.initial_state(w))
    o.step(10)
    u = o.read()[:, 0]
    x = (40.0 - w.rstar_min) / w.dr
    i0 = int(math.floor(x))
    wr = x - i0
    j0 = w.n_theta // 2 - 1
    expect = 0.5 * ((1 - wr) * u[:, j0, i0] + wr * u[:, j0, i0 + 1]) + 0.5 * ((1 - wr) * u[:, j0 + 1, i0] + wr * u[:, j0 + 1, i0 + 1])
    s = o.observe(10)
    assert s.shape == (10, 4, 1)
    assert np.allclose(s[-1, :, 0], expect, rtol=1e-12, atol=1e-300)


# ----------------------------------------------------------------------------------------- P9
def test_precision_ladder_against_mpmath():
    """tiny grid, Kerr a=0.9, s=-2, m=2, 20 steps: double, dd, qd oracle vs a literal mpmath
    stepper at 100 digits whose tables come straight from mpmath."""
    M, a, s, m, n_r, n_t = 1.0, 0.9, -2, 2, 24, 6
    lo, hi = -12.0, 20.0
    dt = 0.5 * (hi - lo) / (n_r - 1)
    u0 = inputs.random_state(n_r, n_t, 1, seed=5)[:, 0]
    ref = mp_ref.MPStepper(M, a, s, m, n_r, n_t, lo, hi, dt, dps=100)
    ref.set_initial(u0)
    ref.step(20)
    ref_l = np.array(ref.read_limbs(4))
    errs = {}
    for prec in (1, 2, 4):
        o = oracle.Oracle(M, a, s, m, n_r, n_t, lo, hi, dt, prec)
        o.set_initial(u0)
        o.step(20)
        got = o.read()
        pad = np.zeros_like(ref_l)
        pad[:, :prec] = got
        errs[prec] = oracle.rel_linf(pad, ref_l)
    print(errs)
    assert max(errs[1].values()) < 1e-13
    assert max(errs[2].values()) < 1e-29
    assert max(errs[4].values()) < 1e-60
    assert max(errs[1].values()) > 1e-18 and max(errs[2].values()) > 1e-36   # the ladder has rungs
