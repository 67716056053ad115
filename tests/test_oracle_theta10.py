"""NEXT-1 pins: the 10th-order angular operator ("we choose the finite-difference angular
differentiation operator to be 10th-order accurate and leave the rest ... 2nd-order Lax-Wendroff")."""
import math
from fractions import Fraction
from math import factorial

import numpy as np
import pytest

from oracle import mp_ref, oracle
from paper_1006_0663_b200 import inputs


def test_weights_match_textbook_closed_form_and_are_exact_on_polynomials():
    """centred stencils of order 2N: c_k = (-1)^(k+1) (N!)^2 / (k (N-k)! (N+k)!), d_k = 2 c_k / k (textbook,
    Fornberg 1988) — an independent route to what fd_weights gets from the Taylor conditions"""
    for order in (2, 10):
        N = order // 2
        c, d = mp_ref.fd_weights(order)
        for k in range(1, N + 1):
            ck = Fraction((-1) ** (k + 1) * factorial(N) ** 2, k * factorial(N - k) * factorial(N + k))
            assert c[k - 1] == ck
            assert d[k] == 2 * ck / k
        assert d[0] == -2 * sum(d[1:])
        # exact on monomials x^p, p <= 2N, at x = 0 (h = 1)
        for p in range(0, 2 * N + 1):
            f = lambda x: Fraction(x) ** p
            d1 = sum(c[k - 1] * (f(k) - f(-k)) for k in range(1, N + 1))
            d2 = d[0] * f(0) + sum(d[k] * (f(k) + f(-k)) for k in range(1, N + 1))
            assert d1 == (1 if p == 1 else 0)
            assert d2 == (2 if p == 2 else 0)


@pytest.mark.parametrize("ell", [4, 6, 8])
def test_lambda10_converges_at_tenth_order(ell):
    errs = []
    for n in (16, 32, 64):
        o = oracle.Oracle(1.0, 0.0, 0, 0, 8, n, -10.0, 10.0, 0.1, 2, theta_order=10)
        th = (np.arange(n) + 0.5) * math.pi / n
        f = np.zeros((2, n))
        f[0] = np.polynomial.legendre.Legendre.basis(ell)(np.cos(th))
        lam = o.apply_lambda(f)
        errs.append(np.abs(lam[0] + lam[1] + ell * (ell + 1) * f[0]).max())
    # 2^10 = 1024 asymptotically; the inputs are doubles, so the finest grid may sit on the 1e-13 rounding floor
    assert errs[0] / errs[1] > 300 and (errs[1] / errs[2] > 300 or errs[2] < 2e-12), errs
    # spin-weighted eigenfunction (s = -2, m = 2): (Lambda - pole potential) f = -4 f
    o = oracle.Oracle(1.0, 0.0, -2, 2, 8, 64, -10.0, 10.0, 0.1, 2, theta_order=10)
    th = (np.arange(64) + 0.5) * math.pi / 64
    f = np.zeros((2, 64))
    f[0] = (1 + np.cos(th)) ** 2
    lam = o.apply_lambda(f)
    pot = ((2 - 2 * np.cos(th)) ** 2 / np.sin(th) ** 2 + 2) * f[0]
    assert np.abs(lam[0] + lam[1] - pot + 4 * f[0]).max() < 1e-8


def test_theta10_precision_ladder_and_symmetry():
    M, a, s, m, n_r, n_t = 1.0, 0.9, -2, 2, 20, 12
    lo, hi = -12.0, 20.0
    dt = 0.05 * (hi - lo) / (n_r - 1)
    u0 = inputs.random_state(n_r, n_t, 1, seed=6)[:, 0]
    ref = mp_ref.MPStepper(M, a, s, m, n_r, n_t, lo, hi, dt, dps=100, theta_order=10)
    ref.set_initial(u0)
    ref.step(12)
    ref_l = np.array(ref.read_limbs(4))
    bound = {1: 1e-13, 2: 1e-29, 4: 1e-60}
    for prec in (1, 2, 4):
        o = oracle.Oracle(M, a, s, m, n_r, n_t, lo, hi, dt, prec, theta_order=10)
        o.set_initial(u0)
        o.step(12)
        pad = np.zeros_like(ref_l)
        pad[:, :prec] = o.read()
        err = oracle.rel_linf(pad, ref_l)
        assert max(err.values()) < bound[prec], (prec, err)
    # the 10th-order and 2nd-order operators give different (but close) answers: the option is live
    o2 = oracle.Oracle(M, a, s, m, n_r, n_t, lo, hi, dt, 1)
    o2.set_initial(u0)
    o2.step(12)
    o10 = oracle.Oracle(M, a, s, m, n_r, n_t, lo, hi, dt, 1, theta_order=10)
    o10.set_initial(u0)
    o10.step(12)
    diff = np.abs(o2.read() - o10.read()).max()
    assert 1e-9 < diff < 0.5
    # reflection symmetry stays bit-exact for a = 0, s = 0 with the wide stencil
    w = inputs.config(1).scaled(n_r=48, steps=30)
    o = oracle.Oracle.from_workload(w, theta_order=10)
    o.set_initial(inputs.initial_state(w))
    o.step(30)
    u = o.read()
    assert np.array_equal(u, u[:, :, ::-1, :])
