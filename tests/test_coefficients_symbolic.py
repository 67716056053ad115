"""Pin P2 (symbolic): the coefficients the oracle uses (oracle/mp_ref.py::coefficients,
DESIGN.md §3) reproduce the Teukolsky master equation, Eq. (1), after the
coordinate change Eqs. (2)-(3) PAPER.md:59-63 and the ansatz Eq. (4) PAPER.md:67.

The paper does not print the matrices M, A, L, so this test is what ties the
derived alpha, beta, kappa, W (and gamma, b_*, g_*) to what the paper does print.

Method: Eq.(1)[e^{i m (phi+h(r))} r^p Phi] / (e^{...} r^p) + (Sigma^2/Delta) * (S0) == 0 with
  S0 = Phi_tt - b^2 Phi_** + alpha Phi_t - beta Phi_* - kappa (Phi_thth + cot Phi_th) + W Phi,
  d_* = (Delta/(r^2+a^2)) d_r, h'(r) = a/Delta,
evaluated at random rational points with every derivative of Phi replaced by an independent
random complex number (so the identity must hold coefficient by coefficient).
Negative controls perturb one constant and must give an O(1) residual.
"""
import random

import pytest
import sympy as sp

from oracle import mp_ref


def _build_residual(s_val, p_val, tweak=None):
    t, r, th, ph = sp.symbols("t r theta phi", real=True)
    M, a = sp.symbols("M a", positive=True)
    m = sp.Symbol("m", real=True)
    s = sp.Integer(s_val)
    p = sp.Integer(p_val)
    Delta = r ** 2 - 2 * M * r + a ** 2
    R = r ** 2 + a ** 2
    h = sp.Function("h")(r)
    Phi = sp.Function("Phi")(t, r, th)
    Psi = sp.exp(sp.I * m * (ph + h)) * r ** p * Phi

    # Eq. (1), term by term
    eq1 = (-(R ** 2 / Delta - a ** 2 * sp.sin(th) ** 2) * sp.diff(Psi, t, 2)
           - 4 * M * a * r / Delta * sp.diff(Psi, t, ph)
           - 2 * s * (r - M * (r ** 2 - a ** 2) / Delta + sp.I * a * sp.cos(th)) * sp.diff(Psi, t)
           + Delta ** (-s) * sp.diff(Delta ** (s + 1) * sp.diff(Psi, r), r)
           + 1 / sp.sin(th) * sp.diff(sp.sin(th) * sp.diff(Psi, th), th)
           + (1 / sp.sin(th) ** 2 - a ** 2 / Delta) * sp.diff(Psi, ph, 2)
           + 2 * s * (a * (r - M) / Delta + sp.I * sp.cos(th) / sp.sin(th) ** 2) * sp.diff(Psi, ph)
           - (s ** 2 * sp.cot(th) ** 2 - s) * Psi)
    eq1 = eq1.doit()
    hp = a / Delta                                           # Eq. (3)
    eq1 = eq1.subs(sp.Derivative(h, (r, 2)), sp.diff(hp, r)).subs(sp.Derivative(h, r), hp)
    eq1 = sp.expand(eq1 / (sp.exp(sp.I * m * (ph + h)) * r ** p))

    # the oracle's coefficient function on sympy symbols; delta_h = r - r_+ enters only via Delta
    rp = M + sp.sqrt(M ** 2 - a ** 2)
    rm = M - sp.sqrt(M ** 2 - a ** 2)
    c = mp_ref.coefficients(r, r - rp, sp.sin(th), sp.cos(th), M, a, s, m, rp - rm, sqrt=sp.sqrt, p=p)
    alpha = c["alpha"][0] + sp.I * c["alpha"][1]
    beta = c["beta"][0] + sp.I * c["beta"][1]
    W = c["W"][0] + sp.I * c["W"][1]
    if tweak == "alpha":        # 4 m M a r -> 5 m M a r
        alpha = alpha + sp.I * m * M * a * r / c["Sigma2"]
    if tweak == "V":            # 4 m a s (r-M) -> 3 m a s (r-M)
        W = W + sp.I * m * a * s * (r - M) / c["Sigma2"]
    b, kappa = c["b"], c["kappa"]
    dstar = lambda f: (Delta / R) * sp.diff(f, r)           # Eq. (2)
    S0 = (sp.diff(Phi, t, 2) - b ** 2 * dstar(dstar(Phi)) + alpha * sp.diff(Phi, t) - beta * dstar(Phi)
          - kappa * (sp.diff(Phi, th, 2) + sp.cos(th) / sp.sin(th) * sp.diff(Phi, th)) + W * Phi)
    res = eq1 + (c["Sigma2"] / Delta) * S0
    # replace Phi and its derivatives by independent symbols
    derivs = sorted(res.atoms(sp.Derivative), key=str)
    subs = {d: sp.Symbol(f"D{k}") for k, d in enumerate(derivs)}
    res = res.subs(subs).subs(Phi, sp.Symbol("D_phi"))
    return res, (t, r, th, ph, M, a, m), list(subs.values()) + [sp.Symbol("D_phi")]


def _evaluate(res, syms, dsyms, rng):
    t, r, th, ph, M, a, m = syms
    vals = {r: sp.Rational(rng.randint(300, 900), 100), th: sp.Rational(rng.randint(20, 290), 100),
            a: sp.Rational(rng.randint(10, 90), 100), M: 1, m: rng.randint(-3, 3),
            t: sp.Rational(rng.randint(0, 100), 10), ph: sp.Rational(rng.randint(0, 60), 10)}
    for d in dsyms:
        vals[d] = sp.Rational(rng.randint(-99, 99), 37) + sp.I * sp.Rational(rng.randint(-99, 99), 41)
    return abs(sp.N(res.subs(vals), 50))


@pytest.mark.parametrize("s_val,p_val", [(0, 3), (-2, 3), (-1, 3), (2, 3), (1, 0), (0, -1), (-2, 0)])
def test_residual_vanishes(s_val, p_val):
    res, syms, dsyms = _build_residual(s_val, p_val)
    rng = random.Random(1006 + 10 * s_val + p_val)
    for _ in range(3):
        assert _evaluate(res, syms, dsyms, rng) < 1e-40


@pytest.mark.parametrize("tweak", ["alpha", "V"])
def test_negative_control_has_power(tweak):
    res, syms, dsyms = _build_residual(-2, 3, tweak=tweak)
    rng = random.Random(7)
    vals = [_evaluate(res, syms, dsyms, rng) for _ in range(3)]
    assert min(vals) > 1e-3


def test_closed_forms_bstar_gstar_and_first_order_form():
    r, th = sp.symbols("r theta", real=True)
    M, a = sp.symbols("M a", positive=True)
    Delta = r ** 2 - 2 * M * r + a ** 2
    R = r ** 2 + a ** 2
    rp = M + sp.sqrt(M ** 2 - a ** 2)
    rm = M - sp.sqrt(M ** 2 - a ** 2)
    c = mp_ref.coefficients(r, r - rp, sp.sin(th), sp.cos(th), M, a, sp.Integer(-2), sp.Integer(2),
                            rp - rm, sqrt=sp.sqrt, p=sp.Integer(3))
    dstar = lambda f: (Delta / R) * sp.diff(f, r)
    pt = {r: sp.Rational(47, 10), th: sp.Rational(11, 10), a: sp.Rational(7, 10), M: 1}
    # b_* = d_* b and g_* = d_* g with g = p Delta / (r R)
    assert abs(sp.N((dstar(c["b"]) - c["b_star"]).subs(pt), 40)) < 1e-30
    assert abs(sp.N((dstar(c["g"]) - c["g_star"]).subs(pt), 40)) < 1e-30
    # gamma = alpha b + beta - b b_*   (Pi_t - b Pi_* = Phi_tt - b^2 Phi_** - b b_* Phi_*, Eq. (5))
    for k in (0, 1):
        bb = c["b_star"] * c["b"] if k == 0 else 0
        lhs = c["gamma"][k]
        rhs = c["alpha"][k] * c["b"] + c["beta"][k] - bb
        assert abs(sp.N((lhs - rhs).subs(pt), 40)) < 1e-30


def test_schwarzschild_limits():
    """a = 0, s = 0, m = 0, p = 3: alpha = 0, beta = 8(r-2M)/r^2, kappa = f/r^2,
    W = -6 (r-2M)(2r-3M)/r^4 (Regge-Wheeler form for psi = r^4 Phi).
    a = 0, s = -2: alpha = -4(r-3M)/r^2, gamma = 0."""
    import mpmath as mp
    with mp.workdps(50):
        r, M = mp.mpf("7.3"), mp.mpf(1)
        c = mp_ref.coefficients(r, r - 2 * M, mp.sin(1.1), mp.cos(1.1), M, mp.mpf(0), 0, 0, 2 * M)
        f = 1 - 2 * M / r
        assert abs(c["alpha"][0]) < 1e-45 and abs(c["alpha"][1]) < 1e-45
        assert abs(c["beta"][0] - 8 * (r - 2 * M) / r ** 2) < 1e-45
        assert abs(c["kappa"] - f / r ** 2) < 1e-45
        assert abs(c["W"][0] + 6 * (r - 2 * M) * (2 * r - 3 * M) / r ** 4) < 1e-45
        assert abs(c["b"] - 1) < 1e-45
        c2 = mp_ref.coefficients(r, r - 2 * M, mp.sin(1.1), mp.cos(1.1), M, mp.mpf(0), -2, 2, 2 * M)
        assert abs(c2["alpha"][0] + 4 * (r - 3 * M) / r ** 2) < 1e-45
        assert abs(c2["gamma"][0]) < 1e-45 and abs(c2["gamma"][1]) < 1e-45
