"""Pins for the oracle's FAST arithmetic tier (oracle/mpf.hpp, FP<N>; "accurate IEEE-style
additions, FMA-based twoProd").  Every operation is compared, on a corpus that includes exact
cases, sparse limbs and massive cancellation at every limb level, against
  (i)  the exact rational result (fractions.Fraction) -- the bound stated beside the operator in mpf.hpp, and
  (ii) the arbitration tier (oracle/mpx.hpp, exact-then-round), which must agree to the same bound.
The stepper built on it is compared with the arbitration-tier stepper and with the mpmath ladder, and the only
shortcuts of the tier (x + 0 = x, x * 0 = 0) are shown to change nothing."""
import math
import random
from fractions import Fraction

import numpy as np
import pytest

from oracle import mp_ref, oracle
from paper_1006_0663_b200 import inputs

U = {2: 2.0 ** -106, 4: 2.0 ** -212}                      # eps^N, eps = 2^-53
BOUND = {("add", 2): 3, ("sub", 2): 3, ("mul", 2): 5, ("mul_d", 2): 5,
         ("add", 4): 1, ("sub", 4): 1, ("mul", 4): 1, ("mul_d", 4): 1}      # <= 1 unit of eps^N: measured 0.13


def frac(limbs):
    return sum((Fraction(float(v)) for v in limbs), Fraction(0))


def normalise(total: Fraction, n):
    out = []
    for _ in range(n):
        hi = float(total)                                 # Fraction -> nearest double
        out.append(hi)
        total -= Fraction(hi)
    return out


def rand_mp(rng, n, scale_exp=0, sparse=False):
    limbs, e = [], scale_exp
    for k in range(n):
        v = math.ldexp(rng.uniform(0.5, 1.0) * rng.choice((-1, 1)), e)
        if sparse and k > 0 and rng.random() < 0.4:
            v = 0.0 if rng.random() < 0.5 else math.ldexp(v, -rng.randint(20, 200))
        limbs.append(v)
        e -= 54 + rng.randint(0, 3)
    return normalise(frac(limbs), n)


def corpus(n, op, count, seed):
    """operand pairs: generic, different scales, sparse limbs, cancellation of the leading k limbs (k = 1..n),
    nested cancellation, few-bit operands, neighbours in the last place"""
    rng = random.Random(seed)
    A, B = [], []
    for t in range(count):
        kind = t % 8
        a = rand_mp(rng, n, rng.randint(-40, 40), sparse=(kind == 2))
        b = rand_mp(rng, n, rng.randint(-40, 40), sparse=(kind == 2))
        if kind == 1:                                    # same scale
            b = rand_mp(rng, n, int(math.frexp(a[0])[1]) - rng.randint(0, 2))
        if op in ("add", "sub"):
            sgn = -1 if op == "add" else 1
            if kind in (3, 4, 5):                        # b = +-a with the limbs below level k replaced
                k = rng.randint(1, n)
                tail = rand_mp(rng, n, int(math.frexp(a[k - 1])[1]) - 53 - rng.randint(0, 60))
                b = normalise(frac(a[:k]) + frac(tail), n)
                b = [sgn * v for v in b]
            if kind == 6:                                # neighbours: b = +-(a + one unit in some limb's last place)
                k = rng.randint(0, n - 1)
                b = normalise(frac(a) + Fraction(math.ulp(a[k])) * rng.choice((-1, 1, 2, -3)), n)
                b = [sgn * v for v in b]
            if kind == 7:                                # leading limbs differ by one ulp, low limbs compensate
                b = normalise(frac(a) * (1 + Fraction(1, 2 ** rng.randint(50, 53 * n - 2))), n)
                b = [sgn * v for v in b]
        elif kind in (3, 4):                             # few significant bits: product exactly representable
            a = normalise(Fraction(rng.getrandbits(26 * n // 2) | 1) * Fraction(2) ** rng.randint(-60, 60), n)
            b = normalise(Fraction(rng.getrandbits(26 * n // 2) | 1) * Fraction(2) ** rng.randint(-60, 60), n)
        A.append(a)
        B.append(b)
    return np.array(A), np.array(B)


def loosely_normalised(limbs, slack=2.0 ** -40):
    """|x[k+1]| <= (1/2 + slack) ulp(x[k]): each limb is the rounding of what remains, up to ties"""
    for k in range(len(limbs) - 1):
        hi, lo = limbs[k], limbs[k + 1]
        if hi == 0.0:
            if lo != 0.0:
                return False
            continue
        if abs(lo) > (0.5 + slack) * math.ulp(hi):
            return False
    return True


@pytest.mark.parametrize("n", [2, 4])
@pytest.mark.parametrize("op", ["add", "sub", "mul", "mul_d"])
def test_fast_tier_against_exact_rationals_and_arbitration_tier(n, op):
    A, B = corpus(n, op, 2400, seed=1000 * n + len(op))
    if op == "mul_d":
        B[:, 1:] = 0.0
    fast = oracle.mp_op_batch(op, n, A, B, tier="fast")
    slow = oracle.mp_op_batch(op, n, A, B, tier="exact")
    worst_exact = worst_tier = 0.0
    exact_hits = 0
    for a, b, f, s in zip(A, B, fast, slow):
        fa, fb = frac(a), frac(b)
        exact = {"add": fa + fb, "sub": fa - fb, "mul": fa * fb, "mul_d": fa * Fraction(float(b[0]))}[op]
        ff, fs = frac(f), frac(s)
        if exact == 0:
            assert ff == 0 and fs == 0
            continue
        e1 = float(abs((ff - exact) / exact))
        e2 = float(abs((ff - fs) / exact))
        worst_exact, worst_tier = max(worst_exact, e1), max(worst_tier, e2)
        assert e1 <= BOUND[(op, n)] * U[n], (list(a), list(b), list(f), e1 / U[n])
        assert e2 <= BOUND[(op, n)] * U[n]
        assert loosely_normalised(list(f)), list(f)
        # N = 4 (merge / cascade + distillation: every step before the last rounding is error-free): a result that
        # fits in n limbs must come back exact.  The textbook N = 2 algorithms do not promise that.
        if frac(normalise(exact, n)) == exact:
            exact_hits += 1
            if n == 4:
                assert ff == exact, (list(a), list(b), list(f))
    print(op, n, "worst error / eps^N vs exact:", worst_exact / U[n], "vs arbitration tier:", worst_tier / U[n],
          "exactly representable cases:", exact_hits)
    assert exact_hits > 100


@pytest.mark.parametrize("n", [2, 4])
def test_fast_tier_identities(n):
    rng = random.Random(11)
    for _ in range(50):
        x = rand_mp(rng, n, rng.randint(-30, 30))
        assert oracle.mp_op("sub", n, x, x, tier="fast") == [0.0] * n
        assert oracle.mp_op("half", n, x, tier="fast") == oracle.mp_op("mul_d", n, x, [0.5], tier="exact")
        assert frac(oracle.mp_op("mul_d", n, x, [2.0 ** 17], tier="fast")) == frac(x) * 2 ** 17
        y = rng.uniform(-10, 10)
        assert oracle.mp_op("add", n, [x[0]], [y], tier="fast")[0] == x[0] + y
        assert frac(oracle.mp_op("mul", n, [x[0]], [y], tier="fast")) == Fraction(x[0]) * Fraction(y)
    a, b = [1.0, 2.0 ** -60], [1.0, -(2.0 ** -60)]
    assert frac(oracle.mp_op("add", n, a, b, tier="fast")) == 2
    assert frac(oracle.mp_op("mul", n, [2.0 ** 30 + 1], [2.0 ** 30 - 1], tier="fast")) == 2 ** 60 - 1


@pytest.mark.parametrize("n", [2, 4])
def test_zero_shortcuts_change_nothing(n):
    """x + 0, 0 + x, x * 0 through the general path give the same limbs as the shortcut"""
    rng = random.Random(12)
    xs = [rand_mp(rng, n, rng.randint(-30, 30), sparse=(k % 2 == 0)) for k in range(100)]
    zero = [0.0] * n
    old = oracle.set_zero_fast_path(False)
    try:
        general = [(oracle.mp_op("add", n, x, zero, tier="fast"), oracle.mp_op("add", n, zero, x, tier="fast"),
                    oracle.mp_op("mul", n, x, zero, tier="fast"), oracle.mp_op("mul_d", n, x, [0.0], tier="fast"))
                   for x in xs]
    finally:
        oracle.set_zero_fast_path(old)
    for x, g in zip(xs, general):
        assert g[0] == x and g[1] == x and g[2] == zero and g[3] == zero
        assert oracle.mp_op("add", n, x, zero, tier="fast") == x
        assert oracle.mp_op("mul", n, x, zero, tier="fast") == zero


def _run(prec, tier, steps, a=0.9, s=-2, m=2, n_r=40, n_t=8, theta_order=2, seed=5):
    lo, hi = -12.0, 20.0
    dt = 0.25 * (hi - lo) / (n_r - 1)
    o = oracle.Oracle(1.0, a, s, m, n_r, n_t, lo, hi, dt, prec, theta_order=theta_order, tier=tier)
    o.set_observer(3.3, 1.1, steps)
    o.set_initial(inputs.random_state(n_r, n_t, prec, seed=seed))
    o.step(steps)
    return o.read(), o.observe(steps)


@pytest.mark.parametrize("prec,tol", [(2, 1e-29), (4, 1e-61)])
@pytest.mark.parametrize("theta_order", [2, 10])
def test_fast_stepper_matches_arbitration_stepper(prec, tol, theta_order):
    """same template, two arithmetic tiers: Kerr, complex coefficients, all limbs populated, 60 steps"""
    n_t = 8 if theta_order == 2 else 12
    u_f, s_f = _run(prec, "fast", 60, n_t=n_t, theta_order=theta_order)
    u_e, s_e = _run(prec, "exact", 60, n_t=n_t, theta_order=theta_order)
    err = oracle.rel_linf(u_f, u_e)
    so = oracle.rel_linf(np.moveaxis(s_f, 0, -1), np.moveaxis(s_e, 0, -1))
    print(prec, theta_order, err, so)
    assert max(err.values()) < tol and max(so.values()) < tol
    assert np.all(u_f[:, :, :, 0] == 0.0) and np.all(u_f[:, :, :, -1] == 0.0)


def test_fast_stepper_zero_shortcuts_are_bitwise_neutral():
    """a REAL problem (a = 0.5, s = m = 0, real data: config 4's structure): imaginary parts stay exactly zero and
    the run is bit-identical with the shortcuts switched off"""
    w = inputs.config(4).scaled(n_r=48, n_theta=8, rstar_min=-20.0, rstar_max=60.0)
    u0 = inputs.initial_state(w)
    res = []
    for on in (True, False):
        old = oracle.set_zero_fast_path(on)
        try:
            o = oracle.Oracle.from_workload(w, tier="fast")
            o.set_initial(u0)
            o.step(40)
            res.append(o.read())
        finally:
            oracle.set_zero_fast_path(old)
    assert np.array_equal(res[0], res[1])
    assert np.all(res[0][1] == 0.0) and np.all(res[0][3] == 0.0) and np.abs(res[0][0, 0]).max() > 0


def test_precision_ladder_against_mpmath_fast_tier():
    """the ladder of tests/test_oracle_invariants.py::test_precision_ladder_against_mpmath with the fast tier:
    dd and qd land on the same rungs"""
    M, a, s, m, n_r, n_t = 1.0, 0.9, -2, 2, 24, 6
    lo, hi = -12.0, 20.0
    dt = 0.5 * (hi - lo) / (n_r - 1)
    u0 = inputs.random_state(n_r, n_t, 1, seed=5)[:, 0]
    ref = mp_ref.MPStepper(M, a, s, m, n_r, n_t, lo, hi, dt, dps=100)
    ref.set_initial(u0)
    ref.step(20)
    ref_l = np.array(ref.read_limbs(4))
    errs = {}
    for prec in (2, 4):
        o = oracle.Oracle(M, a, s, m, n_r, n_t, lo, hi, dt, prec, tier="fast")
        o.set_initial(u0)
        o.step(20)
        pad = np.zeros_like(ref_l)
        pad[:, :prec] = o.read()
        errs[prec] = oracle.rel_linf(pad, ref_l)
    print(errs)
    assert max(errs[2].values()) < 1e-29 and max(errs[4].values()) < 1e-60
    assert max(errs[2].values()) > 1e-36
