"""B0 pins: the CUDA path's own multiprecision layer (csrc/mp.cuh, setup_math.cuh), compiled for the host
inside libteuk.so and driven through the C ABI test hooks — no GPU needed.  Same style of pins as
tests/test_oracle_arith.py (exact rationals, mpmath), but the two arithmetic layers share no code.
The device build of the same header is checked bit-for-bit against the host build in test_gpu_parity.py."""
import math
import random
from fractions import Fraction

import mpmath as mp
import numpy as np
import pytest

teuk = pytest.importorskip("paper_1006_0663_b200.teuk")

EPS = {2: 2.0 ** -104, 4: 2.0 ** -205}


def frac(limbs):
    return sum((Fraction(float(v)) for v in limbs), Fraction(0))


def rand_mp(rng, n, scale_exp=0):
    limbs, e = [], scale_exp
    for _ in range(n):
        limbs.append(math.ldexp(rng.uniform(0.5, 1.0) * rng.choice((-1, 1)), e))
        e -= 54 + rng.randint(0, 3)
    total, out = frac(limbs), []
    for _ in range(n):
        hi = float(total)
        out.append(hi)
        total -= Fraction(hi)
    return out


def op1(op, n, a, b):
    a = list(a) + [0.0] * (n - len(a))
    b = list(b) + [0.0] * (n - len(b))
    return [float(v) for v in teuk.test_mp_op(op, n, np.array([a]), np.array([b]), on_device=False)[0]]


@pytest.mark.parametrize("n", [2, 4])
def test_exact_cases(n):
    assert frac(op1("add", n, [1.0, 2.0 ** -60], [1.0, -(2.0 ** -60)])) == 2
    assert frac(op1("mul", n, [2.0 ** 30 + 1], [2.0 ** 30 - 1])) == 2 ** 60 - 1
    rng = random.Random(5)
    x = rand_mp(rng, n)
    assert frac(op1("sub", n, x, x)) == 0
    assert frac(op1("add", n, x, [0.0])) == frac(x)
    assert frac(op1("mul_d", n, x, [2.0 ** 17])) == frac(x) * 2 ** 17
    assert frac(op1("mul", n, x, [0.5])) == frac(x) / 2
    for p, q in [(1, 3), (22, 7), (-5, 11)]:
        quo = op1("div", n, [float(p)], [float(q)])
        assert abs(frac(quo) - Fraction(p, q)) <= 4 * EPS[n] * abs(Fraction(p, q))


@pytest.mark.parametrize("n", [2, 4])
@pytest.mark.parametrize("op", ["add", "sub", "mul", "div"])
def test_random_against_exact_rationals(n, op):
    rng = random.Random(100 * n + len(op))
    A, B = [], []
    for trial in range(400):
        a = rand_mp(rng, n, rng.randint(-40, 40))
        b = rand_mp(rng, n, rng.randint(-40, 40))
        if trial % 3 == 0 and op in ("add", "sub"):        # massive cancellation
            b = list(a)
            b[n - 1] = b[n - 1] * (1 + rng.uniform(-0.5, 0.5))
            if op == "add":
                b = [-v for v in b]
        if trial % 3 == 1 and op in ("add", "sub"):        # partial cancellation in the leading limbs
            b = list(a)
            b[1] = b[1] * (1 + rng.uniform(-0.5, 0.5))
            if op == "add":
                b = [-v for v in b]
        A.append(a)
        B.append(b)
    out = teuk.test_mp_op(op, n, np.array(A), np.array(B), on_device=False)
    worst = 0.0
    for a, b, o in zip(A, B, out):
        fa, fb = frac(a), frac(b)
        exact = {"add": fa + fb, "sub": fa - fb, "mul": fa * fb, "div": fa / fb}[op]
        scale = max(abs(fa), abs(fb)) if op in ("add", "sub") else abs(exact)     # "sloppy" add contract
        err = abs(frac(o) - exact) / scale
        worst = max(worst, float(err))
        assert err <= (4 if op != "div" else 16) * EPS[n], (a, b, list(o), float(err))
        # limbs non-overlapping and ordered
        for k in range(n - 1):
            assert o[k + 1] == 0.0 or abs(o[k + 1]) <= math.ulp(o[k]) * 1.0000001 or o[k] == 0.0, list(o)
    print(op, n, "worst err / eps:", worst / EPS[n])


@pytest.mark.parametrize("n", [2, 4])
def test_sqrt(n):
    rng = random.Random(9)
    with mp.workprec(1200):
        for _ in range(60):
            a = rand_mp(rng, n, rng.randint(-30, 30))
            a[0] = abs(a[0])
            out = op1("sqrt", n, a, [0.0])
            exact = mp.sqrt(sum(mp.mpf(v) for v in a))
            got = sum(mp.mpf(v) for v in out)
            assert abs((got - exact) / exact) <= 32 * EPS[n]


def test_elementary_functions_against_mpmath():
    def val(l):
        return sum(mp.mpf(v) for v in l)
    with mp.workdps(90):
        assert abs(val(teuk.test_mp_fn("pi")) - mp.pi) / mp.pi < mp.mpf(10) ** -62
        assert abs(val(teuk.test_mp_fn("ln2")) - mp.log(2)) / mp.log(2) < mp.mpf(10) ** -62
        rng = random.Random(4)
        for _ in range(30):
            x = rng.uniform(-300, 300)
            got = val(teuk.test_mp_fn("exp", [x, rng.uniform(-1, 1) * 1e-18 * abs(x)]))
        for x in (-233.7, -40.25, -1.0, 0.0, 1e-9, 0.7, 3.3, 120.0, 350.5):
            lo = x * 1.1e-17
            ref = mp.exp(mp.mpf(x) + mp.mpf(lo))
            got = val(teuk.test_mp_fn("exp", [x, lo]))
            assert abs(got - ref) / ref < mp.mpf(10) ** -60, x
        for x in (1e-101, 3.3e-40, 0.5, 1.0, 1.0000001, 7.0, 1e6):
            ref = mp.log(mp.mpf(x))
            got = val(teuk.test_mp_fn("log", [x]))
            assert abs(got - ref) <= mp.mpf(10) ** -60 * max(1, abs(ref)), x
        for x in (0.0245, 0.5, 1.0, 1.5462526341887264):
            assert abs(val(teuk.test_mp_fn("sin", [x])) - mp.sin(mp.mpf(x))) < mp.mpf(10) ** -62
            assert abs(val(teuk.test_mp_fn("cos", [x])) - mp.cos(mp.mpf(x))) < mp.mpf(10) ** -62
