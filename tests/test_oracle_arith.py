"""Pin P1: the oracle's double-double / quad-double arithmetic (oracle/mpx.hpp; PAPER.md:134 —
datatypes "based on the appropriate number of double-precision floats") against exact rationals
(fractions.Fraction) and mpmath at 1200 bits, plus structural invariants."""
import math
import random
from fractions import Fraction

import mpmath as mp
import pytest

from oracle import oracle

EPS = {2: 2.0 ** -104, 4: 2.0 ** -208}


def frac(limbs):
    return sum((Fraction(float(v)) for v in limbs), Fraction(0))


def rand_mp(rng, n, scale_exp=0):
    """random normalised n-limb number with all limbs populated"""
    limbs = []
    e = scale_exp
    for k in range(n):
        v = math.ldexp(rng.uniform(0.5, 1.0) * rng.choice((-1, 1)), e)
        limbs.append(v)
        e -= 54 + rng.randint(0, 3)
    # renormalise through the oracle itself would be circular: build from an exact rational instead
    total = frac(limbs)
    out = []
    for _ in range(n):
        hi = float(total)           # Fraction -> nearest double (correctly rounded)
        out.append(hi)
        total -= Fraction(hi)
    return out


def is_normalised(limbs):
    for k in range(len(limbs) - 1):
        hi, lo = limbs[k], limbs[k + 1]
        if hi == 0.0:
            if lo != 0.0:
                return False
            continue
        if abs(lo) > 0.5 * math.ulp(hi) * (1 + 1e-9):
            return False
    return True


def rel_err(limbs, exact: Fraction):
    if exact == 0:
        return abs(frac(limbs))
    return abs((frac(limbs) - exact) / exact)


@pytest.mark.parametrize("n", [2, 4])
def test_exact_cases(n):
    # (1 + 2^-60) + (1 - 2^-60) = 2 exactly
    a, b = [1.0, 2.0 ** -60], [1.0, -(2.0 ** -60)]
    assert frac(oracle.mp_op("add", n, a, b)) == 2
    # (2^30 + 1)(2^30 - 1) = 2^60 - 1 needs 61 bits: exact in >= 2 limbs
    assert frac(oracle.mp_op("mul", n, [2.0 ** 30 + 1], [2.0 ** 30 - 1])) == 2 ** 60 - 1
    # scaled copies
    sc = 2.0 ** -900
    assert frac(oracle.mp_op("mul", n, [(2.0 ** 30 + 1) * sc], [2.0 ** 30 - 1])) == Fraction(2 ** 60 - 1) * Fraction(sc)
    # x - x = 0, x + 0 = x, negation limb-wise
    rng = random.Random(5)
    x = rand_mp(rng, n)
    assert oracle.mp_op("sub", n, x, x) == [0.0] * n
    assert oracle.mp_op("add", n, x, [0.0]) == x
    # x * 2^k exact
    assert frac(oracle.mp_op("mul_d", n, x, [2.0 ** 17])) == frac(x) * 2 ** 17
    assert frac(oracle.mp_op("mul", n, x, [0.5])) == frac(x) / 2
    # small rationals p/q * q = p to working precision and p/q reconstructed
    for p, q in [(1, 3), (22, 7), (-5, 11), (1, 1 << 20)]:
        quo = oracle.mp_op("div", n, [float(p)], [float(q)])
        assert rel_err(quo, Fraction(p, q)) <= 4 * EPS[n]
        assert is_normalised(quo)


@pytest.mark.parametrize("n", [2, 4])
@pytest.mark.parametrize("op", ["add", "sub", "mul", "div"])
def test_random_against_exact_rationals(n, op):
    rng = random.Random(100 * n + len(op))
    worst = 0.0
    for trial in range(300):
        a = rand_mp(rng, n, rng.randint(-40, 40))
        b = rand_mp(rng, n, rng.randint(-40, 40))
        if trial % 3 == 0 and op in ("add", "sub"):
            # massive cancellation: b = +-a perturbed in a low limb
            b = list(a)
            b[n - 1] = b[n - 1] * (1 + rng.uniform(-0.5, 0.5))
            if op == "add":
                b = [-v for v in b]
        out = oracle.mp_op(op, n, a, b)
        fa, fb = frac(a), frac(b)
        exact = {"add": fa + fb, "sub": fa - fb, "mul": fa * fb, "div": fa / fb}[op]
        err = rel_err(out, exact)
        worst = max(worst, float(err))
        assert err <= 4 * EPS[n], (a, b, out)
        assert is_normalised(out), out
        if op in ("add", "mul"):                      # commutativity, bitwise
            assert oracle.mp_op(op, n, b, a) == out
    print(op, n, "worst rel err / eps^N:", worst / EPS[n])


@pytest.mark.parametrize("n", [2, 4])
def test_add_is_exact_when_representable(n):
    """sum of two numbers whose exact sum fits in n limbs must come back exact"""
    rng = random.Random(77)
    for _ in range(200):
        bits = 53 * n - 8
        x = rng.getrandbits(bits // 2) * (1 << (bits // 2))
        y = rng.getrandbits(bits // 2)
        a = rand_limbs_from_int(x, n)
        b = rand_limbs_from_int(y, n)
        assert frac(oracle.mp_op("add", n, a, b)) == x + y


def rand_limbs_from_int(v, n):
    total = Fraction(v)
    out = []
    for _ in range(n):
        hi = float(total)
        out.append(hi)
        total -= Fraction(hi)
    assert total == 0
    return out


@pytest.mark.parametrize("n", [2, 4])
def test_sqrt_against_mpmath(n):
    rng = random.Random(9)
    with mp.workprec(1200):
        for _ in range(100):
            a = rand_mp(rng, n, rng.randint(-30, 30))
            a = [abs(a[0])] + a[1:]
            out = oracle.mp_op("sqrt", n, a)
            exact = mp.sqrt(sum(mp.mpf(v) for v in a))
            got = sum(mp.mpf(v) for v in out)
            assert abs((got - exact) / exact) <= 8 * EPS[n]
            assert is_normalised(out)
    assert oracle.mp_op("sqrt", n, [0.0]) == [0.0] * n
    assert frac(oracle.mp_op("sqrt", n, [4.0])) == 2


def test_dd_and_qd_agree_with_fp64_on_doubles():
    """a plain double embeds exactly; first limb of a op b is the IEEE result"""
    rng = random.Random(3)
    for _ in range(200):
        x, y = rng.uniform(-10, 10), rng.uniform(-10, 10)
        for n in (2, 4):
            assert oracle.mp_op("add", n, [x], [y])[0] == x + y
            assert oracle.mp_op("mul", n, [x], [y])[0] == x * y
            assert frac(oracle.mp_op("mul", n, [x], [y])) == Fraction(x) * Fraction(y)   # 106 bits fit in 2 limbs
