"""Pin P2 (numeric) + Eq. (2) pins: the C++ oracle's coefficient tables (teuk_oracle.cpp O3,
quad-double) against oracle/mp_ref.py::coefficients evaluated by mpmath at 100 digits — the same
formulas that tests/test_coefficients_symbolic.py ties to Eq. (1) — including the innermost rows
where r - r_+ is 1e-11 .. 1e-101 (reading A3); and the r(r*) inversion against the
differential form of Eq. (2), and its Schwarzschild closed form."""
import mpmath as mp
import numpy as np
import pytest

from oracle import mp_ref, oracle
from paper_1006_0663_b200 import inputs

TOL = {1: 2.0 ** -52, 2: 2.0 ** -103, 4: 2.0 ** -200}


def _check_window(w, precision, i_lo, n_win):
    o = oracle.Oracle.from_workload(w, precision=precision, i_lo=i_lo, n_win=n_win)
    ti, th = o.tables(False), o.tables(True)
    cot = o.cot()
    worst = 0.0
    with mp.workdps(100):
        rp, rm = mp_ref.horizons(w.M, w.a)
        lo = mp.mpf(w.rstar_min)
        dr = (mp.mpf(w.rstar_max) - lo) / (w.n_r - 1)
        dth = mp.pi / w.n_theta
        for half, tab in ((False, ti), (True, th)):
            rows = tab.shape[-1]
            for i in sorted({0, 1, rows // 2, rows - 1}):
                rs = lo + (i_lo + i + (mp.mpf(1) / 2 if half else 0)) * dr
                r, d = mp_ref.r_of_rstar(rs, w.M, w.a)
                for j in sorted({0, 1, w.n_theta // 2, w.n_theta - 1}):
                    t = (j + mp.mpf(1) / 2) * dth
                    c = mp_ref.coefficients(r, d, mp.sin(t), mp.cos(t), mp.mpf(w.M), mp.mpf(w.a), w.s, w.m, rp - rm)
                    ref = [c["b"], c["alpha"][0], c["alpha"][1], c["gamma"][0], c["gamma"][1],
                           c["W"][0], c["W"][1], c["kappa"]]
                    scale = max(abs(v) for v in ref)
                    for q in range(8):
                        got = mp_ref.from_limbs(tab[q, :, j, i])
                        # relative to the coefficient itself, or (gamma and W are sums of terms that
                        # partly cancel) to the largest coefficient at the point
                        err = abs(got - ref[q]) / max(abs(ref[q]), scale / 64)
                        worst = max(worst, float(err))
                        assert err <= 16 * TOL[precision], (half, i, j, q, float(err))
        for j in range(w.n_theta):
            t = (j + mp.mpf(1) / 2) * dth
            ref = mp.cos(t) / mp.sin(t)
            assert abs(mp_ref.from_limbs(cot[:, j]) - ref) <= 4 * TOL[precision] * max(abs(ref), 1)
    return worst


@pytest.mark.parametrize("cfg,precision", [(1, 1), (2, 1), (2, 2), (4, 4), (2, 4)])
def test_tables_match_mpmath_including_horizon_rows(cfg, precision):
    w = inputs.config(cfg)
    for i_lo in (0, w.n_r // 3, w.n_r - 6):
        worst = _check_window(w, precision, i_lo, 6)
        print(cfg, precision, i_lo, "worst rel err", worst)


def test_sweep_parameters_tables():
    w = inputs.sweep_cell(4096, 32, 2)
    _check_window(w, 2, 0, 5)
    _check_window(w, 2, 2000, 5)


def test_horizon_distance_magnitudes():
    """DESIGN.md reading A3: r - r_+ at the inner edge of each config (why Delta is built from delta)."""
    with mp.workdps(130):
        expect = {1: 1.0e-11, 2: 2.6e-40, 4: 1.4e-101}
        for k, val in expect.items():
            w = inputs.config(k)
            _, d = mp_ref.r_of_rstar(w.rstar_min, w.M, w.a)
            assert 0.3 < float(d / val) < 3.0, (k, mp.nstr(d, 5))


def test_rstar_inversion_satisfies_eq2():
    """dr*/dr = (r^2 + a^2)/Delta (Eq. 2) checked by central differences of the inverse map, and the
    Schwarzschild closed form r* = r + 2M ln(r/2M - 1)."""
    with mp.workdps(60):
        for a in (0.0, 0.5, 0.9, 0.99):
            for rs in (-40, -3.5, 0.0, 7.25, 300):
                eps = mp.mpf(10) ** -20
                r1, _ = mp_ref.r_of_rstar(rs - eps, 1.0, a)
                r2, _ = mp_ref.r_of_rstar(rs + eps, 1.0, a)
                r0, d0 = mp_ref.r_of_rstar(rs, 1.0, a)
                drdrs = (r2 - r1) / (2 * eps)
                Delta = r0 * r0 - 2 * r0 + mp.mpf(a) ** 2
                assert abs(drdrs - Delta / (r0 * r0 + mp.mpf(a) ** 2)) < mp.mpf(10) ** -30
                rp, _ = mp_ref.horizons(1.0, a)
                assert abs((r0 - rp) - d0) < mp.mpf(10) ** -50
        for rs in (-30, 1.0, 55.5):
            r, _ = mp_ref.r_of_rstar(rs, 1.0, 0.0)
            assert abs(r + 2 * mp.log(r / 2 - 1) - rs) < mp.mpf(10) ** -45


def test_theta_tables_exactly_mirrored():
    for n in (6, 16, 33):
        sn, cs, _ = mp_ref.theta_tables(n)
        for j in range(n):
            assert sn[j] == sn[n - 1 - j]
            assert cs[j] == [-v for v in cs[n - 1 - j]]


def test_limb_roundtrip():
    with mp.workdps(100):
        x = mp.pi * mp.mpf(10) ** -37
        assert abs(mp_ref.from_limbs(mp_ref.to_limbs(x)) - x) / x < mp.mpf(2) ** -205
