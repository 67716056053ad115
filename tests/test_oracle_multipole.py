"""NEXT-2 pins (oracle): spin-weighted harmonics and the multipole-projection observer (Fig. 1, PAPER.md:130-132:
tails of the multipoles l' = 0..8; reading A24 defines the projection)."""
import math

import mpmath as mp
import numpy as np
import pytest

from oracle import mp_ref, oracle
from paper_1006_0663_b200 import inputs


def test_swsh_closed_forms_orthonormality_and_eigen_equation():
    with mp.workdps(40):
        th = mp.mpf("0.83")
        assert abs(mp_ref.swsh(-2, 2, 2, th) - mp.sqrt(5 / (64 * mp.pi)) * (1 + mp.cos(th)) ** 2) < 1e-35
        assert abs(mp_ref.swsh(-2, 2, -2, th) - mp.sqrt(5 / (64 * mp.pi)) * (1 - mp.cos(th)) ** 2) < 1e-35
        for l in range(0, 6):
            assert abs(mp_ref.swsh(0, l, 0, th) - mp.sqrt((2 * l + 1) / (4 * mp.pi)) * mp.legendre(l, mp.cos(th))) < 1e-35
        for (s, m, l1, l2) in [(0, 0, 2, 2), (0, 0, 2, 4), (-2, 2, 2, 2), (-2, 2, 2, 3), (-2, 2, 7, 7), (-1, 1, 3, 3), (-2, 0, 4, 6)]:
            v = 2 * mp.pi * mp.quad(lambda t: mp_ref.swsh(s, l1, m, t) * mp_ref.swsh(s, l2, m, t) * mp.sin(t), [0, mp.pi])
            assert abs(v - (1 if l1 == l2 else 0)) < 1e-25
        # (1/sin)(sin Y')' - (m + s cos)^2/sin^2 Y + s Y = -(l - s)(l + s + 1) Y   (the angular part of Eq. (1))
        for (s, l, m) in [(0, 3, 0), (-2, 4, 2), (-1, 2, 1)]:
            Y = lambda t: mp_ref.swsh(s, l, m, t)
            t0 = mp.mpf("1.1")
            lhs = (mp.diff(Y, t0, 2) + mp.cos(t0) / mp.sin(t0) * mp.diff(Y, t0)
                   - (m + s * mp.cos(t0)) ** 2 / mp.sin(t0) ** 2 * Y(t0) + s * Y(t0))
            assert abs(lhs + (l - s) * (l + s + 1) * Y(t0)) < 1e-20


def test_fejer_weights_and_discrete_orthonormality():
    """Fejer-1 weights integrate polynomials of degree < N in cos(theta) exactly, so the projection weights are
    discretely orthonormal to rounding whenever l + l' (+ the spin-weight factors) stays below N"""
    with mp.workdps(40):
        for n in (8, 16, 33):
            wf = mp_ref.fejer_weights(n)
            th = [(j + mp.mpf(1) / 2) * mp.pi / n for j in range(n)]
            assert abs(sum(wf) - 2) < 1e-35
            for p in range(0, n):
                exact = (1 + (-1) ** p) / mp.mpf(p + 1)                      # int_-1^1 x^p dx
                assert abs(sum(w * mp.cos(t) ** p for w, t in zip(wf, th)) - exact) < 1e-30, (n, p)
            # degree n is NOT integrated exactly: the rule has the advertised degree and no more
            p = n if n % 2 == 0 else n + 1
            assert abs(sum(w * mp.cos(t) ** p for w, t in zip(wf, th)) - 2 / mp.mpf(p + 1)) > 1e-20
    for (s_, m_, n) in ((0, 0, 32), (-2, 2, 32)):
        q = np.array(mp_ref.multipole_weights(s_, m_, n, 9))[:, :, 0]
        th = (np.arange(n) + 0.5) * math.pi / n
        lmin = max(abs(s_), abs(m_))
        with mp.workdps(30):
            Y = np.array([[float(mp_ref.swsh(s_, lmin + k, m_, t)) for t in th] for k in range(9)])
        assert np.abs(q @ Y.T - np.eye(9)).max() < 1e-13


@pytest.mark.parametrize("precision", [1, 2])
def test_projection_recovers_the_multipole_content(precision):
    """state = g(r*) (c0 Y_0 + c2 Y_2 + c3 Y_3): the observer returns c_l g(r*_obs) up to the quadrature error, at the
    first sample (one step changes the field by O(dt))"""
    n_r, n_t = 64, 96
    w = inputs.config(1).scaled(n_r=n_r, n_theta=n_t, rstar_min=0.0, rstar_max=63.0, dt_override=1e-6)
    th = (np.arange(n_t) + 0.5) * math.pi / n_t
    rs = np.arange(n_r) * 1.0
    g = np.exp(-((rs - 30.0) ** 2) / 50.0)
    with mp.workdps(30):
        Y = {l: np.array([float(mp_ref.swsh(0, l, 0, t)) for t in th]) for l in (0, 2, 3)}
    c = {0: 0.7, 2: -1.3, 3: 0.4}
    u0 = np.zeros((4, n_t, n_r))
    u0[0] = sum(c[l] * Y[l] for l in c)[:, None] * g[None, :]
    u0[1] = 0.5 * u0[0]
    o = oracle.Oracle.from_workload(w, precision=precision)
    o.set_multipole_observer(30.25, 5, 4)
    o.set_initial(u0)
    o.step(1)
    a = o.observe_multipoles(4)[0, :, :, 0]
    g_obs = 0.75 * g[30] + 0.25 * g[31]
    for l in range(5):
        assert abs(a[l, 0] - c.get(l, 0.0) * g_obs) < 1e-5          # only the O(dt) change of one tiny step remains
        assert abs(a[l, 1] - 0.5 * c.get(l, 0.0) * g_obs) < 1e-5


def test_kerr_mixes_multipoles_schwarzschild_does_not():
    """a = 0: spherical symmetry keeps pure-l data pure; a = 0.9: l' = l +- 2 are excited (the mode
    coupling behind the l + l' + 3 tail rule of Fig. 1)"""
    res = {}
    for a in (0.0, 0.9):
        w = inputs.config(4).scaled(a=a, n_r=241, n_theta=64, rstar_min=-20.0, rstar_max=40.0, precision=1,
                                    centre=(6.0, 0.0), width=(3.0, 0.0))
        o = oracle.Oracle.from_workload(w)
        o.set_multipole_observer(4.0, 5, 400)
        o.set_initial(inputs.initial_state(w))          # pure l = 0 data
        o.step(400)
        s_ = o.observe_multipoles(400)[:, :, :, 0]
        amp = np.abs(s_[..., 0] + 1j * s_[..., 1]).max(axis=0)
        res[a] = amp / amp[0]
    assert res[0.0][2] < 1e-12 and res[0.9][2] > 1e-3       # a = 0: constant-in-theta data stay exactly l' = 0
    assert res[0.0][1] < 1e-12 and res[0.9][1] < 1e-10 and res[0.0][4] < 1e-12             # odd l' never couple to even data (reflection symmetry)
