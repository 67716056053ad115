"""ORACLE (test infrastructure, not product code) — Python front end.

Builds `liboracle.so` from oracle/teuk_oracle.cpp (g++ -O2 -ffp-contract=off -fopenmp), computes
the 1-D tables r(r*), r - r_+, sin/cos(theta_j) with mpmath (oracle/mp_ref.py) and drives the
plain C++ stepper through ctypes.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module; it imports nothing from the
CUDA package except the seeded input recipe's dataclass (which holds no method arithmetic).

Array conventions (same as include/teuk.h): state planes [4][L][N_theta][N_win] fp64, i fastest;
fields Phi_R, Phi_I, Pi_R, Pi_I (Eq. 9); observer series [count][4][L].
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

from . import mp_ref

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = [os.path.join(_HERE, "teuk_oracle.cpp"), os.path.join(_HERE, "mpx.hpp"), os.path.join(_HERE, "mpf.hpp")]
CXXFLAGS = ["-O2", "-std=c++17", "-mfma", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared"]
_lib = None


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(p) for p in _SRC)
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < newest:
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.check_call(["g++", *CXXFLAGS, _SRC[0], "-o", tmp])
        os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        _lib.oracle_create.argtypes = [C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double,
                                       C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, dp, dp, dp, dp, dp, dp,
                                       C.c_int, dp, dp, C.c_int, C.POINTER(C.c_void_p)]
        _lib.oracle_set_observer.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_long]
        _lib.oracle_set_initial.argtypes = [C.c_void_p, dp, C.c_int]
        _lib.oracle_step.argtypes = [C.c_void_p, C.c_long]
        _lib.oracle_read.argtypes = [C.c_void_p, dp]
        _lib.oracle_observe.argtypes = [C.c_void_p, dp, C.c_long, C.POINTER(C.c_long)]
        _lib.oracle_get_tables.argtypes = [C.c_void_p, C.c_int, dp]
        _lib.oracle_set_tables.argtypes = [C.c_void_p, C.c_int, dp]
        _lib.oracle_get_cot.argtypes = [C.c_void_p, dp]
        _lib.oracle_lambda.argtypes = [C.c_void_p, dp, dp]
        _lib.oracle_set_multipole.argtypes = [C.c_void_p, C.c_double, C.c_int, dp, C.c_long]
        _lib.oracle_observe_multipoles.argtypes = [C.c_void_p, dp, C.c_long, C.POINTER(C.c_long)]
        _lib.oracle_destroy.argtypes = [C.c_void_p]
        _lib.oracle_destroy.restype = None
        _lib.oracle_mp_op.argtypes = [C.c_int, C.c_int, dp, dp, dp]
        _lib.oracle_mpf_op.argtypes = [C.c_int, C.c_int, dp, dp, dp]
        _lib.oracle_mp_op_batch.argtypes = [C.c_int, C.c_int, C.c_int, C.c_long, dp, dp, dp]
        _lib.oracle_set_zero_fast_path.argtypes = [C.c_int]
        _lib.oracle_set_threads.argtypes = [C.c_int]
    return _lib


def _dp(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


_OPS = {"add": 0, "sub": 1, "mul": 2, "div": 3, "sqrt": 4, "mul_d": 5, "half": 6}
TIERS = {"exact": 0, "fast": 1}


def mp_op(op: str, n: int, a, b=None, tier: str = "exact") -> list:
    """Test hook (pin P1): one N-limb operation of the oracle's arithmetic (tier "exact": mpx.hpp, "fast": mpf.hpp)."""
    aa = np.array(list(a) + [0.0] * (4 - len(a)), dtype=np.float64)
    bb = np.array(list(b if b is not None else [1.0]) + [0.0] * 4, dtype=np.float64)[:4].copy()
    out = np.zeros(4)
    fn = lib().oracle_mpf_op if TIERS[tier] else lib().oracle_mp_op
    rc = fn(_OPS[op], n, _dp(aa), _dp(bb), _dp(out))
    assert rc == 0
    return [float(v) for v in out[:n]]


def mp_op_batch(op: str, n: int, a: np.ndarray, b: np.ndarray, tier: str = "exact") -> np.ndarray:
    """The same hook on a corpus: a, b [count][n] -> [count][n]."""
    a = np.ascontiguousarray(a, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    assert a.shape == b.shape and a.shape[1] == n
    out = np.zeros_like(a)
    rc = lib().oracle_mp_op_batch(TIERS[tier], _OPS[op], n, a.shape[0], _dp(a), _dp(b), _dp(out))
    assert rc == 0
    return out


def set_zero_fast_path(on: bool) -> bool:
    """Test hook: switch the x + 0 = x / x * 0 = 0 shortcuts of the fast tier (mpf.hpp); returns the old setting."""
    return bool(lib().oracle_set_zero_fast_path(int(on)))


def set_threads(n: int) -> int:
    return lib().oracle_set_threads(n)


_table_cache: dict = {}


class Oracle:
    """Plain CPU solver of PAPER.md §III.B; see teuk_oracle.cpp for the step-by-step citations."""

    def __init__(self, M, a, s, m, n_r, n_theta, rstar_min, rstar_max, dt, precision, i_lo=0, n_win=None,
                 theta_order=2, tier="exact"):
        self.n_win = n_r - i_lo if n_win is None else n_win
        self.n_r, self.n_theta, self.L, self.i_lo = n_r, n_theta, precision, i_lo
        self.s, self.m = s, m
        key = (float(M), float(a), float(rstar_min), float(rstar_max), n_r, i_lo, self.n_win)
        if key not in _table_cache:
            _table_cache[key] = mp_ref.radial_tables(M, a, rstar_min, rstar_max, n_r, i_lo, self.n_win)
        r_l, d_l, dr_l = _table_cache[key]
        sn, cs, dth_l = mp_ref.theta_tables(n_theta)
        wc, wd = mp_ref.fd_weight_limbs(theta_order)
        self._keep = [np.ascontiguousarray(np.array(x, dtype=np.float64)) for x in (r_l, d_l, sn, cs, dr_l, dth_l, wc, wd)]
        self.h = C.c_void_p()
        k = [_dp(x) for x in self._keep]
        rc = lib().oracle_create(M, a, s, m, n_r, n_theta, rstar_min, rstar_max, dt, precision, i_lo, self.n_win,
                                 *k[:6], theta_order, k[6], k[7], TIERS[tier], C.byref(self.h))
        if rc != 0:
            self.h = None
            raise ValueError(f"oracle_create failed: {rc}")

    @classmethod
    def from_workload(cls, w, precision=None, i_lo=0, n_win=None, theta_order=2, tier="exact"):
        return cls(w.M, w.a, w.s, w.m, w.n_r, w.n_theta, w.rstar_min, w.rstar_max, w.dt,
                   precision or w.precision, i_lo, n_win, theta_order, tier)

    def __del__(self):
        if getattr(self, "h", None):
            lib().oracle_destroy(self.h)
            self.h = None

    def _chk(self, rc):
        if rc != 0:
            raise RuntimeError(f"oracle error {rc}")

    def set_observer(self, rstar_obs, theta_obs, capacity):
        self._chk(lib().oracle_set_observer(self.h, rstar_obs, theta_obs, capacity))

    def set_multipole_observer(self, rstar_obs, n_ell, capacity):
        """NEXT-2: per step, project Phi(r*_obs, theta) on _sY_l'm, l' = l_min .. l_min + n_ell - 1 (reading A24)."""
        q = np.ascontiguousarray(np.array(mp_ref.multipole_weights(self.s, self.m, self.n_theta, n_ell), dtype=np.float64))
        self._mpq, self.n_ell = q, n_ell
        self._chk(lib().oracle_set_multipole(self.h, rstar_obs, n_ell, _dp(q), capacity))

    def observe_multipoles(self, max_samples: int) -> np.ndarray:
        """[count][n_ell][2][L]: real and imaginary part of a_l' after each completed step"""
        out = np.zeros((max(max_samples, 1), self.n_ell, 2, self.L))
        cnt = C.c_long(0)
        self._chk(lib().oracle_observe_multipoles(self.h, _dp(out), max_samples, C.byref(cnt)))
        return out[:cnt.value]

    def set_initial(self, planes: np.ndarray):
        """planes: [4][N_theta][N_win] (fp64, low limbs := 0) or [4][L][N_theta][N_win]."""
        p = np.ascontiguousarray(planes, dtype=np.float64)
        limbs_in = 1 if p.ndim == 3 else p.shape[1]
        assert p.shape[0] == 4 and p.shape[-2:] == (self.n_theta, self.n_win)
        self._chk(lib().oracle_set_initial(self.h, _dp(p), limbs_in))

    def step(self, n: int):
        self._chk(lib().oracle_step(self.h, n))

    def read(self) -> np.ndarray:
        out = np.zeros((4, self.L, self.n_theta, self.n_win))
        self._chk(lib().oracle_read(self.h, _dp(out)))
        return out

    def observe(self, max_samples: int) -> np.ndarray:
        out = np.zeros((max(max_samples, 1), 4, self.L))
        cnt = C.c_long(0)
        self._chk(lib().oracle_observe(self.h, _dp(out), max_samples, C.byref(cnt)))
        return out[:cnt.value]

    def tables(self, half: bool) -> np.ndarray:
        """[8][L][N_theta][rows]: b, alpha_R, alpha_I, gamma_R, gamma_I, W_R, W_I, kappa."""
        rows = self.n_win - 1 if half else self.n_win
        out = np.zeros((8, self.L, self.n_theta, rows))
        self._chk(lib().oracle_get_tables(self.h, int(half), _dp(out)))
        return out

    def set_tables(self, half: bool, planes: np.ndarray):
        p = np.ascontiguousarray(planes, dtype=np.float64)
        self._chk(lib().oracle_set_tables(self.h, int(half), _dp(p)))

    def cot(self) -> np.ndarray:
        out = np.zeros((self.L, self.n_theta))
        self._chk(lib().oracle_get_cot(self.h, _dp(out)))
        return out

    def apply_lambda(self, f: np.ndarray) -> np.ndarray:
        """Discrete angular operator Lambda_j[f] on one theta column, [L][N_theta]."""
        p = np.ascontiguousarray(f, dtype=np.float64).reshape(self.L, self.n_theta)
        out = np.zeros_like(p)
        self._chk(lib().oracle_lambda(self.h, _dp(p), _dp(out)))
        return out


def rel_linf(x_limbs: np.ndarray, ref_limbs: np.ndarray) -> dict:
    """DESIGN.md reading A17: per complex field F in {Phi, Pi}: max|F - F_ref| / max|F_ref|, differences
    formed limb-wise in extended precision.  Inputs [4][L][...]; returns {'Phi': e, 'Pi': e}."""
    import mpmath as mp
    out = {}
    with mp.workdps(90):
        for name, (re, im) in {"Phi": (0, 1), "Pi": (2, 3)}.items():
            dre = _limb_diff(x_limbs[re], ref_limbs[re])
            dim = _limb_diff(x_limbs[im], ref_limbs[im])
            ref_abs = np.hypot(ref_limbs[re][0], ref_limbs[im][0])
            den = float(ref_abs.max())
            # locate the worst point with doubles, then evaluate it exactly
            mag = np.hypot(dre[0], dim[0])
            k = int(np.argmax(mag))
            num = mp.sqrt(_mp_at(dre[1], k) ** 2 + _mp_at(dim[1], k) ** 2)
            out[name] = float(num / den) if den > 0 else float(num)
    return out


def _limb_diff(x, ref):
    """x, ref: [L][...]; returns (correctly rounded leading double of sum_k x_k - sum_k ref_k at
    every point, (x, ref) flattened).  The 2L terms are distilled with error-free TwoSum passes
    (bubble-sort order), so the leading value is exact to one rounding even when the leading
    limbs differ by an ulp and the low limbs compensate."""
    L = x.shape[0]
    xf, rf = x.reshape(L, -1), ref.reshape(L, -1)
    terms = [xf[k].copy() for k in reversed(range(L))] + [-rf[k] for k in reversed(range(L))]
    n = len(terms)
    for _ in range(n - 1):
        for i in range(n - 1):
            a, b = terms[i], terms[i + 1]
            s = a + b
            bb = s - a
            e = (a - (s - bb)) + (b - bb)
            terms[i], terms[i + 1] = e, s
    return terms[-1], (xf, rf)


def _mp_at(pair, k):
    import mpmath as mp
    x, ref = pair
    tot = mp.mpf(0)
    for l in range(x.shape[0]):
        tot += mp.mpf(float(x[l, k])) - mp.mpf(float(ref[l, k]))
    return tot
