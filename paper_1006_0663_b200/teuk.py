"""Thin ctypes binding over libteuk.so (include/teuk.h): same names, argument marshalling only.

PyTorch is used for device memory (the workspace tensor) and the CUDA stream; every step of the path
runs in the library's kernels.  Importing this module fails loudly if the library is missing — there
is no CPU fallback."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libteuk.so")
if not os.path.exists(_SO):
    raise ImportError(f"{_SO} not found: build it with `python -m paper_1006_0663_b200.build` "
                      "(or __graft_entry__.build()); the CUDA path has no fallback")
lib = C.CDLL(_SO)

FP64, DD, QD = 1, 2, 4
OK, EINVAL, ENOMEM, ECUDA, ESTATE, ENONFINITE, ECAPACITY = 0, -1, -2, -3, -4, -5, -6
STATIC_SCRATCH_DOUBLES = 512 * 1024

_dp = C.POINTER(C.c_double)
_lp = C.POINTER(C.c_long)
_h = C.c_void_p
SIGNATURES = {
    "teuk_workspace_bytes": (C.c_int, [C.c_int, C.c_int, C.c_int, C.c_int, C.c_long, C.POINTER(C.c_size_t)]),
    "teuk_create": (C.c_int, [C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                              C.c_double, C.c_int, C.c_int, C.c_void_p, C.c_size_t, C.c_long, C.c_void_p, C.POINTER(_h)]),
    "teuk_create_slab": (C.c_int, [C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                   C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_size_t, C.c_long,
                                   C.c_void_p, C.POINTER(_h)]),
    "teuk_set_option": (C.c_int, [_h, C.c_char_p, C.c_double]),
    "teuk_set_observer": (C.c_int, [_h, C.c_double, C.c_double, C.c_long]),
    "teuk_set_initial": (C.c_int, [_h, _dp, C.c_int]),
    "teuk_set_initial_device": (C.c_int, [_h, C.c_void_p, C.c_int]),
    "teuk_step": (C.c_int, [_h, C.c_long]),
    "teuk_read": (C.c_int, [_h, _dp]),
    "teuk_read_device": (C.c_int, [_h, C.c_void_p]),
    "teuk_read_columns_device": (C.c_int, [_h, C.c_int, C.c_int, C.c_void_p]),
    "teuk_write_columns_device": (C.c_int, [_h, C.c_int, C.c_int, C.c_void_p]),
    "teuk_observe": (C.c_int, [_h, _dp, C.c_long, _lp]),
    "teuk_set_multipole_observer": (C.c_int, [_h, C.c_double, C.c_int, C.c_long]),
    "teuk_observe_multipoles": (C.c_int, [_h, _dp, C.c_long, _lp]),
    "teuk_steps_done": (C.c_int, [_h, _lp]),
    "teuk_launch_count": (C.c_int, [_h, _lp]),
    "teuk_step_geometry": (C.c_int, [_h, _lp]),
    "teuk_destroy": (None, [_h]),
    "teuk_strerror": (C.c_char_p, [C.c_int]),
    "teuk_get_tables": (C.c_int, [_h, C.c_int, _dp]),
    "teuk_get_folded": (C.c_int, [_h, C.c_int, C.c_int, _dp]),
    "teuk_get_folded_static": (C.c_int, [_h, C.c_int, C.c_int, _dp]),
    "teuk_get_radial": (C.c_int, [_h, _dp, _dp]),
    "teuk_test_mp_op": (C.c_int, [C.c_int, C.c_int, _dp, _dp, _dp, C.c_long, C.c_int]),
    "teuk_test_mp_fn": (C.c_int, [C.c_int, _dp, _dp]),
    "teuk_bench_fp64": (C.c_int, [C.c_int, C.c_long, _dp, C.c_void_p]),
}
for _name, (_res, _args) in SIGNATURES.items():
    _f = getattr(lib, _name)
    _f.restype = _res
    _f.argtypes = _args


class TeukError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {lib.teuk_strerror(code).decode()} ({code})")


def _chk(rc: int, where: str, allow=()):
    if rc != OK and rc not in allow:
        raise TeukError(rc, where)
    return rc


def _np(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def workspace_bytes(n_r: int, n_theta: int, precision: int, obs_capacity: int, coef_variant: int = -1) -> int:
    """coef_variant: -1 = all coefficient supplies resident (default), 0 = stored planes only, 1 / 2 = recompute tables only"""
    out = C.c_size_t(0)
    _chk(lib.teuk_workspace_bytes(n_r, n_theta, precision, coef_variant, obs_capacity, C.byref(out)), "teuk_workspace_bytes")
    return out.value


class Teuk:
    """One solver handle (teuk_ctx).  Methods are 1:1 with the C calls."""

    def __init__(self, M, a, s, m, n_r, n_theta, rstar_min, rstar_max, dt, precision, obs_capacity=0,
                 device="cuda:0", stream=None, slab=None, guard_bytes=0, coef_variant=-1):
        """slab = (i_lo, n_win): teuk_create_slab, the handle holds that column range of the n_r-node grid.
        guard_bytes > 0 (tests): the workspace is allocated with a guard band of that many bytes on each side, filled with
        the byte 0xA5; `guards_intact()` tells whether any kernel wrote outside the workspace it was given."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1006_0663_b200.teuk needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        n_r_global, i_lo = n_r, 0
        if slab is not None:
            i_lo, n_r = int(slab[0]), int(slab[1])
        self.n_r, self.n_theta, self.L, self.i_lo, self.n_r_global = n_r, n_theta, precision, i_lo, n_r_global
        nbytes = workspace_bytes(n_r, n_theta, precision, obs_capacity, coef_variant)
        self.workspace_nbytes = nbytes
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            guard = (int(guard_bytes) + 255) // 256 * 256
            self.workspace = torch.full((nbytes + 256 + 2 * guard,), 0xA5, dtype=torch.uint8, device=self.device)
            # own non-default stream unless one is given (the legacy default stream cannot be graph-captured)
            self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
            # the tensor is allocated (and filled) on the current stream but used on self.stream from here on
            self.stream.wait_stream(torch.cuda.current_stream(self.device))
            self.workspace.record_stream(self.stream)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) // 256 * 256 + guard
            self._guard = (self._ws_ptr - base - guard, guard, self._ws_ptr - base + nbytes)   # (start of band 1, length, start of band 2)
            self.h = _h()
            if slab is None:
                _chk(lib.teuk_create(M, a, s, m, n_r, n_theta, rstar_min, rstar_max, dt, precision, coef_variant,
                                     C.c_void_p(self._ws_ptr), nbytes, obs_capacity,
                                     C.c_void_p(self.stream.cuda_stream), C.byref(self.h)), "teuk_create")
            else:
                _chk(lib.teuk_create_slab(M, a, s, m, n_r_global, n_theta, rstar_min, rstar_max, dt, precision, coef_variant,
                                          i_lo, n_r,
                                          C.c_void_p(self._ws_ptr), nbytes, obs_capacity,
                                          C.c_void_p(self.stream.cuda_stream), C.byref(self.h)), "teuk_create_slab")

    @classmethod
    def from_workload(cls, w, precision=None, obs_capacity=0, **kw):
        return cls(w.M, w.a, w.s, w.m, w.n_r, w.n_theta, w.rstar_min, w.rstar_max, w.dt,
                   precision or w.precision, obs_capacity, **kw)

    def close(self):
        if getattr(self, "h", None) and lib is not None:
            lib.teuk_destroy(self.h)          # synchronises the handle's stream before the workspace can be recycled
            self.h = None

    def guards_intact(self) -> bool:
        """guard_bytes > 0 only: both guard bands around the workspace still hold their fill pattern"""
        lo, n, hi = self._guard
        self.stream.synchronize()
        w = self.workspace
        return bool((w[lo:lo + n] == 0xA5).all().item() and (w[hi:hi + n] == 0xA5).all().item()) if n else True

    __del__ = close

    def set_option(self, key: str, value: float):
        _chk(lib.teuk_set_option(self.h, key.encode(), float(value)), "teuk_set_option")

    def set_observer(self, rstar_obs, theta_obs, capacity):
        _chk(lib.teuk_set_observer(self.h, rstar_obs, theta_obs, capacity), "teuk_set_observer")

    def set_initial(self, planes):
        """numpy [4][N_theta][N_r] / [4][L][N_theta][N_r] (host) or a CUDA float64 torch tensor of that shape."""
        if isinstance(planes, np.ndarray):
            p = np.ascontiguousarray(planes, dtype=np.float64)
            limbs_in = 1 if p.ndim == 3 else p.shape[1]
            assert p.shape[0] == 4 and p.shape[-2:] == (self.n_theta, self.n_r)
            _chk(lib.teuk_set_initial(self.h, _np(p), limbs_in), "teuk_set_initial")
        else:
            t = planes.contiguous()
            assert t.is_cuda and t.dtype == self.torch.float64
            self.stream.wait_stream(self.torch.cuda.current_stream(self.device))   # t was produced there
            limbs_in = 1 if t.dim() == 3 else t.shape[1]
            assert t.shape[0] == 4 and tuple(t.shape[-2:]) == (self.n_theta, self.n_r)
            _chk(lib.teuk_set_initial_device(self.h, C.c_void_p(t.data_ptr()), limbs_in), "teuk_set_initial_device")

    def set_initial_pinned(self, pinned):
        """host tensor in pinned memory -> teuk_set_initial (H2D inside the call)."""
        limbs_in = 1 if pinned.dim() == 3 else pinned.shape[1]
        _chk(lib.teuk_set_initial(self.h, C.cast(pinned.data_ptr(), _dp), limbs_in), "teuk_set_initial")

    def step(self, n: int):
        _chk(lib.teuk_step(self.h, n), "teuk_step")

    def read(self, out: np.ndarray | None = None) -> np.ndarray:
        if out is None:
            out = np.empty((4, self.L, self.n_theta, self.n_r))
        _chk(lib.teuk_read(self.h, _np(out)), "teuk_read")
        return out

    def read_pinned(self, pinned):
        _chk(lib.teuk_read(self.h, C.cast(pinned.data_ptr(), _dp)), "teuk_read")
        return pinned

    def read_device(self, t=None):
        if t is None:
            t = self.torch.empty((4, self.L, self.n_theta, self.n_r), dtype=self.torch.float64, device=self.device)
        self.stream.wait_stream(self.torch.cuda.current_stream(self.device))     # `t` may still be in use there
        _chk(lib.teuk_read_device(self.h, C.c_void_p(t.data_ptr())), "teuk_read_device")
        t.record_stream(self.stream)
        self.torch.cuda.current_stream(self.device).wait_stream(self.stream)   # consumers run there
        return t

    def read_columns(self, i_first: int, n_cols: int, out=None):
        """local columns i_first .. i_first + n_cols - 1 -> CUDA tensor [4][L][n_theta][n_cols]"""
        if out is None:
            out = self.torch.empty((4, self.L, self.n_theta, n_cols), dtype=self.torch.float64, device=self.device)
        assert out.is_contiguous() and out.numel() == 4 * self.L * self.n_theta * n_cols
        self.stream.wait_stream(self.torch.cuda.current_stream(self.device))     # `out` may still be in use there
        _chk(lib.teuk_read_columns_device(self.h, i_first, n_cols, C.c_void_p(out.data_ptr())), "teuk_read_columns_device")
        self.torch.cuda.current_stream(self.device).wait_stream(self.stream)
        return out

    def write_columns(self, i_first: int, t):
        t = t.contiguous()
        assert t.is_cuda and t.dtype == self.torch.float64 and tuple(t.shape[:3]) == (4, self.L, self.n_theta)
        self.stream.wait_stream(self.torch.cuda.current_stream(self.device))     # t was produced there
        _chk(lib.teuk_write_columns_device(self.h, i_first, t.shape[3], C.c_void_p(t.data_ptr())), "teuk_write_columns_device")
        t.record_stream(self.stream)

    def observe(self, max_samples: int, allow_nonfinite=False):
        out = np.zeros((max(max_samples, 1), 4, self.L))
        cnt = C.c_long(0)
        rc = _chk(lib.teuk_observe(self.h, _np(out), max_samples, C.byref(cnt)), "teuk_observe",
                  allow=(ENONFINITE,) if allow_nonfinite else ())
        self.last_observe_status = rc
        return out[:cnt.value]

    def set_multipole_observer(self, rstar_obs, n_ell, capacity):
        self.n_ell = n_ell
        _chk(lib.teuk_set_multipole_observer(self.h, rstar_obs, n_ell, capacity), "teuk_set_multipole_observer")

    def observe_multipoles(self, max_samples: int) -> np.ndarray:
        out = np.zeros((max(max_samples, 1), self.n_ell, 2, self.L))
        cnt = C.c_long(0)
        _chk(lib.teuk_observe_multipoles(self.h, _np(out), max_samples, C.byref(cnt)), "teuk_observe_multipoles")
        return out[:cnt.value]

    def steps_done(self) -> int:
        n = C.c_long(0)
        _chk(lib.teuk_steps_done(self.h, C.byref(n)), "teuk_steps_done")
        return n.value

    def launch_count(self) -> int:
        n = C.c_long(0)
        _chk(lib.teuk_launch_count(self.h, C.byref(n)), "teuk_launch_count")
        return n.value

    def step_geometry(self) -> dict:
        o = (C.c_long * 6)()
        _chk(lib.teuk_step_geometry(self.h, o), "teuk_step_geometry")
        return dict(zip(("tile_i", "tile_j", "threads", "grid_x", "grid_y", "smem_bytes"), list(o)))

    def tables(self, half: bool) -> np.ndarray:
        rows = self.n_r - 1 if half else self.n_r
        out = np.zeros((8, self.L, self.n_theta, rows))
        _chk(lib.teuk_get_tables(self.h, int(half), _np(out)), "teuk_get_tables")
        return out

    def folded(self, half: bool, coef_variant: int) -> np.ndarray:
        rows = self.n_r - 1 if half else self.n_r
        out = np.zeros((8, self.n_theta, rows))
        _chk(lib.teuk_get_folded(self.h, int(half), coef_variant, _np(out)), "teuk_get_folded")
        return out

    def folded_static(self, half: bool, coef_variant: int, out: np.ndarray | None = None) -> np.ndarray:
        """teuk_get_folded_static: the same planes through the library's fixed device scratch (no allocation in the call)"""
        rows = self.n_r - 1 if half else self.n_r
        if out is None:
            out = np.zeros((8, self.n_theta, rows))
        _chk(lib.teuk_get_folded_static(self.h, int(half), coef_variant, _np(out)), "teuk_get_folded_static")
        return out

    def radial(self):
        r = np.zeros((2 * self.n_r - 1, 4))
        d = np.zeros((2 * self.n_r - 1, 4))
        _chk(lib.teuk_get_radial(self.h, _np(r), _np(d)), "teuk_get_radial")
        return r, d


def test_mp_op(op: str, L: int, a: np.ndarray, b: np.ndarray, on_device: bool) -> np.ndarray:
    code = {"add": 0, "sub": 1, "mul": 2, "div": 3, "sqrt": 4, "mul_d": 5}[op]
    a = np.ascontiguousarray(a, dtype=np.float64).reshape(-1, L)
    b = np.ascontiguousarray(b, dtype=np.float64).reshape(-1, L)
    out = np.zeros_like(a)
    _chk(lib.teuk_test_mp_op(code, L, _np(a), _np(b), _np(out), a.shape[0], int(on_device)), "teuk_test_mp_op")
    return out


def test_mp_fn(fn: str, a=None) -> list:
    code = {"exp": 0, "log": 1, "sin": 2, "cos": 3, "pi": 4, "ln2": 5}[fn]
    x = np.array(list(a if a is not None else [0.0]) + [0.0] * 4, dtype=np.float64)[:4].copy()
    out = np.zeros(4)
    _chk(lib.teuk_test_mp_fn(code, _np(x), _np(out)), "teuk_test_mp_fn")
    return [float(v) for v in out]


def bench_fp64(kind: str, iters: int = 20000, stream=None) -> float:
    code = {"dfma": 0, "dadd": 1, "dmul": 2}[kind]
    out = C.c_double(0)
    _chk(lib.teuk_bench_fp64(code, iters, C.byref(out), C.c_void_p(stream.cuda_stream if stream else 0)),
         "teuk_bench_fp64")
    return out.value
