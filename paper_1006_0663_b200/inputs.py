"""Seeded synthetic inputs shared by the oracle tests, the GPU tests and bench.py.

This module holds NONE of the method's arithmetic (no coefficients, no stencil,
no multiprecision): only the workload table of BASELINE.json / SURVEY.md §8(d)
and the fp64 initial-data recipe of SURVEY.md §8(c)-A14.  Both the oracle
(`oracle/`) and the CUDA path (`paper_1006_0663_b200.teuk`) receive the very
same doubles from here.

Initial data ("compact support at some initial time"):
    Phi_R(i, j) = A * exp(-(r*_i - c)^2 / (2 w^2)) * Y(theta_j),
    Phi_I = Pi_R = Pi_I = 0, rows i = 0 and i = N_r-1 zeroed.
(c, w, A) are drawn from a splitmix64 stream seeded per config.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

import numpy as np

SEED_BASE = 0x10060663
_MASK = (1 << 64) - 1


class SplitMix64:
    """Counter-based 64-bit generator (public-domain recipe by Steele/Lea/Flood)."""

    def __init__(self, seed: int):
        self.state = seed & _MASK

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & _MASK
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
        return z ^ (z >> 31)

    def uniform_pm1(self) -> float:
        """uniform in [-1, 1) with 53 random bits"""
        return (self.next_u64() >> 11) * (2.0 / (1 << 53)) - 1.0


@dataclass(frozen=True)
class Workload:
    name: str
    M: float
    a: float
    s: int
    m: int
    n_r: int
    n_theta: int
    rstar_min: float
    rstar_max: float
    steps: int
    precision: int          # limbs per real: 1 fp64, 2 dd, 4 qd
    profile: str            # "P2" | "P0" | "Y22m2"
    centre: tuple           # (c0, dc)
    width: tuple            # (w0, dw)
    amplitude: tuple        # (A0, dA)
    seed: int
    rstar_obs: float | None = None
    theta_obs: float | None = None
    dt_override: float | None = None

    @property
    def dr(self) -> float:
        return (self.rstar_max - self.rstar_min) / (self.n_r - 1)

    @property
    def dt(self) -> float:
        # dt = 0.5*((max-min)/(N_r-1)) in fp64 unless reduced for stability
        return self.dt_override if self.dt_override is not None else 0.5 * self.dr

    @property
    def observer(self) -> tuple:
        # default = centre of the r* range, theta = pi/2
        ro = self.rstar_obs if self.rstar_obs is not None else 0.5 * (self.rstar_min + self.rstar_max)
        to = self.theta_obs if self.theta_obs is not None else 0.5 * math.pi
        return ro, to

    def scaled(self, **kw) -> "Workload":
        return replace(self, **kw)


def stable_dt(w: Workload, z_max: float | None = None) -> float:
    """Harness time-step rule (reading A15b; pinned by tests/test_oracle_stability.py).  The two-step
    scheme of Eqs. (13)-(14) advances an undamped oscillator  Phi_tt = -omega^2 Phi  with
    amplification 1 + (omega dt)^4/8 per step, so for (s, m) != (0, 0) the stiffest angular mode near the peak of
    kappa = Delta/Sigma^2 (omega^2 ~ kappa_max [4/dtheta^2 + (|m|+|s|)^2 / sin^2(dtheta/2)], the second term being
    the pole potential of (m + s cos)^2/sin^2) grows without bound at BASELINE's dt = 0.5 dr*: config 2 gains
    e^0.125 per step there.  The harness passes dt = min(0.5 dr*, z / omega_max) with
        z = (8 / N_steps)^(1/4),
    i.e. the time step for which the scheme's own amplification of the stiffest mode over the WHOLE run,
    (1 + z^4/8)^N_steps, is at most e (config 2/3: z = 0.141, dt = 0.068 dr*; config 5, 1000 steps: z = 0.299).
    Work per update is unchanged.  Input generation only (fp64 estimate), not part of the method's arithmetic."""
    half_dr = 0.5 * w.dr
    if w.s == 0 and w.m == 0:
        return half_dr
    z = z_max if z_max is not None else (8.0 / max(w.steps, 1)) ** 0.25
    return min(half_dr, z / omega_max(w))


def omega_max(w: Workload) -> float:
    """fp64 estimate of the stiffest angular frequency of the pole rows (see `stable_dt`)."""
    rp = w.M + math.sqrt(w.M * w.M - w.a * w.a)
    r = rp + np.linspace(1e-3, 20.0, 20001)
    delta = r * r - 2.0 * w.M * r + w.a * w.a
    kappa_max = float(np.max(delta / (r * r + w.a * w.a) ** 2))
    dth = math.pi / w.n_theta
    om2 = kappa_max * (4.0 / dth ** 2 + (abs(w.m) + abs(w.s)) ** 2 / math.sin(0.5 * dth) ** 2)
    return math.sqrt(om2)


def config(k: int) -> Workload:
    """BASELINE.json configs 1..4 (SURVEY §8(d) 'Concrete inputs')."""
    if k == 1:
        return Workload("cfg1", 1.0, 0.0, 0, 0, 512, 16, -50.0, 150.0, 2000, 1, "P2",
                        (20.0, 2.0), (4.0, 0.5), (1.0, 0.1), SEED_BASE + 1, 40.0, 0.5 * math.pi)
    if k == 2:
        w = Workload("cfg2", 1.0, 0.9, -2, 2, 16384, 64, -300.0, 700.0, 20000, 1, "Y22m2",
                     (100.0, 5.0), (6.0, 1.0), (1.0, 0.0), SEED_BASE + 2)
        return replace(w, dt_override=stable_dt(w))
    if k == 3:
        return replace(config(2), name="cfg3", precision=2)   # same seed as cfg 2 ("same doubles")
    if k == 4:
        return Workload("cfg4", 1.0, 0.5, 0, 0, 8192, 32, -500.0, 1500.0, 50000, 4, "P0",
                        (50.0, 0.0), (5.0, 0.0), (1.0, 0.0), SEED_BASE + 4, 50.0, 0.5 * math.pi)
    raise ValueError(k)


def sweep_cell(n_r: int, n_theta: int, precision: int) -> Workload:
    """BASELINE.json config 5: a = 0.99, s = -2, m = 2, r* in [-300, 700] (A15), 1000 steps,
    dt from `stable_dt` (z = (8/1000)^(1/4) = 0.299)."""
    w = Workload(f"cfg5_{n_r}x{n_theta}_L{precision}", 1.0, 0.99, -2, 2, n_r, n_theta, -300.0, 700.0,
                 1000, precision, "Y22m2", (100.0, 5.0), (6.0, 1.0), (1.0, 0.0), SEED_BASE + 5)
    return replace(w, dt_override=stable_dt(w))


def theta_profile(profile: str, n_theta: int) -> np.ndarray:
    th = (np.arange(n_theta, dtype=np.float64) + 0.5) * (math.pi / n_theta)
    c = np.cos(th)
    if profile == "P0":
        return np.ones(n_theta)
    if profile == "P2":
        y = 0.5 * (3.0 * c * c - 1.0)
        half = n_theta // 2                  # mirrored so the data are exactly theta -> pi - theta symmetric
        y[n_theta - half:] = y[:half][::-1]
        return y
    if profile == "Y22m2":                   # _{-2}Y_{22}(theta) real profile
        return math.sqrt(5.0 / (64.0 * math.pi)) * (1.0 + c) ** 2
    raise ValueError(profile)


def pulse_parameters(w: Workload) -> tuple:
    g = SplitMix64(w.seed)
    c = w.centre[0] + w.centre[1] * g.uniform_pm1()
    wd = w.width[0] + w.width[1] * g.uniform_pm1()
    amp = w.amplitude[0] + w.amplitude[1] * g.uniform_pm1()
    return c, wd, amp


def initial_state(w: Workload) -> np.ndarray:
    """fp64 array [4][N_theta][N_r] (fields Phi_R, Phi_I, Pi_R, Pi_I; i fastest)."""
    c, wd, amp = pulse_parameters(w)
    rs = w.rstar_min + np.arange(w.n_r, dtype=np.float64) * w.dr
    radial = amp * np.exp(-((rs - c) ** 2) / (2.0 * wd * wd))
    u = np.zeros((4, w.n_theta, w.n_r), dtype=np.float64)
    u[0] = theta_profile(w.profile, w.n_theta)[:, None] * radial[None, :]
    u[:, :, 0] = 0.0
    u[:, :, -1] = 0.0
    return u


def random_state(n_r: int, n_theta: int, limbs: int, seed: int) -> np.ndarray:
    """Generic smooth-ish complex state with all four fields and all limbs populated,
    [4][limbs][N_theta][N_r]; used by parity tests that must exercise every term."""
    rng = np.random.Generator(np.random.PCG64(seed))
    i = np.arange(n_r)[None, :] / max(n_r - 1, 1)
    j = (np.arange(n_theta)[:, None] + 0.5) / n_theta
    out = np.zeros((4, limbs, n_theta, n_r))
    for f in range(4):
        ph = rng.uniform(0, 2 * np.pi, size=4)
        base = (np.sin(6 * np.pi * i + ph[0]) * np.cos(np.pi * j + ph[1])
                + 0.3 * np.sin(14 * np.pi * i + ph[2]) * np.cos(3 * np.pi * j + ph[3]))
        base = base * np.exp(-((i - 0.5) ** 2) / 0.08)
        out[f, 0] = base
        scale = 1.0
        for l in range(1, limbs):
            scale *= 2.0 ** -53
            # low limbs: |lo| <= ulp(hi)/4 so the planes are a valid normalised expansion
            out[f, l] = np.abs(out[f, l - 1]) * 2.0 ** -55 * rng.uniform(-1, 1, size=base.shape)
    out[:, :, :, 0] = 0.0
    out[:, :, :, -1] = 0.0
    return out
