"""ORACLE (test infrastructure, not product code) — arbitrary-precision reference pieces.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference`
legs may import this.  Nothing here is shared with the CUDA path.

Contents
--------
* `coefficients(...)`   the time-independent coefficients of the first-order system
                        (Eqs. 8-12; the matrices M, A, L are "found in
                        [20]" and are re-derived in DESIGN.md §3 from
                        Eqs. (1)-(7)).  Written with + - * / sqrt only,
                        so the SAME function runs on mpmath numbers (numeric reference)
                        and on sympy symbols (tests/test_coefficients_symbolic.py proves
                        the residual against Eq. (1) is identically zero).
* `tortoise(...)`, `r_of_rstar(...)`   Eq. (2) integrated and inverted.
* `radial_tables`, `theta_tables`      the 1-D tables handed to the C++ oracle, as
                        quad-double limbs (mpmath = stand-in for MPFR, 120 digits).
* `MPStepper`           a literal mpmath implementation of the two-step Lax-Wendroff
                        iteration, Eqs. (13)-(14), for tiny grids.

mpmath's log/exp/sin/cos/pi/findroot are used as library primitives.
"""
from __future__ import annotations

import mpmath as mp

P_WEIGHT = 3          # Eq. (4): Psi = exp(i m phi~) r^3 Phi   (reading A4)
MP_DPS = 120


def coefficients(r, delta_h, sin_t, cos_t, M, a, s, m, rp_minus_rm, sqrt=None, p=P_WEIGHT):
    """Coefficients of  Phi_t + b Phi_* = Pi,
                        Pi_t - b Pi_* = -alpha Pi + gamma Phi_* + kappa (Phi_thth + cot Phi_th) - W Phi
    at one (r, theta).  `delta_h` = r - r_+ (kept separately: near the horizon it is
    1e-16 .. 1e-101 and Delta must be formed from it), `rp_minus_rm` = r_+ - r_-.

    Returns dict with real numbers b, kappa and (re, im) pairs alpha, gamma, W.
    Cites: Delta, s, M, a: PAPER.md:51; b: Eq. (6); Sigma^2: Eq. (7) PAPER.md:80;
    D = diag(b,b,-b,-b): Eq. (11); S: Eq. (12) PAPER.md:98.
    """
    if sqrt is None:
        sqrt = mp.sqrt
    r2 = r * r
    a2 = a * a
    R = r2 + a2
    Delta = delta_h * (delta_h + rp_minus_rm)
    sin2 = sin_t * sin_t
    Sig2 = R * R - a2 * Delta * sin2                       # Eq. (7)
    Sig = sqrt(Sig2)
    b = R / Sig                                            # Eq. (6)
    rmM = r - M
    # alpha: coefficient of Phi_t
    al_re = 2 * s * (r * Delta - M * (r2 - a2)) / Sig2
    al_im = (4 * m * M * a * r + 2 * s * a * Delta * cos_t) / Sig2
    # c*: coefficient of -Phi_* before the r^p rescaling
    c_re = (2 * r * Delta + 2 * s * rmM * R) / Sig2
    c_im = (2 * m * a * R) / Sig2
    g = p * Delta / (r * R)
    g_star = (Delta / R) * p * (2 * rmM * r * R - Delta * (3 * r2 + a2)) / (r2 * R * R)
    b2 = b * b
    be_re = 2 * b2 * g + c_re
    be_im = c_im
    kappa = Delta / Sig2
    mc = m + s * cos_t
    V_re = kappa * (mc * mc / sin2 - s)
    V_im = -(4 * m * a * s * rmM) / Sig2
    W_re = V_re - b2 * (g_star + g * g) - c_re * g
    W_im = V_im - c_im * g
    b_star = (Delta / R) * a2 * sin2 * (R * rmM - 2 * r * Delta) / (Sig2 * Sig)
    ga_re = al_re * b + be_re - b * b_star
    ga_im = al_im * b + be_im
    return {"b": b, "kappa": kappa, "alpha": (al_re, al_im), "gamma": (ga_re, ga_im),
            "W": (W_re, W_im), "beta": (be_re, be_im), "b_star": b_star, "g": g, "g_star": g_star,
            "c": (c_re, c_im), "V": (V_re, V_im), "Sigma2": Sig2, "Delta": Delta}


# ----------------------------------------------------------------------------- Eq. (2)
def horizons(M, a):
    M = mp.mpf(M)
    a = mp.mpf(a)
    d = mp.sqrt(M * M - a * a)
    return M + d, M - d


def tortoise(r_minus_rp, M, a):
    """r*(r) with the integration constant of DESIGN.md reading A3:
    r* = r + 2M r_+/(r_+ - r_-) ln((r-r_+)/2M) - 2M r_-/(r_+ - r_-) ln((r-r_-)/2M).
    Argument is delta = r - r_+ so the horizon is approached without cancellation."""
    M = mp.mpf(M)
    rp, rm = horizons(M, a)
    d = mp.mpf(r_minus_rp)
    r = rp + d
    out = r + 2 * M * rp / (rp - rm) * mp.log(d / (2 * M))
    if rm != 0:
        out -= 2 * M * rm / (rp - rm) * mp.log((d + rp - rm) / (2 * M))
    return out


def r_of_rstar(rstar, M, a):
    """Invert Eq. (2): returns (r, delta = r - r_+).  Newton on y = ln(delta/2M):
    dr*/dy = delta * (r^2+a^2)/Delta = (r^2+a^2)/(delta + r_+ - r_-)."""
    M = mp.mpf(M)
    a_ = mp.mpf(a)
    rp, rm = horizons(M, a_)
    rstar = mp.mpf(rstar)
    # starting guess: near horizon r* ~ c_+ y ; far away r* ~ r
    cplus = 2 * M * rp / (rp - rm)
    y = (rstar - rp) / cplus if rstar < rp else mp.log(max(rstar, 2 * rp) / (2 * M))
    tol = mp.mpf(10) ** (-(mp.mp.dps - 8))
    for _ in range(200):
        d = 2 * M * mp.exp(y)
        r = rp + d
        F = tortoise(d, M, a_) - rstar
        dF = (r * r + a_ * a_) / (d + rp - rm)
        step = F / dF
        # damp huge steps (far-field start can overshoot in y)
        if abs(step) > 5:
            step = 5 * mp.sign(step)
        y -= step
        if abs(step) < tol * max(1, abs(y)):
            break
    else:
        raise RuntimeError("r(r*) Newton did not converge")
    d = 2 * M * mp.exp(y)
    return rp + d, d


# ----------------------------------------------------------------------------- limbs
def to_limbs(x, n=4):
    """Round an mpf to an n-limb expansion of doubles (each limb = RN of the remainder)."""
    out = []
    x = mp.mpf(x)
    for _ in range(n):
        hi = float(x)
        out.append(hi)
        x = x - mp.mpf(hi)
    return out


def from_limbs(limbs):
    tot = mp.mpf(0)
    for v in limbs:
        tot += mp.mpf(float(v))
    return tot


def radial_tables(M, a, rstar_min, rstar_max, n_r, i_lo=0, n_win=None):
    """r and delta = r - r_+ at the integer points i_lo..i_lo+n_win-1 and the half points
    between them, interleaved: index 2k -> node i_lo+k, 2k+1 -> node i_lo+k+1/2.
    r*_i = r*_min + i dr*, dr* = (r*_max - r*_min)/(N_r - 1) (reading A13).
    Returns (r_limbs [2n_win-1][4], delta_limbs [2n_win-1][4], dr_limbs[4])."""
    if n_win is None:
        n_win = n_r - i_lo
    with mp.workdps(MP_DPS):
        lo = mp.mpf(rstar_min)
        dr = (mp.mpf(rstar_max) - lo) / (n_r - 1)
        r_l, d_l = [], []
        for k in range(2 * n_win - 1):
            rs = lo + (2 * i_lo + k) * dr / 2
            r, d = r_of_rstar(rs, M, a)
            r_l.append(to_limbs(r))
            d_l.append(to_limbs(d))
        return r_l, d_l, to_limbs(dr)


def theta_tables(n_theta):
    """sin, cos of theta_j = (j + 1/2) pi / N_theta (cell-centred, reading A9), built for
    j < N_theta/2 and mirrored so the tables are exactly symmetric (reading A12).
    Returns (sin_limbs [N][4], cos_limbs [N][4], dtheta_limbs [4])."""
    with mp.workdps(MP_DPS):
        dth = mp.pi / n_theta
        sn = [None] * n_theta
        cs = [None] * n_theta
        for j in range((n_theta + 1) // 2):
            th = (j + mp.mpf(1) / 2) * dth
            sj, cj = to_limbs(mp.sin(th)), to_limbs(mp.cos(th))
            sn[j], cs[j] = sj, cj
            sn[n_theta - 1 - j] = list(sj)
            cs[n_theta - 1 - j] = [-v for v in cj]
        if n_theta % 2 == 1:
            cs[n_theta // 2] = [0.0, 0.0, 0.0, 0.0]
        return sn, cs, to_limbs(dth)


# ----------------------------------------------------------------------------- theta stencils
def fd_weights(order):
    """Centred finite-difference weights of accuracy `order` (2 or 10) on
    2N+1 = order+1 equally spaced points, derived exactly in rationals from the Taylor conditions
        sum_k w_k k^p = p! [p == derivative]   for p = 0..2N   (a Vandermonde system).
    Returns (c, d): first-derivative weights c[k], k = 1..N (antisymmetric: w_{-k} = -c[k], in units 1/h) and
    second-derivative weights d[k], k = 0..N (symmetric, in units 1/h^2), as fractions.Fraction."""
    from fractions import Fraction
    N = order // 2
    pts = list(range(-N, N + 1))
    n = len(pts)

    def solve(deriv):
        A = [[Fraction(x) ** p for x in pts] for p in range(n)]
        rhs = [Fraction(0)] * n
        f = 1
        for q in range(2, deriv + 1):
            f *= q
        rhs[deriv] = Fraction(f)
        # Gauss-Jordan in exact arithmetic
        M = [row + [r] for row, r in zip(A, rhs)]
        for col in range(n):
            piv = next(r for r in range(col, n) if M[r][col] != 0)
            M[col], M[piv] = M[piv], M[col]
            pv = M[col][col]
            M[col] = [v / pv for v in M[col]]
            for r in range(n):
                if r != col and M[r][col] != 0:
                    fct = M[r][col]
                    M[r] = [a - fct * b for a, b in zip(M[r], M[col])]
        return [M[r][n] for r in range(n)]
    w1, w2 = solve(1), solve(2)
    c = [w1[N + k] for k in range(1, N + 1)]
    d = [w2[N + k] for k in range(0, N + 1)]
    assert all(w1[N - k] == -w1[N + k] for k in range(1, N + 1)) and w1[N] == 0
    assert all(w2[N - k] == w2[N + k] for k in range(1, N + 1))
    return c, d


def fd_weight_limbs(order):
    """the same weights as quad-double limbs: (c_limbs [N][4], d_limbs [N+1][4])"""
    c, d = fd_weights(order)
    with mp.workdps(MP_DPS):
        cl = [to_limbs(mp.mpf(v.numerator) / mp.mpf(v.denominator)) for v in c]
        dl = [to_limbs(mp.mpf(v.numerator) / mp.mpf(v.denominator)) for v in d]
    return cl, dl


# ----------------------------------------------------------------------------- multipole projection (NEXT-2)
def swsh(s, l, m, theta):
    """Spin-weighted spherical harmonic _sY_lm(theta, phi = 0) (Goldberg et al. 1967 closed form),
    written with sin/cos of theta/2 so that the poles are regular:
      _sY_lm = (-1)^m sqrt[(l+m)!(l-m)!(2l+1) / (4 pi (l+s)!(l-s)!)]
               * sum_r C(l-s, r) C(l+s, r+s-m) (-1)^(l-r-s) sin^(2l-2r-s+m)(theta/2) cos^(2r+s-m)(theta/2)."""
    if l < max(abs(s), abs(m)):
        return mp.mpf(0)
    pref = (-1) ** m * mp.sqrt(mp.factorial(l + m) * mp.factorial(l - m) * (2 * l + 1)
                               / (4 * mp.pi * mp.factorial(l + s) * mp.factorial(l - s)))
    sh, ch = mp.sin(theta / 2), mp.cos(theta / 2)
    tot = mp.mpf(0)
    for r in range(0, l - s + 1):
        k = r + s - m
        if k < 0 or k > l + s:
            continue
        tot += mp.binomial(l - s, r) * mp.binomial(l + s, k) * (-1) ** (l - r - s) * sh ** (2 * l - 2 * r - s + m) * ch ** (2 * r + s - m)
    return pref * tot


def fejer_weights(n_theta):
    """Fejer's first quadrature rule: nodes x_j = cos(theta_j) with theta_j = (j + 1/2) pi / N are exactly the
    cell-centred theta grid, and  int_0^pi F(theta) sin(theta) dtheta ~ sum_j w_j F(theta_j),
        w_j = (2/N) [1 - 2 sum_{k=1}^{floor(N/2)} cos(2 k theta_j) / (4 k^2 - 1)],
    exact when F is a polynomial of degree < N in cos(theta) (spectrally accurate, unlike the midpoint rule whose
    O(dtheta^2) error would leak the dominant multipole into every other one)."""
    N = n_theta
    out = []
    for j in range(N):
        th = (j + mp.mpf(1) / 2) * mp.pi / N
        acc = mp.mpf(1)
        for k in range(1, N // 2 + 1):
            acc -= 2 * mp.cos(2 * k * th) / (4 * k * k - 1)
        out.append(2 * acc / N)
    return out


def multipole_weights(s, m, n_theta, n_ell):
    """Q[k][j] = 2 pi w_j _sY_{l_min+k, m}(theta_j), w_j = Fejer-1 weights: the projection
         a_l'(t) = int Phi(t, r*_obs, theta) conj(_sY_l'm) dOmega      (Fig. 1; reading A24)
    on the cell-centred theta grid, l_min = max(|s|, |m|).  Returns quad-double limbs [n_ell][n_theta][4]."""
    with mp.workdps(MP_DPS):
        dth = mp.pi / n_theta
        lmin = max(abs(s), abs(m))
        wf = fejer_weights(n_theta)
        out = []
        for k in range(n_ell):
            row = []
            for j in range(n_theta):
                th = (j + mp.mpf(1) / 2) * dth
                row.append(to_limbs(2 * mp.pi * wf[j] * swsh(s, lmin + k, m, th)))
            out.append(row)
        return out


# ----------------------------------------------------------------------------- Eqs. (13)-(14)
class MPStepper:
    """Literal mpmath implementation of one Lax-Wendroff iteration on a tiny
    grid, every quantity (tables included) at `dps` digits.  Used by pin P9 (precision ladder)
    as the brute-force end of the ladder.  State u[f][i][j], f = Phi_R, Phi_I, Pi_R, Pi_I."""

    def __init__(self, M, a, s, m, n_r, n_theta, rstar_min, rstar_max, dt, dps=100, theta_order=2):
        self.dps = dps
        self.theta_order = theta_order
        self.wc, self.wd = fd_weights(theta_order)
        with mp.workdps(dps):
            self.n_r, self.n_t = n_r, n_theta
            self.M, self.a, self.s, self.m = mp.mpf(M), mp.mpf(a), s, m
            self.dt = mp.mpf(dt)
            lo = mp.mpf(rstar_min)
            self.dr = (mp.mpf(rstar_max) - lo) / (n_r - 1)
            self.dth = mp.pi / n_theta
            self.sigma = 1 if abs(m) % 2 == 0 else -1
            rp, rm = horizons(self.M, self.a)
            th = [(j + mp.mpf(1) / 2) * self.dth for j in range(n_theta)]
            self.cot = [mp.cos(t) / mp.sin(t) for t in th]

            def row(rs):
                r, d = r_of_rstar(rs, self.M, self.a)
                return [coefficients(r, d, mp.sin(t), mp.cos(t), self.M, self.a, s, m, rp - rm) for t in th]
            self.ci = [row(lo + i * self.dr) for i in range(n_r)]
            self.ch = [row(lo + (i + mp.mpf(1) / 2) * self.dr) for i in range(n_r - 1)]
            self.u = None

    def set_initial(self, planes):
        """planes: numpy [4][N_theta][N_r] doubles"""
        with mp.workdps(self.dps):
            self.u = [[[mp.mpf(float(planes[f][j][i])) for j in range(self.n_t)] for i in range(self.n_r)]
                      for f in range(4)]
            for f in range(4):
                for j in range(self.n_t):
                    self.u[f][0][j] = mp.mpf(0)
                    self.u[f][self.n_r - 1][j] = mp.mpf(0)

    def _ghost(self, col, idx):
        nt = self.n_t
        if idx < 0:
            return self.sigma * col[-idx - 1]
        if idx >= nt:
            return self.sigma * col[2 * nt - 1 - idx]
        return col[idx]

    def _lam(self, col, j):
        if self.theta_order == 2:
            fm, fp = self._ghost(col, j - 1), self._ghost(col, j + 1)
            return (fp + fm - 2 * col[j]) / self.dth ** 2 + self.cot[j] * (fp - fm) / (2 * self.dth)
        N = self.theta_order // 2
        frac = lambda q: mp.mpf(q.numerator) / mp.mpf(q.denominator)
        second = frac(self.wd[0]) * col[j]
        first = mp.mpf(0)
        for k in range(1, N + 1):
            fp, fm = self._ghost(col, j + k), self._ghost(col, j - k)
            second += frac(self.wd[k]) * (fp + fm)
            first += frac(self.wc[k - 1]) * (fp - fm)
        return second / self.dth ** 2 + self.cot[j] * first / self.dth

    def _substep(self, c, lo4, hi4, j, base4, tau):
        """shared algebra of Eqs. (13)/(14): lo4/hi4 = the two neighbour columns (per field),
        base4 = value the bracket is subtracted from, tau = dt/2 or dt."""
        v = [(hi4[f][j] + lo4[f][j]) / 2 for f in range(4)]
        d = [(hi4[f][j] - lo4[f][j]) / self.dr for f in range(4)]
        mR = [(hi4[0][q] + lo4[0][q]) / 2 for q in range(self.n_t)]
        mI = [(hi4[1][q] + lo4[1][q]) / 2 for q in range(self.n_t)]
        al = mp.mpc(*c["alpha"]); ga = mp.mpc(*c["gamma"]); W = mp.mpc(*c["W"])
        phi, pi_ = mp.mpc(v[0], v[1]), mp.mpc(v[2], v[3])
        dphi = mp.mpc(d[0], d[1])
        lam = mp.mpc(self._lam(mR, j), self._lam(mI, j))
        S = -al * pi_ + ga * dphi + c["kappa"] * lam - W * phi
        b = c["b"]
        return [base4[0] - tau * (b * d[0] - v[2]),
                base4[1] - tau * (b * d[1] - v[3]),
                base4[2] - tau * (-b * d[2] - S.real),
                base4[3] - tau * (-b * d[3] - S.imag)]

    def step(self, n=1):
        with mp.workdps(self.dps):
            nr, nt = self.n_r, self.n_t
            for _ in range(n):
                u = self.u
                h = [[[None] * nt for _ in range(nr - 1)] for _ in range(4)]
                for i in range(nr - 1):
                    lo4 = [u[f][i] for f in range(4)]
                    hi4 = [u[f][i + 1] for f in range(4)]
                    for j in range(nt):
                        mean = [(hi4[f][j] + lo4[f][j]) / 2 for f in range(4)]
                        out = self._substep(self.ch[i][j], lo4, hi4, j, mean, self.dt / 2)
                        for f in range(4):
                            h[f][i][j] = out[f]
                un = [[[mp.mpf(0)] * nt for _ in range(nr)] for _ in range(4)]
                for i in range(1, nr - 1):
                    lo4 = [h[f][i - 1] for f in range(4)]
                    hi4 = [h[f][i] for f in range(4)]
                    for j in range(nt):
                        base = [u[f][i][j] for f in range(4)]
                        out = self._substep(self.ci[i][j], lo4, hi4, j, base, self.dt)
                        for f in range(4):
                            un[f][i][j] = out[f]
                self.u = un

    def read_limbs(self, n=4):
        """[4][n][N_theta][N_r] nested lists of doubles"""
        with mp.workdps(self.dps):
            return [[[[to_limbs(self.u[f][i][j], n)[k] for i in range(self.n_r)] for j in range(self.n_t)]
                     for k in range(n)] for f in range(4)]
