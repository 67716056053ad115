// ORACLE (test infrastructure, not product code): plain CPU implementation of the time step of
// the m-mode-reduced 2+1D Teukolsky equation as the paper's §III.B states it.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// use it.  It shares no code with the CUDA path (paper_1006_0663_b200/csrc/).
//
// What it computes, step by step in the paper's order (DESIGN.md §4 lists every reading A1..A23):
//   O3  coefficient tables b, alpha, gamma, W, kappa at (i, j) and (i+1/2, j) from
//       Eqs. (1),(4)-(7), evaluated in quad-double from 1-D tables r(r*),
//       r - r_+, sin/cos(theta_j) supplied by oracle/mp_ref.py (mpmath), then rounded to T.
//   O5  half step, Eq. (13) PAPER.md:102.
//   O6  full step, Eq. (14); radial Dirichlet rows.
//   polar ghosts f_{-1} = sigma f_0, f_{N} = sigma f_{N-1}, sigma = (-1)^{|m|}.
//   O7  observer at a fixed location, bilinear interpolation (reading A11).
// T is double, MP<2> (double-double) or MP<4> (quad-double) from mpx.hpp (tier 0: every operation exact, then
// rounded -- the arbitration tier), or FP<2> / FP<4> from mpf.hpp (tier 1: accurate IEEE-style operations, ~20x
// faster, pinned against tier 0; used for the full-length golden runs of configs 3 and 4).  The stepper below is
// ONE template: both tiers execute the same statements.  Coefficient tables are always built with MP<4>.
// A sub-window [i_lo, i_lo+n_win) of the radial grid can be stepped on its own (Dirichlet rows at
// the window edges, zeroed at set_initial); by the domain of dependence (i-1..i+1 per step) its
// interior [i_lo+k+1, i_lo+n_win-2-k] equals the full-grid result after k steps.
// Full grid: i_lo=0, n_win=N_r.
#include <cmath>
#include <cstdio>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif
#include "mpx.hpp"
#include "mpf.hpp"

using namespace orc;
typedef MP<4> Q;

enum { OK = 0, EINVAL = -1, ESTATE = -4 };

struct Params {
    double M, a, dt, rmin, rmax;
    int s, m, n_r, n_theta, prec, i_lo, n_win, theta_order;
};

// ---- O3: coefficients at one point, quad-double.  Same formulas as oracle/mp_ref.py::coefficients
// (pinned symbolically against Eq. (1) by tests/test_coefficients_symbolic.py and numerically
// against mpmath by tests/test_oracle_tables.py).  Order of outputs: b, aR, aI, gR, gI, WR, WI, kappa.
static void coefficients(const Params& P, const Q& rpm, const Q& r, const Q& dl, const Q& sn, const Q& cs, Q out[8]) {
    const int p = 3;                                  // Eq. (4)
    Q M(P.M), a(P.a);
    Q s((double)P.s), m((double)P.m);
    Q r2 = r * r, a2 = a * a;
    Q R = r2 + a2;
    Q Delta = dl * (dl + rpm);                        // Delta = (r - r_+)(r - r_-)
    Q sn2 = sn * sn;
    Q Sig2 = R * R - a2 * Delta * sn2;                // Eq. (7)
    Q Sig = sqrt(Sig2);
    Q b = R / Sig;                                    // Eq. (6)
    Q rmM = r - M;
    Q two(2.0), four(4.0), three(3.0), pp((double)p);
    Q alR = two * s * (r * Delta - M * (r2 - a2)) / Sig2;
    Q alI = (four * m * M * a * r + two * s * a * Delta * cs) / Sig2;
    Q cR = (two * r * Delta + two * s * rmM * R) / Sig2;
    Q cI = (two * m * a * R) / Sig2;
    Q g = pp * Delta / (r * R);
    Q gst = (Delta / R) * pp * (two * rmM * r * R - Delta * (three * r2 + a2)) / (r2 * R * R);
    Q b2 = b * b;
    Q beR = two * b2 * g + cR;
    Q beI = cI;
    Q kap = Delta / Sig2;
    Q mc = m + s * cs;
    Q VR = kap * (mc * mc / sn2 - s);
    Q VI = -(four * m * a * s * rmM) / Sig2;
    Q WR = VR - b2 * (gst + g * g) - cR * g;
    Q WI = VI - cI * g;
    Q bst = (Delta / R) * a2 * sn2 * (R * rmM - two * r * Delta) / (Sig2 * Sig);
    Q gaR = alR * b + beR - b * bst;
    Q gaI = alI * b + beI;
    out[0] = b; out[1] = alR; out[2] = alI; out[3] = gaR; out[4] = gaI; out[5] = WR; out[6] = WI; out[7] = kap;
}

template <class T> static inline T half_of(const T& x);
template <> inline double half_of<double>(const double& x) { return 0.5 * x; }
template <> inline MP<2> half_of<MP<2>>(const MP<2>& x) { return mul_d(x, 0.5); }
template <> inline MP<4> half_of<MP<4>>(const MP<4>& x) { return mul_d(x, 0.5); }
template <> inline FP<2> half_of<FP<2>>(const FP<2>& x) { return half(x); }
template <> inline FP<4> half_of<FP<4>>(const FP<4>& x) { return half(x); }

struct Base {
    Params P;
    virtual ~Base() {}
    virtual int build(const double* r_tab, const double* d_tab, const double* sin_tab, const double* cos_tab,
                      const double* dr_l, const double* dth_l, const double* wc_l, const double* wd_l) = 0;
    virtual int set_observer(double ro, double to, long cap) = 0;
    virtual int set_initial(const double* planes, int limbs_in) = 0;
    virtual int step(long n) = 0;
    virtual int read(double* planes) = 0;
    virtual int observe(double* out, long maxs, long* count) = 0;
    virtual int tables(int half, double* out, const double* in) = 0;
    virtual int cot_table(double* out) = 0;
    virtual int lambda(const double* f, double* out) = 0;
    virtual int set_multipole(double ro, int n_ell, const double* q_l, long cap) = 0;
    virtual int observe_multipoles(double* out, long maxs, long* count) = 0;
    long steps_done = 0;
};

template <class T>
struct Solver : Base {
    static constexpr int L = Limbs<T>::n;
    struct C { T b, aR, aI, gR, gI, WR, WI, k; };
    std::vector<C> ci, ch;                // [i*n_theta + j]; ch has n_win-1 rows
    std::vector<T> cot;
    T inv_dr, inv_dth2, inv_2dth, inv_dth, dt, half_dt;
    std::vector<T> wc, wd;                // theta stencil weights (first derivative k = 1..N, second k = 0..N)
    Q dr_q, dth_q;
    int sigma;
    std::vector<T> u[4], un[4], h[4];     // [i*n_theta + j]
    bool have_init = false;
    // observer
    long obs_cap = 0;
    int oi = -1, oj = -1;
    T wr, wt;
    std::vector<T> series;                // [sample][4]
    // multipole-projection observer (NEXT-2; Fig. 1; reading A24)
    long mp_cap = 0;
    int mp_n = 0, mp_i = -1;
    T mp_wr;
    std::vector<T> mp_q;                  // [n_ell][n_theta]
    std::vector<T> mp_series;             // [sample][n_ell][2]

    int build(const double* r_tab, const double* d_tab, const double* sin_tab, const double* cos_tab,
              const double* dr_l, const double* dth_l, const double* wc_l, const double* wd_l) override {
        const int nw = P.n_win, nt = P.n_theta;
        Q M(P.M), a(P.a);
        Q rpm = sqrt(M * M - a * a);
        rpm = rpm + rpm;                                        // r_+ - r_-
        dr_q = Q::from_limbs(dr_l, 4);
        dth_q = Q::from_limbs(dth_l, 4);
        Q one(1.0);
        inv_dr = narrow<T>(one / dr_q);
        inv_dth2 = narrow<T>(one / (dth_q * dth_q));
        inv_2dth = narrow<T>(one / (dth_q + dth_q));
        inv_dth = narrow<T>(one / dth_q);
        const int N = P.theta_order / 2;
        wc.resize(N); wd.resize(N + 1);
        for (int k = 0; k < N; ++k) wc[k] = narrow<T>(Q::from_limbs(wc_l + 4 * k, 4));
        for (int k = 0; k <= N; ++k) wd[k] = narrow<T>(Q::from_limbs(wd_l + 4 * k, 4));
        dt = T(P.dt);
        half_dt = half_of<T>(dt);
        sigma = (std::abs(P.m) % 2 == 0) ? 1 : -1;
        cot.resize(nt);
        for (int j = 0; j < nt; ++j) {
            Q sn = Q::from_limbs(sin_tab + 4 * j, 4), cs = Q::from_limbs(cos_tab + 4 * j, 4);
            cot[j] = narrow<T>(cs / sn);
        }
        ci.resize((size_t)nw * nt);
        ch.resize((size_t)(nw - 1) * nt);
#pragma omp parallel for schedule(dynamic, 4)
        for (int k = 0; k < 2 * nw - 1; ++k) {
            Q r = Q::from_limbs(r_tab + 4 * k, 4), dl = Q::from_limbs(d_tab + 4 * k, 4);
            for (int j = 0; j < nt; ++j) {
                Q sn = Q::from_limbs(sin_tab + 4 * j, 4), cs = Q::from_limbs(cos_tab + 4 * j, 4);
                Q c[8];
                coefficients(P, rpm, r, dl, sn, cs, c);
                C& d = (k % 2 == 0) ? ci[(size_t)(k / 2) * nt + j] : ch[(size_t)(k / 2) * nt + j];
                d.b = narrow<T>(c[0]); d.aR = narrow<T>(c[1]); d.aI = narrow<T>(c[2]); d.gR = narrow<T>(c[3]);
                d.gI = narrow<T>(c[4]); d.WR = narrow<T>(c[5]); d.WI = narrow<T>(c[6]); d.k = narrow<T>(c[7]);
            }
        }
        for (int f = 0; f < 4; ++f) {
            u[f].assign((size_t)nw * nt, T(0.0));
            un[f].assign((size_t)nw * nt, T(0.0));
            h[f].assign((size_t)(nw - 1) * nt, T(0.0));
        }
        return OK;
    }

    int set_observer(double ro, double to, long cap) override {
        if (cap < 0) return EINVAL;
        // reading A11: bilinear weights, fixed at setup, computed in quad-double
        Q x = (Q(ro) - Q(P.rmin)) / dr_q;
        Q y = Q(to) / dth_q - Q(0.5);
        int i0 = (int)std::floor(x.x[0]);
        int j0 = (int)std::floor(y.x[0]);
        if (i0 < 0 || x.x[0] > P.n_r - 1 || j0 < 0 || y.x[0] > P.n_theta - 1) return EINVAL;
        if (i0 > P.n_r - 2) i0 = P.n_r - 2;
        if (j0 > P.n_theta - 2) j0 = P.n_theta - 2;
        wr = narrow<T>(x - Q((double)i0));
        wt = narrow<T>(y - Q((double)j0));
        oi = i0 - P.i_lo;
        oj = j0;
        if (oi < 0 || oi + 1 >= P.n_win) return EINVAL;         // observer outside the stepped window
        obs_cap = cap;
        series.clear();
        series.reserve((size_t)cap * 4);
        return OK;
    }

    int set_multipole(double ro, int n_ell, const double* q_l, long cap) override {
        if (cap < 0 || n_ell < 1 || n_ell > 32) return EINVAL;
        Q x = (Q(ro) - Q(P.rmin)) / dr_q;
        int i0 = (int)std::floor(x.x[0]);
        if (i0 < 0 || x.x[0] > P.n_r - 1) return EINVAL;
        if (i0 > P.n_r - 2) i0 = P.n_r - 2;
        mp_wr = narrow<T>(x - Q((double)i0));
        mp_i = i0 - P.i_lo;
        if (mp_i < 0 || mp_i + 1 >= P.n_win) return EINVAL;
        mp_n = n_ell;
        mp_q.resize((size_t)n_ell * P.n_theta);
        for (size_t k = 0; k < mp_q.size(); ++k) mp_q[k] = narrow<T>(Q::from_limbs(q_l + 4 * k, 4));
        mp_cap = cap;
        mp_series.clear();
        return OK;
    }

    int observe_multipoles(double* out, long maxs, long* count) override {
        long n = mp_n ? (long)(mp_series.size() / (2 * mp_n)) : 0;
        if (n > maxs) n = maxs;
        for (size_t q = 0; q < (size_t)n * mp_n * 2; ++q)
            for (int k = 0; k < L; ++k) out[q * L + k] = Limbs<T>::get(mp_series[q], k);
        *count = n;
        return OK;
    }

    int set_initial(const double* planes, int limbs_in) override {
        if (limbs_in != 1 && limbs_in != L) return EINVAL;
        const int nw = P.n_win, nt = P.n_theta;
        for (int f = 0; f < 4; ++f)
            for (int j = 0; j < nt; ++j)
                for (int i = 0; i < nw; ++i) {
                    double l[4] = {0, 0, 0, 0};
                    for (int k = 0; k < limbs_in; ++k) l[k] = planes[(((size_t)f * limbs_in + k) * nt + j) * nw + i];
                    T v = Limbs<T>::make(l);
                    if (i == 0 || i == nw - 1) v = T(0.0);      // O4 / PAPER.md:112
                    u[f][(size_t)i * nt + j] = v;
                }
        have_init = true;
        steps_done = 0;
        series.clear();
        mp_series.clear();
        return OK;
    }

    // polar ghosts (cell-centred grid, reading A9): f_{-k} = sigma f_{k-1}, f_{N-1+k} = sigma f_{N-k}
    T ghost(const T* f, int idx) const {
        const int nt = P.n_theta;
        if (idx < 0) return sigma > 0 ? f[-idx - 1] : -f[-idx - 1];
        if (idx >= nt) return sigma > 0 ? f[2 * nt - 1 - idx] : -f[2 * nt - 1 - idx];
        return f[idx];
    }
    // theta_order 2:
    //   Lambda_j[f] = ((f_{j+1} + f_{j-1}) - 2 f_j)/dtheta^2 + cot(theta_j) (f_{j+1} - f_{j-1})/(2 dtheta)
    // theta_order 10 ("10th-order accurate" angular operator; 11-point centred stencils whose weights
    // come from oracle/mp_ref.py::fd_weights):
    //   Lambda_j[f] = (d_0 f_j + sum_k d_k (f_{j+k} + f_{j-k}))/dtheta^2 + cot(theta_j) (sum_k c_k (f_{j+k} - f_{j-k}))/dtheta
    T lam(const T* f, int j) const {
        if (P.theta_order == 2) {
            T fm = ghost(f, j - 1), fp = ghost(f, j + 1);
            T second = ((fp + fm) - (f[j] + f[j])) * inv_dth2;
            T first = cot[j] * ((fp - fm) * inv_2dth);
            return second + first;
        }
        const int N = P.theta_order / 2;
        T s2 = wd[0] * f[j];
        T s1 = T(0.0);
        for (int k = 1; k <= N; ++k) {
            T fp = ghost(f, j + k), fm = ghost(f, j - k);
            s2 = s2 + wd[k] * (fp + fm);
            s1 = s1 + wc[k - 1] * (fp - fm);
        }
        return s2 * inv_dth2 + cot[j] * (s1 * inv_dth);
    }

    // one sub-step source + update at a point; v = (mean fields), d = (differences)/dr*, lamR/I = Lambda[mean Phi]
    // returns S_Pi (complex) in the printed order: ((-alpha vPi + gamma dPhi) + kappa Lambda) - W vPhi
    static inline void source_pi(const C& c, const T v[4], const T dPhiR, const T dPhiI, const T lR, const T lI,
                                 T& SR, T& SI) {
        T t1R = -(c.aR * v[2] - c.aI * v[3]);
        T t1I = -(c.aR * v[3] + c.aI * v[2]);
        T t2R = c.gR * dPhiR - c.gI * dPhiI;
        T t2I = c.gR * dPhiI + c.gI * dPhiR;
        T t3R = c.k * lR, t3I = c.k * lI;
        T t4R = c.WR * v[0] - c.WI * v[1];
        T t4I = c.WR * v[1] + c.WI * v[0];
        SR = ((t1R + t2R) + t3R) - t4R;
        SI = ((t1I + t2I) + t3I) - t4I;
    }

    int step(long n) override {
        if (!have_init) return ESTATE;
        if (n < 0) return EINVAL;
        const int nw = P.n_win, nt = P.n_theta;
        for (long it = 0; it < n; ++it) {
            // ---- O5 half step, Eq. (13): i = 0..nw-2 are the points i+1/2
#pragma omp parallel
            {
                std::vector<T> mR(nt), mI(nt);
#pragma omp for schedule(static)
                for (int i = 0; i < nw - 1; ++i) {
                    const size_t a0 = (size_t)i * nt, a1 = (size_t)(i + 1) * nt;
                    for (int j = 0; j < nt; ++j) {
                        mR[j] = half_of<T>(u[0][a1 + j] + u[0][a0 + j]);
                        mI[j] = half_of<T>(u[1][a1 + j] + u[1][a0 + j]);
                    }
                    for (int j = 0; j < nt; ++j) {
                        const C& c = ch[a0 + j];
                        T v[4], d[4];
                        for (int f = 0; f < 4; ++f) {
                            v[f] = half_of<T>(u[f][a1 + j] + u[f][a0 + j]);
                            d[f] = (u[f][a1 + j] - u[f][a0 + j]) * inv_dr;
                        }
                        T SR, SI;
                        source_pi(c, v, d[0], d[1], lam(mR.data(), j), lam(mI.data(), j), SR, SI);
                        // D = diag(b, b, -b, -b) (Eq. 11);  S_Phi = Pi (Eq. 5)
                        h[0][a0 + j] = v[0] - half_dt * (c.b * d[0] - v[2]);
                        h[1][a0 + j] = v[1] - half_dt * (c.b * d[1] - v[3]);
                        h[2][a0 + j] = v[2] - half_dt * (-(c.b * d[2]) - SR);
                        h[3][a0 + j] = v[3] - half_dt * (-(c.b * d[3]) - SI);
                    }
                }
                // ---- O6 full step, Eq. (14): i = 1..nw-2
#pragma omp for schedule(static)
                for (int i = 1; i < nw - 1; ++i) {
                    const size_t am = (size_t)(i - 1) * nt, ap = (size_t)i * nt;
                    for (int j = 0; j < nt; ++j) {
                        mR[j] = half_of<T>(h[0][ap + j] + h[0][am + j]);
                        mI[j] = half_of<T>(h[1][ap + j] + h[1][am + j]);
                    }
                    for (int j = 0; j < nt; ++j) {
                        const C& c = ci[ap + j];
                        T v[4], d[4];
                        for (int f = 0; f < 4; ++f) {
                            v[f] = half_of<T>(h[f][ap + j] + h[f][am + j]);
                            d[f] = (h[f][ap + j] - h[f][am + j]) * inv_dr;
                        }
                        T SR, SI;
                        source_pi(c, v, d[0], d[1], lam(mR.data(), j), lam(mI.data(), j), SR, SI);
                        un[0][ap + j] = u[0][ap + j] - dt * (c.b * d[0] - v[2]);
                        un[1][ap + j] = u[1][ap + j] - dt * (c.b * d[1] - v[3]);
                        un[2][ap + j] = u[2][ap + j] - dt * (-(c.b * d[2]) - SR);
                        un[3][ap + j] = u[3][ap + j] - dt * (-(c.b * d[3]) - SI);
                    }
                }
            }
            for (int f = 0; f < 4; ++f) {                      // radial boundary
                for (int j = 0; j < nt; ++j) {
                    un[f][j] = T(0.0);
                    un[f][(size_t)(nw - 1) * nt + j] = T(0.0);
                }
                u[f].swap(un[f]);
            }
            ++steps_done;
            if (mp_cap > 0 && (long)(mp_series.size() / (2 * mp_n)) < mp_cap) {
                // a_l' = sum_j Q_l'(theta_j) [ (1 - w) Phi(i0, j) + w Phi(i0 + 1, j) ],  j = 0 .. N_theta - 1 in order
                T one(1.0);
                for (int k = 0; k < mp_n; ++k)
                    for (int c = 0; c < 2; ++c) {
                        T acc(0.0);
                        for (int j = 0; j < nt; ++j) {
                            T v = (one - mp_wr) * u[c][(size_t)mp_i * nt + j] + mp_wr * u[c][(size_t)(mp_i + 1) * nt + j];
                            acc = acc + mp_q[(size_t)k * nt + j] * v;
                        }
                        mp_series.push_back(acc);
                    }
            }
            if (obs_cap > 0 && (long)(series.size() / 4) < obs_cap) {   // O7
                T one(1.0);
                for (int f = 0; f < 4; ++f) {
                    const T& u00 = u[f][(size_t)oi * nt + oj];
                    const T& u10 = u[f][(size_t)(oi + 1) * nt + oj];
                    const T& u01 = u[f][(size_t)oi * nt + oj + 1];
                    const T& u11 = u[f][(size_t)(oi + 1) * nt + oj + 1];
                    T lo = (one - wr) * u00 + wr * u10;
                    T hi = (one - wr) * u01 + wr * u11;
                    series.push_back((one - wt) * lo + wt * hi);
                }
            }
        }
        return OK;
    }

    int read(double* planes) override {
        if (!have_init) return ESTATE;
        const int nw = P.n_win, nt = P.n_theta;
        for (int f = 0; f < 4; ++f)
            for (int k = 0; k < L; ++k)
                for (int j = 0; j < nt; ++j)
                    for (int i = 0; i < nw; ++i)
                        planes[(((size_t)f * L + k) * nt + j) * nw + i] = Limbs<T>::get(u[f][(size_t)i * nt + j], k);
        return OK;
    }

    int observe(double* out, long maxs, long* count) override {
        long n = (long)(series.size() / 4);
        if (n > maxs) n = maxs;
        for (long q = 0; q < n; ++q)
            for (int f = 0; f < 4; ++f)
                for (int k = 0; k < L; ++k) out[((size_t)q * 4 + f) * L + k] = Limbs<T>::get(series[(size_t)q * 4 + f], k);
        *count = n;
        return OK;
    }

    int tables(int half, double* out, const double* in) override {   // [8][L][n_theta][rows]
        const int nt = P.n_theta, rows = half ? P.n_win - 1 : P.n_win;
        std::vector<C>& tab = half ? ch : ci;
        for (int i = 0; i < rows; ++i)
            for (int j = 0; j < nt; ++j) {
                C& c = tab[(size_t)i * nt + j];
                T* fld[8] = {&c.b, &c.aR, &c.aI, &c.gR, &c.gI, &c.WR, &c.WI, &c.k};
                for (int q = 0; q < 8; ++q) {
                    double l[4] = {0, 0, 0, 0};
                    for (int k = 0; k < L; ++k) {
                        size_t idx = (((size_t)q * L + k) * nt + j) * rows + i;
                        if (in) l[k] = in[idx]; else out[idx] = Limbs<T>::get(*fld[q], k);
                    }
                    if (in) *fld[q] = Limbs<T>::make(l);
                }
            }
        return OK;
    }

    int cot_table(double* out) override {
        for (int j = 0; j < P.n_theta; ++j)
            for (int k = 0; k < L; ++k) out[(size_t)k * P.n_theta + j] = Limbs<T>::get(cot[j], k);
        return OK;
    }

    int lambda(const double* f, double* out) override {            // f, out: [L][n_theta]
        const int nt = P.n_theta;
        std::vector<T> v(nt);
        for (int j = 0; j < nt; ++j) {
            double l[4] = {0, 0, 0, 0};
            for (int k = 0; k < L; ++k) l[k] = f[(size_t)k * nt + j];
            v[j] = Limbs<T>::make(l);
        }
        for (int j = 0; j < nt; ++j) {
            T r = lam(v.data(), j);
            for (int k = 0; k < L; ++k) out[(size_t)k * nt + j] = Limbs<T>::get(r, k);
        }
        return OK;
    }
};

// test hook for pin P1: out = a (op) b on N-limb numbers; op: 0 add, 1 sub, 2 mul, 3 div, 4 sqrt(a), 5 a*b[0]
template <int N> static int mp_op_n(int op, const double* a, const double* b, double* out) {
    MP<N> x = Limbs<MP<N>>::make(a), y = Limbs<MP<N>>::make(b), r;
    switch (op) {
        case 0: r = x + y; break;
        case 1: r = x - y; break;
        case 2: r = x * y; break;
        case 3: r = x / y; break;
        case 4: r = sqrt(x); break;
        case 5: r = mul_d(x, b[0]); break;
        default: return EINVAL;
    }
    for (int k = 0; k < N; ++k) out[k] = r.x[k];
    return OK;
}

// the same hook for the fast tier (mpf.hpp); op 6: half(a)
template <int N> static int mpf_op_n(int op, const double* a, const double* b, double* out) {
    FP<N> x = Limbs<FP<N>>::make(a), y = Limbs<FP<N>>::make(b), r;
    switch (op) {
        case 0: r = x + y; break;
        case 1: r = x - y; break;
        case 2: r = x * y; break;
        case 5: r = mul_d(x, b[0]); break;
        case 6: r = half(x); break;
        default: return EINVAL;
    }
    for (int k = 0; k < N; ++k) out[k] = r.x[k];
    return OK;
}

// ------------------------------------------------------------------------------------ C ABI
extern "C" {

int oracle_create(double M, double a, int s, int m, int n_r, int n_theta, double rmin, double rmax, double dt,
                  int precision, int i_lo, int n_win, const double* r_tab, const double* d_tab, const double* sin_tab,
                  const double* cos_tab, const double* dr_l, const double* dth_l, int theta_order, const double* wc_l,
                  const double* wd_l, int tier, void** out) {
    if (!(M > 0) || !(std::fabs(a) < M) || n_r < 3 || n_theta < 2 || !(dt > 0) || !(rmin < rmax) || !out) return EINVAL;
    if ((theta_order != 2 && theta_order != 10) || n_theta < theta_order / 2) return EINVAL;
    if (i_lo < 0 || n_win < 3 || i_lo + n_win > n_r) return EINVAL;
    Base* b = nullptr;
    if (precision == 1) b = new Solver<double>();
    else if (precision == 2 && tier == 0) b = new Solver<MP<2>>();
    else if (precision == 4 && tier == 0) b = new Solver<MP<4>>();
    else if (precision == 2 && tier == 1) b = new Solver<FP<2>>();
    else if (precision == 4 && tier == 1) b = new Solver<FP<4>>();
    else return EINVAL;
    b->P = Params{M, a, dt, rmin, rmax, s, m, n_r, n_theta, precision, i_lo, n_win, theta_order};
    int rc = b->build(r_tab, d_tab, sin_tab, cos_tab, dr_l, dth_l, wc_l, wd_l);
    if (rc != OK) { delete b; return rc; }
    *out = b;
    return OK;
}
int oracle_set_observer(void* h, double ro, double to, long cap) { return ((Base*)h)->set_observer(ro, to, cap); }
int oracle_set_initial(void* h, const double* planes, int limbs_in) { return ((Base*)h)->set_initial(planes, limbs_in); }
int oracle_step(void* h, long n) { return ((Base*)h)->step(n); }
int oracle_read(void* h, double* planes) { return ((Base*)h)->read(planes); }
int oracle_observe(void* h, double* out, long maxs, long* count) { return ((Base*)h)->observe(out, maxs, count); }
int oracle_get_tables(void* h, int half, double* out) { return ((Base*)h)->tables(half, out, nullptr); }
int oracle_set_tables(void* h, int half, const double* in) { return ((Base*)h)->tables(half, nullptr, in); }
int oracle_get_cot(void* h, double* out) { return ((Base*)h)->cot_table(out); }
int oracle_lambda(void* h, const double* f, double* out) { return ((Base*)h)->lambda(f, out); }
int oracle_set_multipole(void* h, double ro, int n_ell, const double* q_l, long cap) { return ((Base*)h)->set_multipole(ro, n_ell, q_l, cap); }
int oracle_observe_multipoles(void* h, double* out, long maxs, long* count) { return ((Base*)h)->observe_multipoles(out, maxs, count); }
int oracle_steps_done(void* h, long* n) { *n = ((Base*)h)->steps_done; return OK; }
void oracle_destroy(void* h) { delete (Base*)h; }
int oracle_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n;
    return 1;
#endif
}

int oracle_mp_op(int op, int N, const double* a, const double* b, double* out) {
    if (N == 2) return mp_op_n<2>(op, a, b, out);
    if (N == 4) return mp_op_n<4>(op, a, b, out);
    return EINVAL;
}

int oracle_mpf_op(int op, int N, const double* a, const double* b, double* out) {
    if (N == 2) return mpf_op_n<2>(op, a, b, out);
    if (N == 4) return mpf_op_n<4>(op, a, b, out);
    return EINVAL;
}
// batched form of both hooks for the corpus tests: n operand pairs, rows of N doubles
int oracle_mp_op_batch(int tier, int op, int N, long n, const double* a, const double* b, double* out) {
    for (long k = 0; k < n; ++k) {
        int rc = tier ? oracle_mpf_op(op, N, a + k * N, b + k * N, out + k * N)
                      : oracle_mp_op(op, N, a + k * N, b + k * N, out + k * N);
        if (rc != OK) return rc;
    }
    return OK;
}
int oracle_set_zero_fast_path(int on) { int old = g_zero_fast_path; g_zero_fast_path = on; return old; }

}  // extern "C"
