// ORACLE (test infrastructure, not product code) -- the FAST arithmetic tier.
//
// mpx.hpp (MP<N>) is the arbitration tier: every operation exact, then rounded; ~700 cycles per
// operation, which puts configs 3 and 4 at full length (2.1e10 / 1.3e10 updates) out of reach.
// This header is the tier SURVEY.md 8(c) contracts ("accurate IEEE-style additions, FMA-based
// twoProd"): FP<N>, the same number format (N non-overlapping doubles, leading limb first;
// PAPER.md:134, reading A20), with operations that keep every term of order >= eps^N and stay
// accurate under cancellation, but round once per operation with a bound of a few eps^N instead
// of 1/2 ulp of the last limb.  It is pinned operation by operation against MP<N>
// (tests/test_oracle_fast_tier.py: random, exact and massive-cancellation operands; the bounds
// asserted there are the ones stated beside each operator below) and the stepper built on it is
// pinned against the MP<N> stepper and the mpmath ladder.  It shares no code with the CUDA
// arithmetic (csrc/mp.cuh: branch-free fixed sequences, "sloppy" adds) -- different algorithms:
//   N = 2: the textbook double-word algorithms (two TwoSums per add; TwoProd + FMA cross terms).
//   N = 4: sort / cascade the exact partial terms, then DISTILL: one bottom-up chain of TwoSums
//          (an error-free transformation of the vector) and one top-down chain that emits a limb
//          whenever a rounding error appears.  Only TwoSum (no ordering precondition) is used, so
//          the value is preserved exactly whatever the operand magnitudes; ordering only decides
//          how well separated the limbs come out.
// The only fast paths are the exact identities x + 0 = x and x * 0 = 0 (config 4 is a real
// problem: half of its complex arithmetic has a zero operand); tests switch them off and check
// that nothing changes.  Compile with -ffp-contract=off (explicit std::fma only).
#pragma once
#include "mpx.hpp"

namespace orc {

static int g_zero_fast_path = 1;      // test hook: oracle_set_zero_fast_path

// Requires |a| >= |b| or a == 0 (Dekker).  Used only where that holds by construction.
static inline void quick_two_sum(double a, double b, double& s, double& e) {
    s = a + b;
    e = b - (s - a);
}

template <int N>
struct FP {
    double x[N];
    FP() { for (int k = 0; k < N; ++k) x[k] = 0.0; }
    FP(double d) { x[0] = d; for (int k = 1; k < N; ++k) x[k] = 0.0; }
    FP(int d) : FP((double)d) {}
};

template <int N> struct Limbs<FP<N>> {
    static constexpr int n = N;
    static double get(const FP<N>& v, int k) { return v.x[k]; }
    static FP<N> make(const double* p) { FP<N> r; for (int k = 0; k < N; ++k) r.x[k] = p[k]; return r; }
};

template <int N> static inline FP<N> operator-(const FP<N>& a) {
    FP<N> r;
    for (int k = 0; k < N; ++k) r.x[k] = -a.x[k];
    return r;
}

// Multiplication by 1/2: exact limb by limb (a power of two; no underflow at the magnitudes of the run).
template <int N> static inline FP<N> half(const FP<N>& a) {
    FP<N> r;
    for (int k = 0; k < N; ++k) r.x[k] = 0.5 * a.x[k];
    return r;
}

// ---- distillation: NIN doubles t[0..] (roughly decreasing) -> NOUT limbs r[0..] with the same sum
// up to the rounding of the LAST limb.  Pass 1 (bottom-up TwoSum chain) leaves v[0] = fl(sum) and
// the individual rounding errors in v[1..]; it is an exact transformation of the vector.  Pass 2
// (top-down) adds v[i] into a running value q and emits fl(q + v[i]) as the next limb whenever the
// addition was inexact, carrying the exact error on; zero errors are absorbed.  The last limb takes
// what is left by plain additions.
template <int NIN, int NOUT>
static inline void distill(const double* t, double* r) {
    double v[NIN];
    double s = t[NIN - 1];
    for (int i = NIN - 2; i >= 0; --i) {
        double e;
        two_sum(t[i], s, s, e);
        v[i + 1] = e;
    }
    v[0] = s;
    for (int k = 0; k < NOUT; ++k) r[k] = 0.0;
    int j = 0;
    double q = v[0];
    for (int i = 1; i < NIN; ++i) {
        if (j == NOUT - 1) { q += v[i]; continue; }
        double sum, err;
        two_sum(q, v[i], sum, err);
        if (err != 0.0) { r[j++] = sum; q = err; }
        else q = sum;
    }
    r[j] = q;
}

// ---- N-limb addition, |error| <= eps^N |a + b| (eps = 2^-53; the pin measures 0.13 eps^N), cancellation included:
// merge the 2N limbs by decreasing magnitude, distil to N+1 limbs, distil again to N.
template <int N> static inline FP<N> operator+(const FP<N>& a, const FP<N>& b) {
    if (g_zero_fast_path) {
        if (b.x[0] == 0.0) return a;
        if (a.x[0] == 0.0) return b;
    }
    double f[2 * N];
    int i = 0, j = 0;
    for (int k = 0; k < 2 * N; ++k) {
        if (j >= N || (i < N && std::fabs(a.x[i]) >= std::fabs(b.x[j]))) f[k] = a.x[i++];
        else f[k] = b.x[j++];
    }
    double w[N + 1];
    distill<2 * N, N + 1>(f, w);
    FP<N> r;
    distill<N + 1, N>(w, r.x);
    return r;
}
template <int N> static inline FP<N> operator-(const FP<N>& a, const FP<N>& b) { return a + (-b); }

// Exact cascade accumulator of N+1 doubles: acc[k] holds terms of order eps^k relative to the
// product.  put(k, t) adds t into acc[k] with TwoSum and passes the rounding error down to
// acc[k+1], ...; what falls below acc[N] is of order eps^(N+1) and is dropped.
template <int N>
struct Cascade {
    double acc[N + 1];
    Cascade() { for (int k = 0; k <= N; ++k) acc[k] = 0.0; }
    void put(int k, double t) {
        for (; k <= N && t != 0.0; ++k) two_sum(acc[k], t, acc[k], t);
    }
    FP<N> result() const {
        double w[N + 1];
        distill<N + 1, N + 1>(acc, w);
        FP<N> r;
        distill<N + 1, N>(w, r.x);
        return r;
    }
};

// ---- N-limb multiplication, |error| <= eps^N |a b| (measured 0.11 eps^N): partial products a_i b_j with i + j < N
// exactly (TwoProd: product to order i+j, its error to order i+j+1), those with i + j = N rounded.
template <int N> static inline FP<N> operator*(const FP<N>& a, const FP<N>& b) {
    if (g_zero_fast_path && (a.x[0] == 0.0 || b.x[0] == 0.0)) return FP<N>(0.0);
    Cascade<N> c;
    for (int ord = 0; ord <= N; ++ord)
        for (int i = 0; i < N; ++i) {
            int j = ord - i;
            if (j < 0 || j >= N) continue;
            if (ord == N) { c.put(N, a.x[i] * b.x[j]); continue; }
            double p, e;
            two_prod(a.x[i], b.x[j], p, e);
            c.put(ord, p);
            c.put(ord + 1, e);
        }
    return c.result();
}

// N-limb times double, same bound.
template <int N> static inline FP<N> mul_d(const FP<N>& a, double d) {
    if (g_zero_fast_path && (a.x[0] == 0.0 || d == 0.0)) return FP<N>(0.0);
    Cascade<N> c;
    for (int i = 0; i < N; ++i) {
        double p, e;
        two_prod(a.x[i], d, p, e);
        c.put(i, p);
        c.put(i + 1, e);
    }
    return c.result();
}

// ---- N = 2: the textbook double-word algorithms.
// Addition with two TwoSums ("accurate" double-word sum): |error| <= 3 eps^2 |a + b|.
template <> inline FP<2> operator+(const FP<2>& a, const FP<2>& b) {
    if (g_zero_fast_path) {
        if (b.x[0] == 0.0) return a;
        if (a.x[0] == 0.0) return b;
    }
    double sh, sl, th, tl;
    two_sum(a.x[0], b.x[0], sh, sl);
    two_sum(a.x[1], b.x[1], th, tl);
    double c = sl + th;
    double vh, vl;
    quick_two_sum(sh, c, vh, vl);
    double w = tl + vl;
    FP<2> r;
    quick_two_sum(vh, w, r.x[0], r.x[1]);
    return r;
}
// Product: TwoProd of the leading limbs, cross terms and a_1 b_1 by FMA: |error| <= 5 eps^2 |a b|.
template <> inline FP<2> operator*(const FP<2>& a, const FP<2>& b) {
    if (g_zero_fast_path && (a.x[0] == 0.0 || b.x[0] == 0.0)) return FP<2>(0.0);
    double p, e;
    two_prod(a.x[0], b.x[0], p, e);
    double t = a.x[1] * b.x[1];
    t = std::fma(a.x[0], b.x[1], t);
    t = std::fma(a.x[1], b.x[0], t);
    e = e + t;
    FP<2> r;
    quick_two_sum(p, e, r.x[0], r.x[1]);
    return r;
}
template <> inline FP<2> mul_d(const FP<2>& a, double d) {
    if (g_zero_fast_path && (a.x[0] == 0.0 || d == 0.0)) return FP<2>(0.0);
    double p, e;
    two_prod(a.x[0], d, p, e);
    e = std::fma(a.x[1], d, e);
    FP<2> r;
    quick_two_sum(p, e, r.x[0], r.x[1]);
    return r;
}

}  // namespace orc
