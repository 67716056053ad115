// ORACLE (test infrastructure, not product code).  Scalar N-limb floating-point expansions
// ("double-double" N=2, "quad-double" N=4; "high-precision datatypes ... are
// implemented using a representation based on the appropriate number of double-precision
// floats"; reading A20 in DESIGN.md).
//
// Design: every operation is EXACT-THEN-ROUND.  The exact sum (or the sum of all partial
// products of order >= eps^N) is accumulated as a non-overlapping floating-point expansion
// using the error-free transformations TwoSum / TwoProd(FMA) (Knuth; Dekker; Shewchuk's
// Grow-Expansion), and only then rounded to N limbs.  This is slow and has no fast paths, so
// it can be checked by eye; it shares no code with the CUDA arithmetic layer (csrc/mp.cuh).
// Compile with -ffp-contract=off: the only FMAs are the explicit std::fma calls.
#pragma once
#include <cmath>
#include <cstring>

namespace orc {

static inline void two_sum(double a, double b, double& s, double& e) {
    s = a + b;
    double bb = s - a;
    e = (a - (s - bb)) + (b - bb);
}
static inline void two_prod(double a, double b, double& p, double& e) {
    p = a * b;
    e = std::fma(a, b, -p);
}

// Exact accumulator: a non-overlapping expansion, components in increasing magnitude.
template <int CAP>
struct Acc {
    double e[CAP];
    int n = 0;
    void add(double b) {                 // Grow-Expansion with zero elimination
        double q = b;
        int k = 0;
        for (int i = 0; i < n; ++i) {
            double s, h;
            two_sum(q, e[i], s, h);
            q = s;
            if (h != 0.0) e[k++] = h;
        }
        if (q != 0.0 || k == 0) e[k++] = q;
        n = k;
    }
    // Round to N limbs: leading limb = fl(total) (up to a final-ulp tie), each further limb the
    // rounded remainder; result satisfies |x[k+1]| <= ulp(x[k])/2.
    template <int N>
    void round_to(double* x) const {
        Acc<CAP> w = *this;
        for (int k = 0; k < N; ++k) {
            // approximate the remaining total from the small end, then remove it exactly
            double t = 0.0;
            for (int i = 0; i < w.n; ++i) t += w.e[i];
            // one correction pass makes t the correctly rounded total in all but tie cases
            Acc<CAP> c = w;
            c.add(-t);
            double t2 = 0.0;
            for (int i = 0; i < c.n; ++i) t2 += c.e[i];
            double tt = t + t2;
            x[k] = tt;
            w.add(-tt);
        }
    }
};

template <int N>
struct MP {
    double x[N];
    MP() { for (int k = 0; k < N; ++k) x[k] = 0.0; }
    MP(double d) { x[0] = d; for (int k = 1; k < N; ++k) x[k] = 0.0; }
    MP(int d) : MP((double)d) {}
    static MP from_limbs(const double* p, int n_in) {      // exact if n_in <= N, else rounded
        Acc<16> acc;
        for (int k = 0; k < n_in; ++k) acc.add(p[k]);
        MP r;
        acc.template round_to<N>(r.x);
        return r;
    }
};

template <int N> static inline MP<N> operator-(const MP<N>& a) {
    MP<N> r;
    for (int k = 0; k < N; ++k) r.x[k] = -a.x[k];
    return r;
}
template <int N> static inline MP<N> operator+(const MP<N>& a, const MP<N>& b) {
    Acc<3 * N + 8> acc;
    for (int k = N - 1; k >= 0; --k) { acc.add(a.x[k]); acc.add(b.x[k]); }
    MP<N> r;
    acc.template round_to<N>(r.x);
    return r;
}
template <int N> static inline MP<N> operator-(const MP<N>& a, const MP<N>& b) { return a + (-b); }

template <int N> static inline MP<N> operator*(const MP<N>& a, const MP<N>& b) {
    // all partial products a_i b_j with i + j <= N-1 exactly (TwoProd), those with i + j == N
    // rounded (their rounding error is O(eps^(N+1))); higher orders dropped.
    Acc<2 * N * N + 8> acc;
    for (int ord = N; ord >= 0; --ord)
        for (int i = 0; i < N; ++i) {
            int j = ord - i;
            if (j < 0 || j >= N) continue;
            if (ord == N) {
                acc.add(a.x[i] * b.x[j]);
            } else {
                double p, e;
                two_prod(a.x[i], b.x[j], p, e);
                acc.add(e);
                acc.add(p);
            }
        }
    MP<N> r;
    acc.template round_to<N>(r.x);
    return r;
}

template <int N> static inline MP<N> mul_d(const MP<N>& a, double d) {    // exact product, then round
    Acc<3 * N + 8> acc;
    for (int i = N - 1; i >= 0; --i) {
        double p, e;
        two_prod(a.x[i], d, p, e);
        acc.add(e);
        acc.add(p);
    }
    MP<N> r;
    acc.template round_to<N>(r.x);
    return r;
}

template <int N> static inline MP<N> operator/(const MP<N>& a, const MP<N>& b) {
    // long division with an EXACT remainder: N+2 quotient digits q_k = fl(fl(rem) / b_0),
    // rem <- rem - q_k * b held exactly in the accumulator; quotient = round(sum q_k).
    Acc<2 * N * (N + 3) + 8> rem;
    Acc<2 * N + 8> q;
    for (int k = N - 1; k >= 0; --k) rem.add(a.x[k]);
    for (int k = 0; k < N + 2; ++k) {
        double r0 = 0.0;
        for (int i = 0; i < rem.n; ++i) r0 += rem.e[i];
        double qk = r0 / b.x[0];
        q.add(qk);
        for (int i = N - 1; i >= 0; --i) {
            double p, e;
            two_prod(b.x[i], qk, p, e);
            rem.add(-e);
            rem.add(-p);
        }
    }
    MP<N> r;
    q.template round_to<N>(r.x);
    return r;
}

template <int N> static inline MP<N> sqrt(const MP<N>& a) {
    if (a.x[0] == 0.0) return MP<N>(0.0);
    MP<N> x(std::sqrt(a.x[0]));
    for (int it = 0; it < 4; ++it)                       // Newton: x <- x + (a - x^2) / (2x)
        x = x + (a - x * x) / (x + x);
    return x;
}

// double overloads so the stepper can be templated on T in {double, MP<2>, MP<4>}
static inline double sqrt(double a) { return std::sqrt(a); }

template <class T> struct Limbs;
template <> struct Limbs<double> {
    static constexpr int n = 1;
    static double get(const double& v, int) { return v; }
    static double make(const double* p) { return p[0]; }
};
template <int N> struct Limbs<MP<N>> {
    static constexpr int n = N;
    static double get(const MP<N>& v, int k) { return v.x[k]; }
    static MP<N> make(const double* p) { MP<N> r; for (int k = 0; k < N; ++k) r.x[k] = p[k]; return r; }
};

// Round a quad-double to T (leading limbs of a normalised expansion).
template <class T> static inline T narrow(const MP<4>& q) {
    double l[4];
    Acc<16> acc;
    for (int k = 3; k >= 0; --k) acc.add(q.x[k]);
    acc.template round_to<Limbs<T>::n>(l);
    return Limbs<T>::make(l);
}

}  // namespace orc
