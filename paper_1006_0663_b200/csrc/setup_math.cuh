// Quad-double elementary functions needed ONLY by the time-independent setup (teuk_create):
// exp, log (for inverting the tortoise coordinate, Eq. (2)), sin, cos (theta tables),
// and the constants pi and ln 2 computed from series in quad-double itself (no hard-coded digits).
// Host and device; accuracy ~1e-62 relative (checked against mpmath in tests/test_device_arith.py).
#pragma once
#include "mp.cuh"

namespace tk {

MPX R4 q_from_int(long v) { return from_double<4>((double)v); }
MPX R4 q_div_int(const R4& a, long v) { return div(a, from_double<4>((double)v)); }

struct QConst {
    R4 pi, ln2;
};

// atanh(1/n)-type and atan(1/n) series: sum_k sgn^k / ((2k+1) n^(2k+1))
MPX R4 q_inv_series(long n, bool alternating) {
    R4 n2 = q_from_int(n * n);
    R4 pw = div(from_double<4>(1.0), q_from_int(n));          // 1/n^(2k+1)
    R4 sum = pw;
    for (int k = 1; k < 160; ++k) {
        pw = div(pw, n2);
        R4 term = q_div_int(pw, 2 * k + 1);
        if (alternating && (k & 1)) term = neg(term);
        sum = add(sum, term);
        if (fabs(term.x[0]) < 1e-75 * fabs(sum.x[0])) break;
    }
    return sum;
}

inline QConst q_constants() {
    QConst c;
    // Machin: pi = 16 atan(1/5) - 4 atan(1/239);  ln 2 = 2 atanh(1/3)
    R4 a5 = q_inv_series(5, true), a239 = q_inv_series(239, true);
    c.pi = sub(scale2(a5, 16.0), scale2(a239, 4.0));
    c.ln2 = scale2(q_inv_series(3, false), 2.0);
    return c;
}

// exp(x) for |x| < ~700: x = k ln2 + r, r scaled by 2^-9, Taylor for expm1, nine doublings
// (s <- 2s + s^2 keeps relative accuracy), then 2^k.
MPX R4 q_exp(const R4& x, const R4& ln2) {
    double kd = nearbyint(x.x[0] / ln2.x[0]);
    R4 r = sub(x, mul_d(ln2, kd));
    r = scale2(r, 1.0 / 512.0);
    R4 term = r, s = r;
    for (int n = 2; n < 30; ++n) {
        term = q_div_int(mul(term, r), n);
        s = add(s, term);
        if (fabs(term.x[0]) < 1e-72 * fabs(s.x[0]) || term.x[0] == 0.0) break;
    }
    for (int i = 0; i < 9; ++i) s = add(scale2(s, 2.0), mul(s, s));
    R4 e = add(s, from_double<4>(1.0));
    int k = (int)kd;
    // 2^k in two factors so that subnormal-range results do not overflow the scale factor
    int k1 = k / 2, k2 = k - k1;
    return scale2(scale2(e, ldexp(1.0, k1)), ldexp(1.0, k2));
}

// log(x), x > 0: Newton on exp, y <- y + x exp(-y) - 1
MPX R4 q_log(const R4& x, const R4& ln2) {
    R4 y = from_double<4>(log(x.x[0]));
    for (int it = 0; it < 3; ++it) {
        R4 e = q_exp(neg(y), ln2);
        y = add(y, sub(mul(x, e), from_double<4>(1.0)));
    }
    return y;
}

// sin and cos for 0 <= x <= ~2 by their Taylor series (largest term ~ x^2/2: no harmful cancellation)
MPX void q_sincos(const R4& x, R4& sn, R4& cs) {
    R4 x2 = mul(x, x);
    R4 ts = x, tc = from_double<4>(1.0);
    sn = ts;
    cs = tc;
    for (int n = 1; n < 60; ++n) {
        tc = neg(q_div_int(mul(tc, x2), (long)(2 * n - 1) * (2 * n)));
        ts = neg(q_div_int(mul(ts, x2), (long)(2 * n) * (2 * n + 1)));
        cs = add(cs, tc);
        sn = add(sn, ts);
        if (fabs(tc.x[0]) < 1e-75 && fabs(ts.x[0]) < 1e-75) break;
    }
}

}  // namespace tk
