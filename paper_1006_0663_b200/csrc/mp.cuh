// Device (and host-compilable) multiprecision arithmetic layer of the CUDA path: fp64, double-double
// (L = 2, the paper's "quadruple") and quad-double (L = 4, "octal").
// Written from the definitions of the error-free transformations (TwoSum: Knuth/Moller; FastTwoSum:
// Dekker; TwoProd by FMA); it shares no code with oracle/.  Design choices for sm_100a:
//   * every EFT is spelt with __dadd_rn/__dmul_rn/__fma_rn so nvcc can neither contract nor
//     reassociate it (nvcc's default -fmad=true stays on for the fp64 kernel);
//   * all operations are BRANCH-FREE (the paper blames the QD library's branching and irregular memory
//     access for its 1x "quadruple" result on Tesla): renormalisation is a fixed
//     sequence of TwoSum / FastTwoSum passes without zero tests;
//   * limbs live in registers as x[0] (leading) .. x[L-1]; in memory every limb is its own plane.
// Accuracy contract (checked by tests/test_device_arith.py against exact rationals): add/sub/mul
// relative error <= 4 * 2^-104 (dd) and <= 16 * 2^-205 (qd) measured against max(|a|,|b|) for
// add/sub ("sloppy" sense under cancellation) and against |ab| for mul; div/sqrt a few units more.
#pragma once
#include <cmath>

#if defined(__CUDACC__)
#define MPX __host__ __device__ __forceinline__
#else
#define MPX inline
#endif

namespace tk {

MPX double dadd(double a, double b) {
#ifdef __CUDA_ARCH__
    return __dadd_rn(a, b);
#else
    return a + b;
#endif
}
MPX double dsub(double a, double b) {
#ifdef __CUDA_ARCH__
    return __dadd_rn(a, -b);
#else
    return a - b;
#endif
}
MPX double dmul(double a, double b) {
#ifdef __CUDA_ARCH__
    return __dmul_rn(a, b);
#else
    return a * b;
#endif
}
MPX double dfma(double a, double b, double c) {
#ifdef __CUDA_ARCH__
    return __fma_rn(a, b, c);
#else
    return std::fma(a, b, c);
#endif
}

// s + e = a + b exactly, s = fl(a + b); no ordering assumption (6 flops)
MPX void two_sum(double a, double b, double& s, double& e) {
    s = dadd(a, b);
    double bb = dsub(s, a);
    e = dadd(dsub(a, dsub(s, bb)), dsub(b, bb));
}
// same, valid when |a| >= |b| or a == 0 (3 flops)
MPX void fast_two_sum(double a, double b, double& s, double& e) {
    s = dadd(a, b);
    e = dsub(b, dsub(s, a));
}
// p + e = a * b exactly
MPX void two_prod(double a, double b, double& p, double& e) {
    p = dmul(a, b);
    e = dfma(a, b, -p);
}
// a + b + c -> (a, b, c) with a = leading sum, b, c the first- and second-order errors (exact)
MPX void three_sum(double& a, double& b, double& c) {
    double t1, t2, t3;
    two_sum(a, b, t1, t2);
    two_sum(c, t1, a, t3);
    two_sum(t2, t3, b, c);
}
// a + b + c -> (a, b): second-order error dropped
MPX void three_sum2(double& a, double& b, double c) {
    double t1, t2, t3;
    two_sum(a, b, t1, t2);
    two_sum(c, t1, a, t3);
    b = dadd(t2, t3);
}

template <int L> struct Real { double x[L]; };
typedef Real<1> R1;
typedef Real<2> R2;
typedef Real<4> R4;

template <int L> MPX Real<L> from_double(double d) {
    Real<L> r;
    r.x[0] = d;
#pragma unroll
    for (int k = 1; k < L; ++k) r.x[k] = 0.0;
    return r;
}
template <int L> MPX Real<L> neg(const Real<L>& a) {
    Real<L> r;
#pragma unroll
    for (int k = 0; k < L; ++k) r.x[k] = -a.x[k];
    return r;
}
// exact scaling by a power of two (no overflow/underflow checks)
template <int L> MPX Real<L> scale2(const Real<L>& a, double p2) {
    Real<L> r;
#pragma unroll
    for (int k = 0; k < L; ++k) r.x[k] = dmul(a.x[k], p2);
    return r;
}

// ------------------------------------------------------------------------------------- fp64
MPX R1 add(const R1& a, const R1& b) { R1 r; r.x[0] = a.x[0] + b.x[0]; return r; }
MPX R1 sub(const R1& a, const R1& b) { R1 r; r.x[0] = a.x[0] - b.x[0]; return r; }
MPX R1 mul(const R1& a, const R1& b) { R1 r; r.x[0] = a.x[0] * b.x[0]; return r; }
MPX R1 mul_d(const R1& a, double d) { R1 r; r.x[0] = a.x[0] * d; return r; }
MPX R1 div(const R1& a, const R1& b) { R1 r; r.x[0] = a.x[0] / b.x[0]; return r; }

// ------------------------------------------------------------------------------------- dd
MPX R2 add(const R2& a, const R2& b) {
    // TwoSum of the heads, tails added in plain fp64, one FastTwoSum: 11 flops.  Absolute error
    // <= 2^-105 (|a| + |b|) (the "sloppy" contract: relative to the operands, not to a cancelled sum).
    double s, e;
    two_sum(a.x[0], b.x[0], s, e);
    e = dadd(e, dadd(a.x[1], b.x[1]));
    R2 r;
    fast_two_sum(s, e, r.x[0], r.x[1]);
    return r;
}
MPX R2 sub(const R2& a, const R2& b) { return add(a, neg(b)); }
MPX R2 mul(const R2& a, const R2& b) {
    double p, e;
    two_prod(a.x[0], b.x[0], p, e);
    e = dfma(a.x[0], b.x[1], e);
    e = dfma(a.x[1], b.x[0], e);
    R2 r;
    fast_two_sum(p, e, r.x[0], r.x[1]);
    return r;
}
MPX R2 mul_d(const R2& a, double d) {
    double p, e;
    two_prod(a.x[0], d, p, e);
    e = dfma(a.x[1], d, e);
    R2 r;
    fast_two_sum(p, e, r.x[0], r.x[1]);
    return r;
}
MPX R2 div(const R2& a, const R2& b) {
    // three quotient digits, remainder updated in dd
    double q0 = a.x[0] / b.x[0];
    R2 r = sub(a, mul_d(b, q0));
    double q1 = r.x[0] / b.x[0];
    r = sub(r, mul_d(b, q1));
    double q2 = r.x[0] / b.x[0];
    R2 q;
    fast_two_sum(q0, q1, q.x[0], q.x[1]);
    R2 t = from_double<2>(q2);
    return add(q, t);
}

// ------------------------------------------------------------------------------------- qd
// Renormalisation of five components into four limbs; two fixed, branch-free sequences:
//  * renorm5: no ordering assumption (sums may have cancelled): an error-free bottom-up TwoSum pass, then
//    one top-down TwoSum pass; the result is exact up to the single rounded add at the end and its limbs
//    are ulp-non-overlapping (|x[k+1]| <= ulp(x[k])), which is all the other operations assume;
//  * renorm4_ordered: for products, whose components are ordered by construction (|c[k+1]| <~ eps |c[k]|):
//    FastTwoSum passes (3 flops each, half the dependency depth).
MPX R4 renorm5(double c0, double c1, double c2, double c3, double c4) {
    double s, e, t0, t1, t2, t3, t4;
    two_sum(c3, c4, s, t4);
    two_sum(c2, s, s, t3);
    two_sum(c1, s, s, t2);
    two_sum(c0, s, t0, t1);
    R4 r;
    r.x[0] = t0;
    two_sum(t1, t2, r.x[1], e);
    two_sum(e, t3, r.x[2], e);
    r.x[3] = dadd(e, t4);
    return r;
}
MPX R4 renorm4_ordered(double c0, double c1, double c2, double c3) {
    double s, e, t1, t2, t3;
    fast_two_sum(c2, c3, s, t3);
    fast_two_sum(c1, s, s, t2);
    R4 r;
    fast_two_sum(c0, s, r.x[0], t1);
    fast_two_sum(t1, t2, r.x[1], e);
    fast_two_sum(e, t3, r.x[2], r.x[3]);
    return r;
}

MPX R4 add(const R4& a, const R4& b) {
    // limb-wise TwoSum, then each order collects the errors of the order above it
    double s0, s1, s2, s3, e0, e1, e2, e3;
    two_sum(a.x[0], b.x[0], s0, e0);
    two_sum(a.x[1], b.x[1], s1, e1);
    two_sum(a.x[2], b.x[2], s2, e2);
    two_sum(a.x[3], b.x[3], s3, e3);
    two_sum(s1, e0, s1, e0);              // order 1; e0 is now of order 2
    three_sum(s2, e1, e0);                // order 2; e1 (order 3), e0 (order 4)
    three_sum2(s3, e2, e1);               // order 3; e2 (order 4)
    double t4 = dadd(dadd(e3, e0), e2);   // order 4
    return renorm5(s0, s1, s2, s3, t4);
}
MPX R4 sub(const R4& a, const R4& b) { return add(a, neg(b)); }

MPX R4 mul(const R4& a, const R4& b) {
    // partial products a_i b_j: exact (TwoProd) for i + j <= 2, rounded for i + j == 3, dropped beyond
    double p0, q0, p1, q1, p2, q2, p3, q3, p4, q4, p5, q5;
    two_prod(a.x[0], b.x[0], p0, q0);
    two_prod(a.x[0], b.x[1], p1, q1);
    two_prod(a.x[1], b.x[0], p2, q2);
    two_prod(a.x[0], b.x[2], p3, q3);
    two_prod(a.x[1], b.x[1], p4, q4);
    two_prod(a.x[2], b.x[0], p5, q5);
    // order 1: q0 + p1 + p2
    three_sum(p1, p2, q0);                // p1 (order 1), p2 (order 2), q0 (order 3)
    // order 2: p2 + q1 + q2 + p3 + p4 + p5, errors go to order 3
    double s2, e1, e2, e3, e4, e5;
    two_sum(p2, q1, s2, e1);
    two_sum(s2, q2, s2, e2);
    two_sum(s2, p3, s2, e3);
    two_sum(s2, p4, s2, e4);
    two_sum(s2, p5, s2, e5);
    // order 3: rounded products and every error collected so far
    double s3 = dmul(a.x[0], b.x[3]);
    s3 = dfma(a.x[1], b.x[2], s3);
    s3 = dfma(a.x[2], b.x[1], s3);
    s3 = dfma(a.x[3], b.x[0], s3);
    double t = dadd(dadd(q3, q4), dadd(q5, q0));
    double v = dadd(dadd(e1, e2), dadd(e3, dadd(e4, e5)));
    s3 = dadd(s3, dadd(t, v));
    return renorm4_ordered(p0, p1, s2, s3);
}

MPX R4 mul_d(const R4& a, double d) {
    double p0, q0, p1, q1, p2, q2;
    two_prod(a.x[0], d, p0, q0);
    two_prod(a.x[1], d, p1, q1);
    two_prod(a.x[2], d, p2, q2);
    double p3 = dmul(a.x[3], d);
    two_sum(q0, p1, p1, q0);              // order 1; q0 order 2
    three_sum(p2, q1, q0);                // order 2; q1 order 3, q0 order 4
    p3 = dadd(dadd(p3, q2), dadd(q1, q0));
    return renorm4_ordered(p0, p1, p2, p3);
}

MPX R4 div(const R4& a, const R4& b) {
    // long division, five quotient digits, remainder kept in qd
    double q0 = a.x[0] / b.x[0];
    R4 r = sub(a, mul_d(b, q0));
    double q1 = r.x[0] / b.x[0];
    r = sub(r, mul_d(b, q1));
    double q2 = r.x[0] / b.x[0];
    r = sub(r, mul_d(b, q2));
    double q3 = r.x[0] / b.x[0];
    r = sub(r, mul_d(b, q3));
    double q4 = r.x[0] / b.x[0];
    return renorm5(q0, q1, q2, q3, q4);
}

template <int L> MPX Real<L> msqrt(const Real<L>& a) {
    if (a.x[0] <= 0.0) return from_double<L>(0.0);
    Real<L> x = from_double<L>(sqrt(a.x[0]));
#pragma unroll 1
    for (int it = 0; it < (L == 1 ? 0 : (L == 2 ? 2 : 3)); ++it) {     // Newton: x <- (x + a/x)/2
        x = scale2(add(x, div(a, x)), 0.5);
    }
    return x;
}

// narrow a quad-double to L limbs (leading limbs of a renormalised expansion)
template <int L> MPX Real<L> narrow(const R4& q) {
    Real<L> r;
#pragma unroll
    for (int k = 0; k < L; ++k) r.x[k] = q.x[k];
    return r;
}
template <int L> MPX R4 widen(const Real<L>& a) {
    R4 r;
#pragma unroll
    for (int k = 0; k < 4; ++k) r.x[k] = k < L ? a.x[k] : 0.0;
    return r;
}

}  // namespace tk
