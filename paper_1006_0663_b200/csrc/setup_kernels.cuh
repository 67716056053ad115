// Time-independent setup on the device, all in quad-double:
//   radial_kernel : r(r*) at the 2 N_r - 1 integer and half points by Newton on Eq. (2) (PAPER.md:59,
//                   integration constant of DESIGN.md reading A3), unknown y = ln((r - r_+)/2M) so the
//                   horizon distance delta = r - r_+ (1e-11 .. 1e-101 at the inner edge) is exact.
//   coef_kernel   : b (Eqs. 6-7) and alpha, gamma, W, kappa of the source S
//                   (Eq. 12; derived from Eq. (1)) at every
//                   (r*, theta) point, folded with dt, dr*, dtheta (see step_kernel.cuh) and rounded to L limbs.
#pragma once
#include "mp.cuh"
#include "setup_math.cuh"

namespace tk {

struct SetupConsts {
    R4 M, a, rp, rpm;        // mass, spin, r_+, r_+ - r_-
    R4 cplus, cminus;        // 2 M r_+ / (r_+ - r_-), 2 M r_- / (r_+ - r_-)
    R4 rmin, dr, dth, ln2;
    R4 tau_h, tau_f;         // dt/2, dt
    int s, m, n_r, n_theta, pitch;
    long plane;
    int k0;                  // radial slab (NEXT-4): this handle's column 0 is global column k0/2; r*_k = rmin + (k0 + k) dr/2
};

MPX R4 q_tortoise(const SetupConsts& C, const R4& y, R4& delta_out, R4& r_out) {
    // r* = r + c_+ ln((r - r_+)/2M) - c_- ln((r - r_-)/2M),  delta = 2M e^y
    R4 delta = mul(scale2(C.M, 2.0), q_exp(y, C.ln2));
    R4 r = add(C.rp, delta);
    R4 arg = div(add(delta, C.rpm), scale2(C.M, 2.0));
    R4 rs = add(r, mul(C.cplus, y));
    rs = sub(rs, mul(C.cminus, q_log(arg, C.ln2)));
    delta_out = delta;
    r_out = r;
    return rs;
}

__global__ void radial_kernel(SetupConsts C, double* __restrict__ r_tab, double* __restrict__ d_tab) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= 2 * C.n_r - 1) return;
    // r*_k = r*_min + k dr*/2
    R4 rs = add(C.rmin, mul_d(scale2(C.dr, 0.5), (double)(k + C.k0)));
    // fp64 Newton for the starting value
    double M = C.M.x[0], rp = C.rp.x[0], rpm = C.rpm.x[0], cp = C.cplus.x[0], cm = C.cminus.x[0], a = C.a.x[0];
    double rsd = rs.x[0];
    double y = (rsd < rp) ? (rsd - rp) / cp : log(fmax(rsd, 2.0 * rp) / (2.0 * M));
    for (int it = 0; it < 100; ++it) {
        double d = 2.0 * M * exp(y), r = rp + d;
        double F = r + cp * y - cm * log((d + rpm) / (2.0 * M)) - rsd;
        double dF = (r * r + a * a) / (d + rpm);
        double st = F / dF;
        if (st > 5.0) st = 5.0;
        if (st < -5.0) st = -5.0;
        y -= st;
        if (fabs(st) < 1e-15 * fmax(1.0, fabs(y))) break;
    }
    // quad-double Newton (quadratic: 1e-15 -> 1e-30 -> 1e-60 -> below qd epsilon)
    R4 yq = from_double<4>(y), delta, r;
    for (int it = 0; it < 4; ++it) {
        R4 F = sub(q_tortoise(C, yq, delta, r), rs);
        R4 dF = div(add(mul(r, r), mul(C.a, C.a)), add(delta, C.rpm));
        yq = sub(yq, div(F, dF));
    }
    delta = mul(scale2(C.M, 2.0), q_exp(yq, C.ln2));
    r = add(C.rp, delta);
#pragma unroll
    for (int l = 0; l < 4; ++l) {
        r_tab[4 * k + l] = r.x[l];
        d_tab[4 * k + l] = delta.x[l];
    }
}

// 8 coefficients at one point, unfolded: b, alpha_R, alpha_I, gamma_R, gamma_I, W_R, W_I, kappa.
// Psi = e^{i m phi~} r^3 Phi (Eq. 4).
MPX void q_coefficients(const SetupConsts& C, const R4& r, const R4& dl, const R4& sn, const R4& cs, R4 out[8]) {
    const R4 M = C.M, a = C.a;
    const double s = (double)C.s, m = (double)C.m;
    R4 r2 = mul(r, r), a2 = mul(a, a);
    R4 R = add(r2, a2);
    R4 Dl = mul(dl, add(dl, C.rpm));
    R4 sn2 = mul(sn, sn);
    R4 Sig2 = sub(mul(R, R), mul(mul(a2, Dl), sn2));
    R4 Sig = msqrt(Sig2);
    R4 iS2 = div(from_double<4>(1.0), Sig2);
    R4 b = div(R, Sig);
    R4 rmM = sub(r, M);
    R4 rD = mul(r, Dl);
    // alpha = [2 s (r Delta - M (r^2 - a^2)) + i (4 m M a r + 2 s a Delta cos)] / Sigma^2
    R4 alR = mul(mul_d(sub(rD, mul(M, sub(r2, a2))), 2.0 * s), iS2);
    R4 alI = mul(add(mul_d(mul(mul(M, a), r), 4.0 * m), mul_d(mul(mul(a, Dl), cs), 2.0 * s)), iS2);
    // c = [2 r Delta + 2 s (r - M) R + i 2 m a R] / Sigma^2
    R4 cR = mul(add(scale2(rD, 2.0), mul_d(mul(rmM, R), 2.0 * s)), iS2);
    R4 cI = mul(mul_d(mul(a, R), 2.0 * m), iS2);
    // g = 3 Delta / (r R),  g_* = (Delta/R) 3 [2 (r-M) r R - Delta (3 r^2 + a^2)] / (r^2 R^2)
    R4 DoR = div(Dl, R);
    R4 g = mul_d(div(DoR, r), 3.0);
    R4 gnum = sub(mul(scale2(rmM, 2.0), mul(r, R)), mul(Dl, add(mul_d(r2, 3.0), a2)));
    R4 gst = mul_d(div(mul(DoR, gnum), mul(r2, mul(R, R))), 3.0);
    R4 b2 = mul(b, b);
    R4 beR = add(mul(scale2(b2, 2.0), g), cR);
    R4 kap = mul(Dl, iS2);
    R4 mc = add(from_double<4>(m), mul_d(cs, s));
    R4 VR = mul(kap, sub(div(mul(mc, mc), sn2), from_double<4>(s)));
    R4 VI = neg(mul(mul_d(mul(a, rmM), 4.0 * m * s), iS2));
    R4 WR = sub(sub(VR, mul(b2, add(gst, mul(g, g)))), mul(cR, g));
    R4 WI = sub(VI, mul(cI, g));
    // b_* = (Delta/R) a^2 sin^2 [R (r-M) - 2 r Delta] / Sigma^3
    R4 bst = div(mul(mul(DoR, mul(a2, sn2)), sub(mul(R, rmM), scale2(rD, 2.0))), mul(Sig2, Sig));
    R4 gaR = sub(add(mul(alR, b), beR), mul(b, bst));
    R4 gaI = add(mul(alI, b), cI);
    out[0] = b; out[1] = alR; out[2] = alI; out[3] = gaR; out[4] = gaI; out[5] = WR; out[6] = WI; out[7] = kap;
}

// grid: x over the radial points of ONE family (half == 0: integer points, N_r columns; half == 1: half
// points, N_r - 1 columns), y over theta.  fold == 0 writes the unfolded coefficients (test hook).
template <int L>
__global__ void coef_kernel(SetupConsts C, const double* __restrict__ r_tab, const double* __restrict__ d_tab,
                            const double* __restrict__ sin_tab, const double* __restrict__ cos_tab, int half, int fold,
                            double* __restrict__ out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    int cols = half ? C.n_r - 1 : C.n_r;
    if (i >= cols) return;
    int k = 2 * i + half;
    R4 r, dl, sn, cs;
#pragma unroll
    for (int l = 0; l < 4; ++l) {
        r.x[l] = r_tab[4 * k + l];
        dl.x[l] = d_tab[4 * k + l];
        sn.x[l] = sin_tab[4 * j + l];
        cs.x[l] = cos_tab[4 * j + l];
    }
    R4 c[8];
    q_coefficients(C, r, dl, sn, cs, c);
    if (fold) {
        R4 tau = half ? C.tau_h : C.tau_f;
        R4 tdr = div(tau, C.dr);
        R4 th2 = scale2(tau, 0.5);
        R4 tk = div(th2, mul(C.dth, C.dth));
        c[0] = mul(c[0], tdr);
        c[1] = mul(c[1], th2); c[2] = mul(c[2], th2);
        c[3] = mul(c[3], tdr); c[4] = mul(c[4], tdr);
        c[5] = mul(c[5], th2); c[6] = mul(c[6], th2);
        c[7] = mul(c[7], tk);
    }
    long idx = (long)j * C.pitch + i;
#pragma unroll
    for (int q = 0; q < 8; ++q)
#pragma unroll
        for (int l = 0; l < L; ++l) out[((long)q * L + l) * C.plane + idx] = c[q].x[l];
}

}  // namespace tk

namespace tk {

// ---------------------------------------------------------------------------------------------------------------
// Semi-recompute coefficient supply (variant (b); fp64 only).  Every coefficient of §3 is
// q^k x (function of r) x (function of theta) with q = 1/Sigma^2, so instead of 16 two-dimensional planes the step
// kernel reads ONE plane per point family (isig = 1/Sigma) plus 16 one-dimensional r-tables and 3 theta-tables:
//   c0 = T0 isig                      c1 = T1 q                     c2 = (T2a + T2b cos) q
//   c3 = q (T3a isig + T3b - q sin^2 T3c)                           c4 = q ((T4a + T4b cos) isig + T4c)
//   c5 = q (T5a Tth + T5b)            c6 = q T6                     c7 = q T7,          q = isig^2,
// Tth = (m + s cos)^2 / sin^2 - s.  HBM traffic: 64 B of state + 16 B of isig per update instead of 192 B.
// Table order in memory: R-family f (0: integer points, tau = dt; 1: half points, tau = dt/2), table t = 0..15:
//   T0 T1 T2a T2b T3a T3b T3c T4a T4b T4c T5a T5b T6 T7 (14 used, 2 spare), each `pitch` doubles.
constexpr int RC_NT = 16;

__global__ void rtab_kernel(SetupConsts C, const double* __restrict__ r_tab, const double* __restrict__ d_tab,
                            double* __restrict__ rt) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= 2 * C.n_r - 1) return;
    const int fam = k & 1, col = k >> 1;
    R4 r, dl;
#pragma unroll
    for (int l = 0; l < 4; ++l) { r.x[l] = r_tab[4 * k + l]; dl.x[l] = d_tab[4 * k + l]; }
    const R4 M = C.M, a = C.a;
    const double s = (double)C.s, m = (double)C.m;
    R4 r2 = mul(r, r), a2 = mul(a, a);
    R4 R = add(r2, a2);
    R4 Dl = mul(dl, add(dl, C.rpm));
    R4 rmM = sub(r, M), rD = mul(r, Dl);
    R4 AR = mul_d(sub(rD, mul(M, sub(r2, a2))), 2.0 * s);
    R4 AI0 = mul_d(mul(mul(M, a), r), 4.0 * m);
    R4 AI1 = mul_d(mul(a, Dl), 2.0 * s);
    R4 CR = add(scale2(rD, 2.0), mul_d(mul(rmM, R), 2.0 * s));
    R4 CI = mul_d(mul(a, R), 2.0 * m);
    R4 DoR = div(Dl, R);
    R4 g = mul_d(div(DoR, r), 3.0);
    R4 gnum = sub(mul(scale2(rmM, 2.0), mul(r, R)), mul(Dl, add(mul_d(r2, 3.0), a2)));
    R4 RR = mul(R, R);
    R4 gst = mul_d(div(mul(DoR, gnum), mul(r2, RR)), 3.0);
    R4 BR = add(mul(scale2(RR, 2.0), g), CR);
    R4 BB = mul(mul(a2, Dl), sub(mul(R, rmM), scale2(rD, 2.0)));
    R4 WR0 = neg(add(mul(RR, add(gst, mul(g, g))), mul(CR, g)));
    R4 WIr = neg(add(mul_d(mul(a, rmM), 4.0 * m * s), mul(CI, g)));
    R4 tau = fam ? C.tau_h : C.tau_f;
    R4 tdr = div(tau, C.dr), th2 = scale2(tau, 0.5);
    R4 tk = div(th2, mul(C.dth, C.dth));
    R4 T[RC_NT];
    T[0] = mul(tdr, R);
    T[1] = mul(th2, AR);
    T[2] = mul(th2, AI0);
    T[3] = mul(th2, AI1);
    T[4] = mul(tdr, mul(AR, R));
    T[5] = mul(tdr, BR);
    T[6] = mul(tdr, BB);
    T[7] = mul(tdr, mul(AI0, R));
    T[8] = mul(tdr, mul(AI1, R));
    T[9] = mul(tdr, CI);
    T[10] = mul(th2, Dl);
    T[11] = mul(th2, WR0);
    T[12] = mul(th2, WIr);
    T[13] = mul(tk, Dl);
    T[14] = RR;                       // spare slots keep R^2 and a^2 Delta (used by isig_kernel's checks / debugging)
    T[15] = mul(a2, Dl);
#pragma unroll
    for (int t = 0; t < RC_NT; ++t) rt[((long)fam * RC_NT + t) * C.pitch + col] = T[t].x[0];
}

// isig = 1/Sigma at every point of both families, evaluated in quad-double, rounded to fp64.
__global__ void isig_kernel(SetupConsts C, const double* __restrict__ r_tab, const double* __restrict__ d_tab,
                            const double* __restrict__ sin_tab, int half, double* __restrict__ out) {
    int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    int cols = half ? C.n_r - 1 : C.n_r;
    if (i >= cols) return;
    int k = 2 * i + half;
    R4 r, dl, sn;
#pragma unroll
    for (int l = 0; l < 4; ++l) { r.x[l] = r_tab[4 * k + l]; dl.x[l] = d_tab[4 * k + l]; sn.x[l] = sin_tab[4 * j + l]; }
    R4 a2 = mul(C.a, C.a);
    R4 R = add(mul(r, r), a2);
    R4 Dl = mul(dl, add(dl, C.rpm));
    R4 Sig2 = sub(mul(R, R), mul(mul(a2, Dl), mul(sn, sn)));
    R4 is = div(from_double<4>(1.0), msqrt(Sig2));
    out[(long)j * C.pitch + i] = is.x[0];
}

}  // namespace tk
