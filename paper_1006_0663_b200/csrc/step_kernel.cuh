// Fused Lax-Wendroff step kernel: half step Eq. (13) + full step Eq. (14), radial
// Dirichlet rows and polar parity ghosts and the observer node extraction
// in ONE launch per iteration; the intermediate u^{n+1/2}_{i+1/2} lives only in shared
// memory.  Templated on the limb count L (1 fp64, 2 double-double, 4 quad-double).
//
// Folded coefficient planes (built once by setup_coefficients, tau = dt/2 for the half step and dt
// for the full step; everything a product of time-independent factors):
//   c0 = tau b / dr*            c1,c2 = tau alpha / 2        c3,c4 = tau gamma / dr*
//   c5,c6 = tau W / 2           c7 = tau kappa / (2 dtheta^2)
// and the 1-D table cj[j] = cot(theta_j) dtheta / 2.  With sig = u_hi + u_lo, del = u_hi - u_lo
// (the two radial neighbours) and Lam = ((sig+ + sig-) - 2 sig) + cj (sig+ - sig-) over theta:
//   new_Phi = base_Phi - c0 del_Phi + (tau/2) sig_Pi
//   new_Pi  = base_Pi  + c0 del_Pi  + [ -(c1 + i c2) sig_Pi + (c3 + i c4) del_Phi + c7 Lam - (c5 + i c6) sig_Phi ]
// base = sig/2 for the half step, u^n for the full step.  Multiplications by 1/2 and 2 are exact.
#pragma once
#include <cstdint>
#include "mp.cuh"

namespace tk {

struct StepParams {
    const double* u_in;      // [4][L] planes of n_theta x pitch
    double* u_out;
    const double* coef_i;    // [8][L] planes, integer points (full step)
    const double* coef_h;    // [8][L] planes, half points (column i <-> i + 1/2)
    const double* cj;        // [L][n_theta]
    int n_r, n_theta, pitch;
    long plane;              // n_theta * pitch
    int ti, tj;              // output tile
    double sigma;            // +1 even |m|, -1 odd |m|
    double tq_half, tq_full; // tau/2 = dt/4, dt/2
    double* obs_raw;         // [cap][4 nodes][4][L] or null
    const long* step_base;
    long obs_cap;
    int step_off;
    int oi, oj;              // lower-left observer node
};

// 8-byte asynchronous global -> shared copy; ok = false copies nothing and writes zeros (src-size 0), so lanes whose
// column lies outside the grid take the same instruction as everyone else
__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc, bool ok) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gsrc),
                 "r"(ok ? 8 : 0)
                 : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int L> struct Ld {
    static __device__ __forceinline__ Real<L> g(const double* __restrict__ p, long stride, long idx) {
        Real<L> r;
#pragma unroll
        for (int l = 0; l < L; ++l) r.x[l] = __ldg(p + l * stride + idx);
        return r;
    }
    static __device__ __forceinline__ Real<L> s(const double* p, int stride, int idx) {
        Real<L> r;
#pragma unroll
        for (int l = 0; l < L; ++l) r.x[l] = p[l * stride + idx];
        return r;
    }
    static __device__ __forceinline__ void st(double* p, long stride, long idx, const Real<L>& v) {
#pragma unroll
        for (int l = 0; l < L; ++l) p[l * stride + idx] = v.x[l];
    }
};

template <int L> __device__ __forceinline__ Real<L> sgn(const Real<L>& a, double s) {
    Real<L> r;
#pragma unroll
    for (int l = 0; l < L; ++l) r.x[l] = a.x[l] * s;     // s = +-1: exact
    return r;
}

// One sub-step at one point.  T: tile accessor giving Real<L> at (component, row offset, column).
// lo/hi are the two radial neighbour columns in the tile; rows jm/jp are the theta neighbours
// (already mirrored) with signs sm/sp.
template <int L> struct GlobalCoef {       // coefficient q straight from the global planes (coalesced, read-only path)
    const double* __restrict__ p;
    long stride, idx;
    __device__ __forceinline__ Real<L> get(int q) const { return Ld<L>::g(p + (long)q * L * stride, stride, idx); }
};

// Weights of the wide (10th-order) theta stencils as quad-double limbs; narrowed to L in the kernel.
struct ThetaWeights {
    double wd[6][4];     // second derivative, k = 0..5 (units 1/dtheta^2)
    double wc[5][4];     // first derivative, k = 1..5 (units 1/dtheta)
};

template <int L, class Tile, class Coef>
__device__ __forceinline__ void substep_core(const Real<L> sg[4], const Real<L> dl[4], const Real<L> lam[2], const Coef& cf,
                                             double tq, bool half, const Real<L> base_in[4], Real<L> out[4]);

// stencil half-width 1: Lam = ((sig+ + sig-) - 2 sig) + cj (sig+ - sig-)
template <int L, class Tile, class Coef>
__device__ __forceinline__ void substep(const Tile& t, int row, int rm, int rp, double sm, double sp, int clo, int chi,
                                        const Coef& cf, const Real<L>& cjv,
                                        double tq, bool half, const Real<L> base_in[4], Real<L> out[4]) {
    Real<L> sg[4], dl[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        Real<L> lo = t.get(c, row, clo), hi = t.get(c, row, chi);
        sg[c] = add(hi, lo);
        dl[c] = sub(hi, lo);
    }
    // angular operator on sig_Phi (components 0, 1)
    Real<L> lam[2];
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        Real<L> up = sgn(add(t.get(c, rp, chi), t.get(c, rp, clo)), sp);
        Real<L> dn = sgn(add(t.get(c, rm, chi), t.get(c, rm, clo)), sm);
        Real<L> second = sub(add(up, dn), scale2(sg[c], 2.0));
        Real<L> first = mul(cjv, sub(up, dn));
        lam[c] = add(second, first);
    }
    substep_core<L, Tile, Coef>(sg, dl, lam, cf, tq, half, base_in, out);
}

// stencil half-width 5 (10th order):  Lam = d0 sig + sum_k d_k (sig_{+k} + sig_{-k}) + 2 cj sum_k c_k (sig_{+k} - sig_{-k}),
// ghost rows mirrored about the axis with sign sigma (f_{-k} = sigma f_{k-1}, f_{N-1+k} = sigma f_{N-k}).
// The tile must hold every theta row (column kernel below).
template <int L, class Tile, class STile, class Coef>
__device__ __forceinline__ void substep_wide(const Tile& t, const STile& st, int scol, int row, int nt, double sigma, int clo,
                                             int chi, const Coef& cf, const Real<L>& cjv, const ThetaWeights& W, double tq,
                                             bool half, const Real<L> base_in[4], Real<L> out[4]) {
    // st: staged tile of sig_Phi = Phi_hi + Phi_lo (2 components) at every row, column scol <-> this point
    Real<L> sg[4], dl[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        Real<L> lo = t.get(c, row, clo), hi = t.get(c, row, chi);
        sg[c] = (c < 2) ? st.get(c, row, scol) : add(hi, lo);
        dl[c] = sub(hi, lo);
    }
    Real<L> lam[2];
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        Real<L> w0;
#pragma unroll
        for (int l = 0; l < L; ++l) w0.x[l] = W.wd[0][l];
        Real<L> s2 = mul(w0, sg[c]);
        Real<L> s1 = from_double<L>(0.0);
        if (L == 1 && row >= 5 && row + 5 < nt) {
            // fp64 (instruction-bound): rows away from the axis need no mirroring -> straight-line unrolled code;
            // dd/qd (FP64-pipe bound) keep the single compact loop (the extra code path cost them registers)
#pragma unroll
            for (int k = 1; k <= 5; ++k) {
                Real<L> up = st.get(c, row + k, scol);
                Real<L> dn = st.get(c, row - k, scol);
                Real<L> wd, wc;
#pragma unroll
                for (int l = 0; l < L; ++l) { wd.x[l] = W.wd[k][l]; wc.x[l] = W.wc[k - 1][l]; }
                s2 = add(s2, mul(wd, add(up, dn)));
                s1 = add(s1, mul(wc, sub(up, dn)));
            }
        } else {
#pragma unroll 1
            for (int k = 1; k <= 5; ++k) {
                int ru = row + k, rd = row - k;
                double su = 1.0, sd = 1.0;
                if (ru >= nt) { ru = 2 * nt - 1 - ru; su = sigma; }
                if (rd < 0) { rd = -rd - 1; sd = sigma; }
                Real<L> up = sgn(st.get(c, ru, scol), su);
                Real<L> dn = sgn(st.get(c, rd, scol), sd);
                Real<L> wd, wc;
#pragma unroll
                for (int l = 0; l < L; ++l) { wd.x[l] = W.wd[k][l]; wc.x[l] = W.wc[k - 1][l]; }
                s2 = add(s2, mul(wd, add(up, dn)));
                s1 = add(s1, mul(wc, sub(up, dn)));
            }
        }
        lam[c] = add(s2, mul(cjv, scale2(s1, 2.0)));
    }
    substep_core<L, Tile, Coef>(sg, dl, lam, cf, tq, half, base_in, out);
}

template <int L, class Tile, class Coef>
__device__ __forceinline__ void substep_core(const Real<L> sg[4], const Real<L> dl[4], const Real<L> lam[2], const Coef& cf,
                                             double tq, bool half, const Real<L> base_in[4], Real<L> out[4]) {
    Real<L> c0 = cf.get(0);
    Real<L> c1 = cf.get(1);
    Real<L> c2 = cf.get(2);
    Real<L> c3 = cf.get(3);
    Real<L> c4 = cf.get(4);
    Real<L> c5 = cf.get(5);
    Real<L> c6 = cf.get(6);
    Real<L> c7 = cf.get(7);
    // tau * S_Pi, summed in the printed order of S: -alpha Pi + gamma Phi_* + kappa Lam - W Phi
    Real<L> sR = neg(sub(mul(c1, sg[2]), mul(c2, sg[3])));
    Real<L> sI = neg(add(mul(c1, sg[3]), mul(c2, sg[2])));
    sR = add(sR, sub(mul(c3, dl[0]), mul(c4, dl[1])));
    sI = add(sI, add(mul(c3, dl[1]), mul(c4, dl[0])));
    sR = add(sR, mul(c7, lam[0]));
    sI = add(sI, mul(c7, lam[1]));
    sR = sub(sR, sub(mul(c5, sg[0]), mul(c6, sg[1])));
    sI = sub(sI, add(mul(c5, sg[1]), mul(c6, sg[0])));
    Real<L> b0, b1, b2, b3;
    if (half) {
        b0 = scale2(sg[0], 0.5); b1 = scale2(sg[1], 0.5); b2 = scale2(sg[2], 0.5); b3 = scale2(sg[3], 0.5);
    } else {
        b0 = base_in[0]; b1 = base_in[1]; b2 = base_in[2]; b3 = base_in[3];
    }
    out[0] = add(sub(b0, mul(c0, dl[0])), mul_d(sg[2], tq));
    out[1] = add(sub(b1, mul(c0, dl[1])), mul_d(sg[3], tq));
    out[2] = add(add(b2, mul(c0, dl[2])), sR);
    out[3] = add(add(b3, mul(c0, dl[3])), sI);
}

template <int L> struct SmemTile {
    const double* p;
    int rows, cols, row0;       // row0 = global row of tile row 0
    __device__ __forceinline__ Real<L> get(int c, int grow, int col) const {
        return Ld<L>::s(p + (c * L) * rows * cols, rows * cols, (grow - row0) * cols + col);
    }
};

template <int L> struct RegCoef {          // the 8 coefficients of one point, register resident
    Real<L> c[8];
    __device__ __forceinline__ const Real<L>& get(int q) const { return c[q]; }
};
template <int L>
__device__ __forceinline__ void load_coef(RegCoef<L>& rc, const double* __restrict__ p, long stride, long idx) {
#pragma unroll
    for (int q = 0; q < 8; ++q) rc.c[q] = Ld<L>::g(p + (long)q * L * stride, stride, idx);
}

// Generic fused step kernel (all precisions; the default for dd and qd).
//  * TI_/TJ_ > 0: compile-time tile (index arithmetic folds to constants); 0: run-time tile from P.ti/P.tj.
//  * MAXT/MINB: launch bounds (register budget = 65536 / (MAXT * MINB)); the qd kernel is latency-bound at
//    1 block x 8 warps, so shapes trading registers for resident warps are instantiated and selectable.
//  * L <= 2: the coefficients of a thread's NEXT point are fetched into registers while it computes the current
//    one, and the first set of each phase is requested before the preceding barrier (ncu on the first dd
//    kernel: 48 % of stall cycles were long-scoreboard waits on exactly these loads).  qd has no registers to
//    spare for that and is FP64-pipe bound anyway.
template <int L, int TI_ = 0, int TJ_ = 0, int MAXT = 256, int MINB = 1>
__global__ void __launch_bounds__(MAXT, MINB) step_kernel(StepParams P) {
    extern __shared__ double smem[];
    const int TI = TI_ ? TI_ : P.ti, TJ = TJ_ ? TJ_ : P.tj;
    const int UC = TI + 2, UR = TJ + 4, HC = TI + 1, HR = TJ + 2;
    double* us = smem;                       // [4L][UR][UC]
    double* hs = smem + 4 * L * UR * UC;     // [4L][HR][HC]
    const int i0 = blockIdx.x * TI, j0 = blockIdx.y * TJ;
    const int iu0 = i0 - 1, ju0 = j0 - 2, jh0 = j0 - 1;
    const int nt = P.n_theta, nr = P.n_r;
    const int tid = threadIdx.x, nth = MAXT;
    constexpr bool PF = (L <= 2);

    // work item -> tile coordinates; returns whether the item exists and lies inside the grid
    auto item1 = [&](int idx, int& tc, int& tr, int& ih, int& jh) {
        tr = idx / HC; tc = idx - tr * HC;
        ih = iu0 + tc; jh = jh0 + tr;
        return idx < HR * HC && ih >= 0 && ih <= nr - 2 && jh >= 0 && jh < nt;
    };
    auto item2 = [&](int idx, int& tc, int& tr, int& i, int& j) {
        tr = idx / TI; tc = idx - tr * TI;
        i = i0 + tc; j = j0 + tr;
        return idx < TJ * TI && i < nr && j < nt;
    };

    RegCoef<L> cc;
    int idx = tid, tc, tr, gi, gj;
    bool v = item1(idx, tc, tr, gi, gj);
    if (PF && v) load_coef(cc, P.coef_h, P.plane, (long)gj * P.pitch + gi);

    // ---- phase 0: stage the u^n tile (+1 column, +2 rows of halo); outside the grid -> 0.
    //      8-byte cp.async with zero-fill: every element of the tile is in flight at once (ONE round trip to L2/HBM per
    //      block, no staging registers); the register-batched loop this replaces took ceil(n_stage / (8 nth)) = 3 (dd)
    //      or 4 (qd) dependent round trips, during which the block's warps left the FP64 pipe idle
    const int n_stage = 4 * L * UR * UC;
    for (int k = tid; k < n_stage; k += nth) {
        int c = k % UC, rest = k / UC;
        int r = rest % UR, pl = rest / UR;
        int ui = iu0 + c, uj = ju0 + r;
        bool ok = ui >= 0 && ui < nr && uj >= 0 && uj < nt;
        cp_async8(us + k, ok ? P.u_in + pl * P.plane + (long)uj * P.pitch + ui : P.u_in, ok);
    }
    cp_async_commit();
    cp_async_wait<0>();
    __syncthreads();

    SmemTile<L> ut{us, UR, UC, ju0};
    // ---- phase 1: half step, Eq. (13), at (ih + 1/2, jh) for the columns/rows the full step needs
    while (idx < HR * HC) {
        int nidx = idx + nth, ntc, ntr, ngi, ngj;
        bool nv = item1(nidx, ntc, ntr, ngi, ngj);
        RegCoef<L> cn;
        if (PF && nv) load_coef(cn, P.coef_h, P.plane, (long)ngj * P.pitch + ngi);
        if (v) {
            const int ih = gi, jh = gj;
            if (!PF) load_coef(cc, P.coef_h, P.plane, (long)jh * P.pitch + ih);
            int rm = jh - 1, rp = jh + 1;
            double sm = 1.0, sp = 1.0;
            if (rm < 0) { rm = 0; sm = P.sigma; }
            if (rp >= nt) { rp = nt - 1; sp = P.sigma; }
            Real<L> cjv = Ld<L>::g(P.cj, nt, jh);
            Real<L> out[4];
            substep<L>(ut, jh, rm, rp, sm, sp, tc, tc + 1, cc, cjv, P.tq_half, true, out, out);
#pragma unroll
            for (int c = 0; c < 4; ++c)
#pragma unroll
                for (int l = 0; l < L; ++l) hs[(c * L + l) * HR * HC + tr * HC + tc] = out[c].x[l];
        }
        if (PF) cc = cn;
        idx = nidx; tc = ntc; tr = ntr; gi = ngi; gj = ngj; v = nv;
    }
    // first full-step coefficient set: requested before the barrier
    idx = tid;
    v = item2(idx, tc, tr, gi, gj);
    bool interior = v && gi != 0 && gi != nr - 1;
    if (PF && interior) load_coef(cc, P.coef_i, P.plane, (long)gj * P.pitch + gi);
    __syncthreads();

    SmemTile<L> ht{hs, HR, HC, jh0};
    // ---- phase 2: full step, Eq. (14), + radial Dirichlet rows + observer nodes
    while (idx < TJ * TI) {
        int nidx = idx + nth, ntc, ntr, ngi, ngj;
        bool nv = item2(nidx, ntc, ntr, ngi, ngj);
        bool ninterior = nv && ngi != 0 && ngi != nr - 1;
        RegCoef<L> cn;
        if (PF && ninterior) load_coef(cn, P.coef_i, P.plane, (long)ngj * P.pitch + ngi);
        if (v) {
            const int i = gi, j = gj;
            Real<L> out[4];
            if (!interior) {
#pragma unroll
                for (int c = 0; c < 4; ++c) out[c] = from_double<L>(0.0);
            } else {
                if (!PF) load_coef(cc, P.coef_i, P.plane, (long)j * P.pitch + i);
                int rm = j - 1, rp = j + 1;
                double sm = 1.0, sp = 1.0;
                if (rm < 0) { rm = 0; sm = P.sigma; }
                if (rp >= nt) { rp = nt - 1; sp = P.sigma; }
                Real<L> base[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) base[c] = ut.get(c, j, tc + 1);
                Real<L> cjv = Ld<L>::g(P.cj, nt, j);
                // h columns: tile col tc <-> i - 1/2, tc + 1 <-> i + 1/2
                substep<L>(ht, j, rm, rp, sm, sp, tc, tc + 1, cc, cjv, P.tq_full, false, base, out);
            }
            long g = (long)j * P.pitch + i;
#pragma unroll
            for (int c = 0; c < 4; ++c) Ld<L>::st(P.u_out + (long)c * L * P.plane, P.plane, g, out[c]);
            if (P.obs_raw != nullptr) {
                int di = i - P.oi, dj = j - P.oj;
                if ((di == 0 || di == 1) && (dj == 0 || dj == 1)) {
                    long k = *P.step_base + P.step_off;
                    if (k < P.obs_cap) {
                        double* o = P.obs_raw + ((k * 4 + (dj * 2 + di)) * 4) * L;
#pragma unroll
                        for (int c = 0; c < 4; ++c)
#pragma unroll
                            for (int l = 0; l < L; ++l) o[c * L + l] = out[c].x[l];
                    }
                }
            }
        }
        if (PF) cc = cn;
        idx = nidx; tc = ntc; tr = ntr; gi = ngi; gj = ngj; v = nv; interior = ninterior;
    }
}


// ---------------------------------------------------------------------------------------------------------------
// Pair kernel (dd / qd): TWO threads per point.  Lanes 2k and 2k+1 of a warp own the real and the imaginary part of
// one point: lane part p computes Phi component p and Pi component 2+p.  Every sum / difference of the two radial
// neighbours is formed once, by the lane that owns the component, and the three the OTHER part needs (sig of the
// other Phi and Pi component, del of the other Phi component) travel by __shfl_xor, so the FP64 work per point is
// exactly step_kernel's, operation for operation (sub(a, b) = add(a, neg(b)) and the +-1 factors are exact: results
// are bitwise those of step_kernel).  Why: the straight-line qd sub-step is ~100 KB of code per phase and each warp
// walks it once per point - ncu attributes 24 % of the qd kernel's stall samples to instruction fetch ("no_instruction");
// here the body is half as long, each thread needs half the live values (more resident warps), and a warp covers 16
// points per pass of the code.  Compile-time tile only.
template <int L> __device__ __forceinline__ Real<L> partner(const Real<L>& a, unsigned mask) {
    Real<L> r;
#pragma unroll
    for (int l = 0; l < L; ++l) r.x[l] = __shfl_xor_sync(mask, a.x[l], 1);
    return r;
}

// tau * S_Pi and the two outputs of part p, in substep_core's order; sx = -1 (real part) / +1 (imaginary part) on the
// cross terms
template <int L>
__device__ __forceinline__ void pair_tail(const GlobalCoef<L>& g, double sx, const Real<L>& sgP, const Real<L>& sgQ,
                                          const Real<L>& sgPi, const Real<L>& sgQi, const Real<L>& dlP, const Real<L>& dlQ,
                                          const Real<L>& dlPi, const Real<L>& lam, double tq, bool half, const Real<L>& baseP,
                                          const Real<L>& basePi, Real<L>& outP, Real<L>& outPi) {
    Real<L> s = neg(add(mul(g.get(1), sgPi), sgn(mul(g.get(2), sgQi), sx)));
    s = add(s, add(mul(g.get(3), dlP), sgn(mul(g.get(4), dlQ), sx)));
    s = add(s, mul(g.get(7), lam));
    s = sub(s, add(mul(g.get(5), sgP), sgn(mul(g.get(6), sgQ), sx)));
    const Real<L> c0 = g.get(0);
    const Real<L> bP = half ? scale2(sgP, 0.5) : baseP;
    const Real<L> bPi = half ? scale2(sgPi, 0.5) : basePi;
    outP = add(sub(bP, mul(c0, dlP)), mul_d(sgPi, tq));
    outPi = add(add(bPi, mul(c0, dlPi)), s);
}

// one sub-step for part p of one point; t: tile accessor; cf/stride/idx: the point's 8 folded coefficients in global memory
template <int L, class Tile>
__device__ __forceinline__ void substep_pair(const Tile& t, int p, double sx, unsigned mask, int row, int rm, int rp, double sm,
                                             double sp, int clo, int chi, const double* __restrict__ cf, long stride, long idx,
                                             const Real<L>& cjv, double tq, bool half, const Real<L>& baseP, const Real<L>& basePi,
                                             Real<L>& outP, Real<L>& outPi) {
    const int cP = p, cPi = 2 + p;
    GlobalCoef<L> g{cf, stride, idx};
    Real<L> lo = t.get(cP, row, clo), hi = t.get(cP, row, chi);
    const Real<L> sgP = add(hi, lo), dlP = sub(hi, lo);
    lo = t.get(cPi, row, clo); hi = t.get(cPi, row, chi);
    const Real<L> sgPi = add(hi, lo), dlPi = sub(hi, lo);
    const Real<L> sgQ = partner(sgP, mask), dlQ = partner(dlP, mask), sgQi = partner(sgPi, mask);
    // angular operator on this part's sig_Phi
    const Real<L> up = sgn(add(t.get(cP, rp, chi), t.get(cP, rp, clo)), sp);
    const Real<L> dn = sgn(add(t.get(cP, rm, chi), t.get(cP, rm, clo)), sm);
    const Real<L> second = sub(add(up, dn), scale2(sgP, 2.0));
    const Real<L> first = mul(cjv, sub(up, dn));
    const Real<L> lam = add(second, first);
    pair_tail<L>(g, sx, sgP, sgQ, sgPi, sgQi, dlP, dlQ, dlPi, lam, tq, half, baseP, basePi, outP, outPi);
}

// stencil half-width 5 (substep_wide) for part p of one point; st: staged sig_Phi tile (both components, so the other
// part's sig_Phi is a shared-memory read, not a shuffle)
template <int L, class Tile, class STile>
__device__ __forceinline__ void substep_wide_pair(const Tile& t, const STile& st, int scol, int p, double sx, unsigned mask, int row,
                                                  int nt, double sigma, int clo, int chi, const double* __restrict__ cf,
                                                  long stride, long idx, const Real<L>& cjv, const ThetaWeights& W, double tq,
                                                  bool half, const Real<L>& baseP, const Real<L>& basePi, Real<L>& outP,
                                                  Real<L>& outPi) {
    const int cP = p, cPi = 2 + p;
    GlobalCoef<L> g{cf, stride, idx};
    const Real<L> sgP = st.get(cP, row, scol), sgQ = st.get(1 - p, row, scol);
    Real<L> lo = t.get(cP, row, clo), hi = t.get(cP, row, chi);
    const Real<L> dlP = sub(hi, lo);
    lo = t.get(cPi, row, clo); hi = t.get(cPi, row, chi);
    const Real<L> sgPi = add(hi, lo), dlPi = sub(hi, lo);
    const Real<L> dlQ = partner(dlP, mask), sgQi = partner(sgPi, mask);
    Real<L> w0;
#pragma unroll
    for (int l = 0; l < L; ++l) w0.x[l] = W.wd[0][l];
    Real<L> s2 = mul(w0, sgP);
    Real<L> s1 = from_double<L>(0.0);
#pragma unroll 1
    for (int k = 1; k <= 5; ++k) {
        int ru = row + k, rd = row - k;
        double su = 1.0, sd = 1.0;
        if (ru >= nt) { ru = 2 * nt - 1 - ru; su = sigma; }
        if (rd < 0) { rd = -rd - 1; sd = sigma; }
        Real<L> up = sgn(st.get(cP, ru, scol), su);
        Real<L> dn = sgn(st.get(cP, rd, scol), sd);
        Real<L> wd, wc;
#pragma unroll
        for (int l = 0; l < L; ++l) { wd.x[l] = W.wd[k][l]; wc.x[l] = W.wc[k - 1][l]; }
        s2 = add(s2, mul(wd, add(up, dn)));
        s1 = add(s1, mul(wc, sub(up, dn)));
    }
    const Real<L> lam = add(s2, mul(cjv, scale2(s1, 2.0)));
    pair_tail<L>(g, sx, sgP, sgQ, sgPi, sgQi, dlP, dlQ, dlPi, lam, tq, half, baseP, basePi, outP, outPi);
}

template <int L, int TI, int TJ, int NTHR, int MINB>
__global__ void __launch_bounds__(NTHR, MINB) step_kernel_pair(StepParams P) {
    static_assert(NTHR % 64 == 0, "two lanes per point, whole warps");
    extern __shared__ double smem[];
    constexpr int UC = TI + 2, UR = TJ + 4, HC = TI + 1, HR = TJ + 2, NP = NTHR / 2;
    double* us = smem;                       // [4L][UR][UC]
    double* hs = smem + 4 * L * UR * UC;     // [4L][HR][HC]
    const int i0 = blockIdx.x * TI, j0 = blockIdx.y * TJ;
    const int iu0 = i0 - 1, ju0 = j0 - 2, jh0 = j0 - 1;
    const int nt = P.n_theta, nr = P.n_r;
    const int tid = threadIdx.x;
    const int p = tid & 1, cP = p, cPi = 2 + p;
    const double sx = p ? 1.0 : -1.0;

    // ---- phase 0: the u^n tile, as in step_kernel
    constexpr int n_stage = 4 * L * UR * UC;
    for (int k = tid; k < n_stage; k += NTHR) {
        int c = k % UC, rest = k / UC;
        int r = rest % UR, pl = rest / UR;
        int ui = iu0 + c, uj = ju0 + r;
        bool ok = ui >= 0 && ui < nr && uj >= 0 && uj < nt;
        cp_async8(us + k, ok ? P.u_in + pl * P.plane + (long)uj * P.pitch + ui : P.u_in, ok);
    }
    cp_async_commit();
    cp_async_wait<0>();
    __syncthreads();

    SmemTile<L> ut{us, UR, UC, ju0};
    // ---- phase 1: half step, Eq. (13)
    for (int q0 = 0; q0 < HR * HC; q0 += NP) {
        const int q = q0 + (tid >> 1);
        const int tr = q / HC, tc = q - tr * HC;
        const int ih = iu0 + tc, jh = jh0 + tr;
        const bool v = q < HR * HC && ih >= 0 && ih <= nr - 2 && jh >= 0 && jh < nt;
        const unsigned mask = __ballot_sync(0xffffffffu, v);
        if (v) {
            int rm = jh - 1, rp = jh + 1;
            double sm = 1.0, sp = 1.0;
            if (rm < 0) { rm = 0; sm = P.sigma; }
            if (rp >= nt) { rp = nt - 1; sp = P.sigma; }
            Real<L> cjv = Ld<L>::g(P.cj, nt, jh);
            Real<L> oP, oPi;
            substep_pair<L>(ut, p, sx, mask, jh, rm, rp, sm, sp, tc, tc + 1, P.coef_h, P.plane, (long)jh * P.pitch + ih, cjv,
                            P.tq_half, true, oP, oPi, oP, oPi);
#pragma unroll
            for (int l = 0; l < L; ++l) {
                hs[(cP * L + l) * HR * HC + tr * HC + tc] = oP.x[l];
                hs[(cPi * L + l) * HR * HC + tr * HC + tc] = oPi.x[l];
            }
        }
    }
    __syncthreads();

    SmemTile<L> ht{hs, HR, HC, jh0};
    // ---- phase 2: full step, Eq. (14), + radial Dirichlet rows + observer nodes
    for (int q0 = 0; q0 < TJ * TI; q0 += NP) {
        const int q = q0 + (tid >> 1);
        const int tr = q / TI, tc = q - tr * TI;
        const int i = i0 + tc, j = j0 + tr;
        const bool v = q < TJ * TI && i < nr && j < nt;
        const bool interior = v && i != 0 && i != nr - 1;
        const unsigned mask = __ballot_sync(0xffffffffu, interior);
        if (v) {
            Real<L> oP = from_double<L>(0.0), oPi = from_double<L>(0.0);
            if (interior) {
                int rm = j - 1, rp = j + 1;
                double sm = 1.0, sp = 1.0;
                if (rm < 0) { rm = 0; sm = P.sigma; }
                if (rp >= nt) { rp = nt - 1; sp = P.sigma; }
                Real<L> bP = ut.get(cP, j, tc + 1), bPi = ut.get(cPi, j, tc + 1);
                Real<L> cjv = Ld<L>::g(P.cj, nt, j);
                substep_pair<L>(ht, p, sx, mask, j, rm, rp, sm, sp, tc, tc + 1, P.coef_i, P.plane, (long)j * P.pitch + i, cjv,
                                P.tq_full, false, bP, bPi, oP, oPi);
            }
            const long g = (long)j * P.pitch + i;
            Ld<L>::st(P.u_out + (long)cP * L * P.plane, P.plane, g, oP);
            Ld<L>::st(P.u_out + (long)cPi * L * P.plane, P.plane, g, oPi);
            if (P.obs_raw != nullptr) {
                int di = i - P.oi, dj = j - P.oj;
                if ((di == 0 || di == 1) && (dj == 0 || dj == 1)) {
                    long k = *P.step_base + P.step_off;
                    if (k < P.obs_cap) {
                        double* o = P.obs_raw + ((k * 4 + (dj * 2 + di)) * 4) * L;
#pragma unroll
                        for (int l = 0; l < L; ++l) { o[cP * L + l] = oP.x[l]; o[cPi * L + l] = oPi.x[l]; }
                    }
                }
            }
        }
    }
}


// ---------------------------------------------------------------------------------------------------------------
// Column kernel for the 10th-order theta operator (NEXT-1): a block owns TI radial columns and ALL
// N_theta rows, so the +-5-row reach of each sub-step needs no theta halo (ghost rows are mirrored reads) and the
// only redundant work is the one extra half-step column per block, (TI+1)/TI.  Same fusion as step_kernel.
template <int L, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) step_kernel_col(StepParams P, ThetaWeights W) {
    extern __shared__ double smem[];
    const int TI = P.ti, nt = P.n_theta, nr = P.n_r;
    const int UC = TI + 2, HC = TI + 1;
    double* us = smem;                       // [4L][nt][UC]
    double* hs = smem + 4 * L * nt * UC;     // [4L][nt][HC]
    double* ss = hs + 4 * L * nt * HC;       // [2L][nt][HC]  staged sig_Phi = Phi_hi + Phi_lo (each sum formed once, used 11x)
    const int i0 = blockIdx.x * TI, iu0 = i0 - 1;
    const int tid = threadIdx.x, nth = MAXT;

    // stage the u^n columns (8-byte zero-fill cp.async: the whole tile in flight at once, as in step_kernel)
    const int n_stage = 4 * L * nt * UC;
    for (int k = tid; k < n_stage; k += nth) {
        int c = k % UC, rest = k / UC;
        int r = rest % nt, pl = rest / nt;
        int ui = iu0 + c;
        bool ok = ui >= 0 && ui < nr;
        cp_async8(us + k, ok ? P.u_in + pl * P.plane + (long)r * P.pitch + ui : P.u_in, ok);
    }
    cp_async_commit();
    cp_async_wait<0>();
    __syncthreads();

    SmemTile<L> ut{us, nt, UC, 0};
    for (int idx = tid; idx < 2 * nt * HC; idx += nth) {
        int tc = idx % HC, rest = idx / HC;
        int tr = rest % nt, c = rest / nt;
        Real<L> sgm = add(ut.get(c, tr, tc + 1), ut.get(c, tr, tc));
#pragma unroll
        for (int l = 0; l < L; ++l) ss[(c * L + l) * nt * HC + tr * HC + tc] = sgm.x[l];
    }
    __syncthreads();
    SmemTile<L> st1{ss, nt, HC, 0};
    for (int idx = tid; idx < nt * HC; idx += nth) {
        int tr = idx / HC, tc = idx - tr * HC;
        int ih = iu0 + tc;
        if (ih < 0 || ih > nr - 2) continue;
        RegCoef<L> cc;
        load_coef(cc, P.coef_h, P.plane, (long)tr * P.pitch + ih);
        Real<L> cjv = Ld<L>::g(P.cj, nt, tr);
        Real<L> out[4];
        substep_wide<L>(ut, st1, tc, tr, nt, P.sigma, tc, tc + 1, cc, cjv, W, P.tq_half, true, out, out);
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int l = 0; l < L; ++l) hs[(c * L + l) * nt * HC + tr * HC + tc] = out[c].x[l];
    }
    __syncthreads();

    SmemTile<L> ht{hs, nt, HC, 0};
    for (int idx = tid; idx < 2 * nt * TI; idx += nth) {      // sig of the half-step field, [2L][nt][TI]
        int tc = idx % TI, rest = idx / TI;
        int tr = rest % nt, c = rest / nt;
        Real<L> sgm = add(ht.get(c, tr, tc + 1), ht.get(c, tr, tc));
#pragma unroll
        for (int l = 0; l < L; ++l) ss[(c * L + l) * nt * TI + tr * TI + tc] = sgm.x[l];
    }
    __syncthreads();
    SmemTile<L> st2{ss, nt, TI, 0};
    for (int idx = tid; idx < nt * TI; idx += nth) {
        int tr = idx / TI, tc = idx - tr * TI;
        int i = i0 + tc, j = tr;
        if (i >= nr) continue;
        Real<L> out[4];
        if (i == 0 || i == nr - 1) {
#pragma unroll
            for (int c = 0; c < 4; ++c) out[c] = from_double<L>(0.0);
        } else {
            RegCoef<L> cc;
            load_coef(cc, P.coef_i, P.plane, (long)j * P.pitch + i);
            Real<L> base[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) base[c] = ut.get(c, j, tc + 1);
            Real<L> cjv = Ld<L>::g(P.cj, nt, j);
            substep_wide<L>(ht, st2, tc, j, nt, P.sigma, tc, tc + 1, cc, cjv, W, P.tq_full, false, base, out);
        }
        long g = (long)j * P.pitch + i;
#pragma unroll
        for (int c = 0; c < 4; ++c) Ld<L>::st(P.u_out + (long)c * L * P.plane, P.plane, g, out[c]);
        if (P.obs_raw != nullptr) {
            int di = i - P.oi, dj = j - P.oj;
            if ((di == 0 || di == 1) && (dj == 0 || dj == 1)) {
                long k = *P.step_base + P.step_off;
                if (k < P.obs_cap) {
                    double* o = P.obs_raw + ((k * 4 + (dj * 2 + di)) * 4) * L;
#pragma unroll
                    for (int c = 0; c < 4; ++c)
#pragma unroll
                        for (int l = 0; l < L; ++l) o[c * L + l] = out[c].x[l];
                }
            }
        }
    }
}

// Pair version of step_kernel_col (same layout, same staging of sig_Phi): two lanes per point as in step_kernel_pair.
template <int L, int NTHR, int MINB>
__global__ void __launch_bounds__(NTHR, MINB) step_kernel_col_pair(StepParams P, ThetaWeights W) {
    static_assert(NTHR % 64 == 0, "two lanes per point, whole warps");
    extern __shared__ double smem[];
    constexpr int NP = NTHR / 2;
    const int TI = P.ti, nt = P.n_theta, nr = P.n_r;
    const int UC = TI + 2, HC = TI + 1;
    double* us = smem;                       // [4L][nt][UC]
    double* hs = smem + 4 * L * nt * UC;     // [4L][nt][HC]
    double* ss = hs + 4 * L * nt * HC;       // [2L][nt][HC]
    const int i0 = blockIdx.x * TI, iu0 = i0 - 1;
    const int tid = threadIdx.x;
    const int p = tid & 1, cP = p, cPi = 2 + p;
    const double sx = p ? 1.0 : -1.0;

    const int n_stage = 4 * L * nt * UC;
    for (int k = tid; k < n_stage; k += NTHR) {
        int c = k % UC, rest = k / UC;
        int r = rest % nt, pl = rest / nt;
        int ui = iu0 + c;
        bool ok = ui >= 0 && ui < nr;
        cp_async8(us + k, ok ? P.u_in + pl * P.plane + (long)r * P.pitch + ui : P.u_in, ok);
    }
    cp_async_commit();
    cp_async_wait<0>();
    __syncthreads();

    SmemTile<L> ut{us, nt, UC, 0};
    for (int idx = tid; idx < 2 * nt * HC; idx += NTHR) {
        int tc = idx % HC, rest = idx / HC;
        int tr = rest % nt, c = rest / nt;
        Real<L> sgm = add(ut.get(c, tr, tc + 1), ut.get(c, tr, tc));
#pragma unroll
        for (int l = 0; l < L; ++l) ss[(c * L + l) * nt * HC + tr * HC + tc] = sgm.x[l];
    }
    __syncthreads();
    SmemTile<L> st1{ss, nt, HC, 0};
    for (int q0 = 0; q0 < nt * HC; q0 += NP) {
        const int q = q0 + (tid >> 1);
        const int tr = q / HC, tc = q - tr * HC;
        const int ih = iu0 + tc;
        const bool v = q < nt * HC && ih >= 0 && ih <= nr - 2;
        const unsigned mask = __ballot_sync(0xffffffffu, v);
        if (v) {
            Real<L> cjv = Ld<L>::g(P.cj, nt, tr);
            Real<L> oP, oPi;
            substep_wide_pair<L>(ut, st1, tc, p, sx, mask, tr, nt, P.sigma, tc, tc + 1, P.coef_h, P.plane, (long)tr * P.pitch + ih,
                                 cjv, W, P.tq_half, true, oP, oPi, oP, oPi);
#pragma unroll
            for (int l = 0; l < L; ++l) {
                hs[(cP * L + l) * nt * HC + tr * HC + tc] = oP.x[l];
                hs[(cPi * L + l) * nt * HC + tr * HC + tc] = oPi.x[l];
            }
        }
    }
    __syncthreads();

    SmemTile<L> ht{hs, nt, HC, 0};
    for (int idx = tid; idx < 2 * nt * TI; idx += NTHR) {
        int tc = idx % TI, rest = idx / TI;
        int tr = rest % nt, c = rest / nt;
        Real<L> sgm = add(ht.get(c, tr, tc + 1), ht.get(c, tr, tc));
#pragma unroll
        for (int l = 0; l < L; ++l) ss[(c * L + l) * nt * TI + tr * TI + tc] = sgm.x[l];
    }
    __syncthreads();
    SmemTile<L> st2{ss, nt, TI, 0};
    for (int q0 = 0; q0 < nt * TI; q0 += NP) {
        const int q = q0 + (tid >> 1);
        const int tr = q / TI, tc = q - tr * TI;
        const int i = i0 + tc, j = tr;
        const bool v = q < nt * TI && i < nr;
        const bool interior = v && i != 0 && i != nr - 1;
        const unsigned mask = __ballot_sync(0xffffffffu, interior);
        if (v) {
            Real<L> oP = from_double<L>(0.0), oPi = from_double<L>(0.0);
            if (interior) {
                Real<L> bP = ut.get(cP, j, tc + 1), bPi = ut.get(cPi, j, tc + 1);
                Real<L> cjv = Ld<L>::g(P.cj, nt, j);
                substep_wide_pair<L>(ht, st2, tc, p, sx, mask, j, nt, P.sigma, tc, tc + 1, P.coef_i, P.plane, (long)j * P.pitch + i,
                                     cjv, W, P.tq_full, false, bP, bPi, oP, oPi);
            }
            const long g = (long)j * P.pitch + i;
            Ld<L>::st(P.u_out + (long)cP * L * P.plane, P.plane, g, oP);
            Ld<L>::st(P.u_out + (long)cPi * L * P.plane, P.plane, g, oPi);
            if (P.obs_raw != nullptr) {
                int di = i - P.oi, dj = j - P.oj;
                if ((di == 0 || di == 1) && (dj == 0 || dj == 1)) {
                    long k = *P.step_base + P.step_off;
                    if (k < P.obs_cap) {
                        double* o = P.obs_raw + ((k * 4 + (dj * 2 + di)) * 4) * L;
#pragma unroll
                        for (int l = 0; l < L; ++l) { o[cP * L + l] = oP.x[l]; o[cPi * L + l] = oPi.x[l]; }
                    }
                }
            }
        }
    }
}

}  // namespace tk
