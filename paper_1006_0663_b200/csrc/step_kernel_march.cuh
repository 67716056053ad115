// fp64 step kernel, "column march" (round 2; the default fp64 path).  Same iteration as every other step kernel --
// half step Eq. (13) + full step Eq. (14), radial Dirichlet rows and polar ghosts,
// observer nodes in one launch -- with the SEMI-RECOMPUTE coefficient supply of H1b variant (b)
// (one 1/Sigma plane per point family + 1-D tables; 64 + 16 = 80 B of HBM traffic per update), but organised so that
// almost every instruction is arithmetic:
//   * a WARP owns a strip of 30 output columns and marches down theta; lane l holds column 30 s - 1 + l.  The column
//     to the right comes from lane l + 1 by shuffle, so each u value is loaded from global memory exactly once per
//     warp (coalesced 256-byte rows, two rows prefetched into registers) and nothing is staged in shared memory;
//   * the half-step field never leaves registers: lane l computes h at (30 s - 1/2 + l, j), the full step at column
//     30 s + l takes h(i - 1/2) from itself and h(i + 1/2) from lane l + 1 by shuffle.  No barriers, warps are
//     independent;
//   * sig_Phi = Phi_hi + Phi_lo is formed once per row and kept in a three-row register window for the angular
//     operator Lambda (the tile kernels form it three times and read the tile six times per sub-step);
//   * the 28 r-only table entries of a column (rc_eval) are fetched once per strip segment, not once per point;
//   * the grid is persistent: the strip-rows (strip-major) are dealt out in equal contiguous shares, one per resident
//     warp, so there is no wave tail and no block-launch overhead.  A share that starts inside a strip pays a two-row
//     theta halo (redundant half steps), ~5 % at the bench sizes.
// Redundant work in r*: 32 lanes load, 31 compute half steps, 30 produce outputs.
#pragma once
#include "step_kernel_tma.cuh"     // RcCoef, rc_eval, StepParams

namespace tk {

constexpr int MARCH_W = 30;         // output columns per warp
constexpr int MARCH_WARPS = 4;      // warps per block
constexpr int MARCH_NRT = 14;       // r-tables used by rc_eval

struct MarchParams {
    const double* isig_i;           // 1/Sigma at integer points [n_theta][pitch]
    const double* isig_h;           // 1/Sigma at half points (column i <-> i + 1/2)
    const double* rt;               // r-tables [2 families][16][pitch]: family 0 integer points, 1 half points
    const double* th;               // theta tables [3][n_theta]: sin^2, cos, Tth
    long rows_per_warp;             // share of strip-rows per warp
    long total_rows;                // n_strips * n_theta
};

__device__ __forceinline__ double shfl_down1(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// Lambda~ = ((up + dn) - 2 s) + cj (up - dn)
__device__ __forceinline__ double lam_op(double up, double dn, double s, double cj) {
    return ((up + dn) - 2.0 * s) + cj * (up - dn);
}

// one sub-step at one point from sig = hi + lo, del = hi - lo (radial neighbours), lam[2] = Lambda~[sig_Phi]; see the
// header of step_kernel.cuh for the folded coefficients c0..c7.  base = sig / 2 (half step) or u^n (full step).
__device__ __forceinline__ void march_core(const double sg[4], const double dl[4], const double lam[2], const RcCoef& cf,
                                           double tq, const double base[4], double out[4]) {
    const double* c = cf.c;
    double sR = -(c[1] * sg[2] - c[2] * sg[3]);
    double sI = -(c[1] * sg[3] + c[2] * sg[2]);
    sR = sR + (c[3] * dl[0] - c[4] * dl[1]);
    sI = sI + (c[3] * dl[1] + c[4] * dl[0]);
    sR = sR + c[7] * lam[0];
    sI = sI + c[7] * lam[1];
    sR = sR - (c[5] * sg[0] - c[6] * sg[1]);
    sI = sI - (c[5] * sg[1] + c[6] * sg[0]);
    out[0] = (base[0] - c[0] * dl[0]) + sg[2] * tq;
    out[1] = (base[1] - c[0] * dl[1]) + sg[3] * tq;
    out[2] = (base[2] + c[0] * dl[2]) + sR;
    out[3] = (base[3] + c[0] * dl[3]) + sI;
}

struct MarchRow {                   // one prefetched row: u at the lane's column, 1/Sigma at its half and integer point
    double u[4], ish, isi;
};

template <bool RT_REGS>
__global__ void __launch_bounds__(32 * MARCH_WARPS, RT_REGS ? 2 : 3) step_kernel_f64_march(StepParams P, MarchParams Q) {
    extern __shared__ double sm[];
    const int nt = P.n_theta, nr = P.n_r;
    double* tht = sm;                                                // [4][nt]: cj, sin^2, cos, Tth
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double* rts = sm + 4 * nt + warp * (2 * MARCH_NRT * 32);         // per warp [2][14][32]
    for (int k = threadIdx.x; k < 4 * nt; k += blockDim.x) tht[k] = (k < nt) ? __ldg(P.cj + k) : __ldg(Q.th + (k - nt));
    __syncthreads();
    const double sigma = P.sigma;

    const long gw = (long)blockIdx.x * MARCH_WARPS + warp;
    long t = gw * Q.rows_per_warp;
    const long t_end = min(t + Q.rows_per_warp, Q.total_rows);
    while (t < t_end) {
        const int s = (int)(t / nt);
        const int ja = (int)(t - (long)s * nt);
        const int jb = (int)min((long)nt, ja + (t_end - t));
        t += jb - ja;

        const int cu = MARCH_W * s - 1 + lane;                      // this lane's column (lo of its half point)
        const int ci = cu + 1;                                      // its output column (lanes 0..29)
        const bool lo_ok = cu >= 0 && cu < nr;
        const bool h_ok = cu >= 0 && ci < nr;                       // half point (cu, cu + 1) exists
        const bool i_ok = ci < nr && lane < MARCH_W;
        const bool interior = i_ok && ci > 0 && ci < nr - 1;
        // r-only table entries of this lane's half point and output column
        double rth[MARCH_NRT], rti[MARCH_NRT];
        __syncwarp();
#pragma unroll
        for (int q = 0; q < MARCH_NRT; ++q) {
            const double vh = h_ok ? __ldg(Q.rt + (long)(16 + q) * P.pitch + cu) : 0.0;
            const double vi = (ci < nr) ? __ldg(Q.rt + (long)q * P.pitch + ci) : 0.0;
            if (RT_REGS) { rth[q] = vh; rti[q] = vi; }
            else { rts[q * 32 + lane] = vh; rts[(MARCH_NRT + q) * 32 + lane] = vi; }
        }
        __syncwarp();

        const int ha = max(ja - 1, 0), hb = min(jb + 1, nt);        // half-step rows
        const int ua = max(ha - 1, 0), ub = min(hb + 1, nt);        // u rows
        const double* up_lo = P.u_in + cu;
        auto fetch = [&](MarchRow& w, int r) {
            const long off = (long)r * P.pitch;
#pragma unroll
            for (int c = 0; c < 4; ++c) w.u[c] = lo_ok ? __ldg(up_lo + c * P.plane + off) : 0.0;
            w.ish = h_ok ? __ldg(Q.isig_h + off + cu) : 0.0;
            w.isi = (ci < nr) ? __ldg(Q.isig_i + off + ci) : 0.0;
        };
        MarchRow pf[2];
        if (ua < ub) fetch(pf[0], ua);
        if (ua + 1 < ub) fetch(pf[1], ua + 1);

        // rolling register windows, slot = iteration count modulo 3 (row r), (r - 1), (r - 2)
        double SU[3][2], HI[3][4], ISI[3], SGP[3][2], DL[3][4], ISH[3];      // u side: sig_Phi, u at column ci, 1/Sigma, sig_Pi, del
        double SH[3][2], SHP[3][2], DH[3][4];                                 // h side: sig_Phi, sig_Pi, del of the half-step field
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            ISI[a] = ISH[a] = 0.0;
#pragma unroll
            for (int c = 0; c < 4; ++c) { HI[a][c] = DL[a][c] = DH[a][c] = 0.0; }
#pragma unroll
            for (int c = 0; c < 2; ++c) { SU[a][c] = SGP[a][c] = SH[a][c] = SHP[a][c] = 0.0; }
        }

        for (int rb = ua; rb <= jb + 1; rb += 6) {
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                const int r = rb + k;
                constexpr int dummy = 0; (void)dummy;
                const int n0 = k % 3, n1 = (k + 2) % 3, n2 = (k + 1) % 3;       // slots of rows r, r - 1, r - 2 (and r - 3 = n0)
                // ---- A: row r of u arrives
                if (r < ub) {
                    MarchRow& w = pf[k % 2];
                    double lo[4];
#pragma unroll
                    for (int c = 0; c < 4; ++c) lo[c] = w.u[c];
                    ISH[n0] = w.ish;
                    ISI[n0] = w.isi;
                    if (r + 2 < ub) fetch(w, r + 2);
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const double hi = shfl_down1(lo[c]);
                        HI[n0][c] = hi;
                        DL[n0][c] = hi - lo[c];
                        if (c < 2) SU[n0][c] = hi + lo[c]; else SGP[n0][c - 2] = hi + lo[c];
                    }
                }
                // ---- B: half step at row q = r - 1, Eq. (13)
                const int q = r - 1;
                if (q >= ha && q < hb) {
                    double sg[4] = {SU[n1][0], SU[n1][1], SGP[n1][0], SGP[n1][1]};
                    double lam[2], base[4], h[4];
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const double dn = (q > 0) ? SU[n2][c] : sigma * SU[n1][c];
                        const double up = (q + 1 < nt) ? SU[n0][c] : sigma * SU[n1][c];
                        lam[c] = lam_op(up, dn, sg[c], tht[q]);
                    }
#pragma unroll
                    for (int c = 0; c < 4; ++c) base[c] = 0.5 * sg[c];
                    RcCoef cf;
                    if (RT_REGS) rc_eval(cf, ISH[n1], rth, 1, tht[nt + q], tht[2 * nt + q], tht[3 * nt + q]);
                    else rc_eval(cf, ISH[n1], rts + lane, 32, tht[nt + q], tht[2 * nt + q], tht[3 * nt + q]);
                    march_core(sg, DL[n1], lam, cf, P.tq_half, base, h);
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const double hn = shfl_down1(h[c]);            // h at (ci + 1/2, q)
                        DH[n1][c] = hn - h[c];
                        if (c < 2) SH[n1][c] = hn + h[c]; else SHP[n1][c - 2] = hn + h[c];
                    }
                }
                // ---- C: full step at row q2 = r - 2, Eq. (14); radial Dirichlet rows; observer nodes
                const int q2 = r - 2;
                if (q2 >= ja && q2 < jb) {
                    double sg[4] = {SH[n2][0], SH[n2][1], SHP[n2][0], SHP[n2][1]};
                    double lam[2], out[4];
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        const double dn = (q2 > 0) ? SH[n0][c] : sigma * SH[n2][c];
                        const double up = (q2 + 1 < nt) ? SH[n1][c] : sigma * SH[n2][c];
                        lam[c] = lam_op(up, dn, sg[c], tht[q2]);
                    }
                    RcCoef cf;
                    if (RT_REGS) rc_eval(cf, ISI[n2], rti, 1, tht[nt + q2], tht[2 * nt + q2], tht[3 * nt + q2]);
                    else rc_eval(cf, ISI[n2], rts + MARCH_NRT * 32 + lane, 32, tht[nt + q2], tht[2 * nt + q2], tht[3 * nt + q2]);
                    march_core(sg, DH[n2], lam, cf, P.tq_full, HI[n2], out);
                    if (i_ok) {
                        const long g = (long)q2 * P.pitch + ci;
#pragma unroll
                        for (int c = 0; c < 4; ++c) P.u_out[(long)c * P.plane + g] = interior ? out[c] : 0.0;
                        if (P.obs_raw != nullptr) {
                            const int di = ci - P.oi, dj = q2 - P.oj;
                            if ((di == 0 || di == 1) && (dj == 0 || dj == 1)) {
                                const long ks = *P.step_base + P.step_off;
                                if (ks < P.obs_cap) {
                                    double* o = P.obs_raw + ((ks * 4 + (dj * 2 + di)) * 4);
#pragma unroll
                                    for (int c = 0; c < 4; ++c) o[c] = interior ? out[c] : 0.0;
                                }
                            }
                        }
                    }
                }
            }
        }
    }
}

}  // namespace tk
