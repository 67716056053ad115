// NEXT-3 (the paper cites temporal-locality stencil work): fp64 step kernel that
// advances TWO iterations of Eqs. (13)-(14) per launch on a shared-memory resident trapezoid.
// The time-independent coefficient tiles are fetched once and used by both iterations, and u^{n+1} never reaches
// HBM, so the algorithmic traffic per update halves: (4 read + 4 written state + 16 coefficient doubles) / 2
// = 96 B/update instead of 192 B (plus halo re-reads, which neighbouring blocks find in L2).
//
// Output tile TI x TJ of u^{n+2}; dependency cone (r* reach 1 and theta reach 2 per iteration):
//   level 0  u^n          cols i0-2 .. i0+TI+1   rows j0-4 .. j0+TJ+3     TMA tile, zero-filled outside the grid
//   level 1  h^{n+1/2}    half pts i0-2 .. i0+TI rows j0-3 .. j0+TJ+2     smem
//   level 2  u^{n+1}      cols i0-1 .. i0+TI     rows j0-2 .. j0+TJ+1     smem, IN PLACE over u^n (a full step reads
//                                                                          u^n only at its own point)
//   level 3  h^{n+3/2}    half pts i0-1 .. i0+TI-1, rows j0-1 .. j0+TJ    smem, over level 1
//   level 4  u^{n+2}      TI x TJ                                         global
// Half-point coefficients: one TMA tile (8 planes) covering level 1, re-read by level 3.  Integer-point
// coefficients: each thread loads the 8 coefficients of "its" points straight into registers (coalesced rows)
// BEFORE waiting for the state tile; the TI x TJ interior points are owned by the same thread at levels 2 and 4, so
// those registers serve both iterations and the integer-point tile needs no shared memory at all (103 KB per
// block, 2 blocks/SM).  Same arithmetic as the single-step kernels (substep<1>); radial Dirichlet rows, polar
// parity ghosts and observer samples of BOTH iterations are produced here.
#pragma once
#include "step_kernel_tma.cuh"

namespace tk {

template <int TI, int TJ> struct Tb2Geom {
    static constexpr int UC = TI + 4, UR = TJ + 8;            // u tile, first column i0-2 (even: 16-byte TMA alignment)
    static constexpr int CC = TI + 4, H1R = TJ + 6;           // half-point coefficient tile, first half point i0-2
    static constexpr int H1C = TI + 3;                        // level-1 tile
    static constexpr int H2C = TI + 1, H2R = TJ + 2;          // level-3 tile
    static constexpr int RING = (TI + 2) * (TJ + 4) - TI * TJ;   // level-2 points outside the TI x TJ interior
    static constexpr int a128(int v) { return (v + 127) / 128 * 128; }
    static constexpr int US_B = a128(4 * UR * UC * 8);
    static constexpr int CH_B = a128(8 * H1R * CC * 8);
    static constexpr int HS_B = a128(4 * H1R * H1C * 8);
    static constexpr int TOTAL = US_B + CH_B + HS_B + 128;
};

struct RegCoef1 {
    double c[8];
    __device__ __forceinline__ R1 get(int q) const { R1 r; r.x[0] = c[q]; return r; }
};

template <int TI, int TJ>
__global__ void __launch_bounds__(256, 2) step2_kernel_f64_tma(const __grid_constant__ CUtensorMap tm_u,
                                                              const __grid_constant__ CUtensorMap tm_ch, StepParams P) {
    using G = Tb2Geom<TI, TJ>;
    static_assert(TI == 32 && TJ % 8 == 0, "one warp lane per interior column, 8 warps over the rows");
    constexpr int UC = G::UC, UR = G::UR, CC = G::CC, H1R = G::H1R, H1C = G::H1C, H2C = G::H2C, H2R = G::H2R;
    constexpr int KIN = TJ / 8;
    extern __shared__ __align__(128) unsigned char raw[];
    __shared__ __align__(8) uint64_t bar[2];
    unsigned char* base = raw;
    double* us = (double*)base;
    double* chs = (double*)(base + G::US_B);
    double* hs = (double*)(base + G::US_B + G::CH_B);
    // blockIdx.x runs over the theta tiles (fastest) so that blocks sharing theta halos run at the same time
    const int i0 = blockIdx.y * TI, j0 = blockIdx.x * TJ;
    const int nt = P.n_theta, nr = P.n_r;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(&bar[1], 8 * H1R * CC * 8);
        tma_load_3d(chs, &tm_ch, i0 - 2, j0 - 3, 0, &bar[1]);
    }
    // integer-point coefficients of this thread's points -> registers (time independent: issued before the wait)
    RegCoef1 cin[KIN], crg;
#pragma unroll
    for (int k = 0; k < KIN; ++k) {
        int i = i0 + lane, j = j0 + warp + 8 * k;
        bool ok = i < nr && j < nt;
        long g = (long)j * P.pitch + i;
#pragma unroll
        for (int q = 0; q < 8; ++q) cin[k].c[q] = ok ? __ldg(P.coef_i + q * P.plane + g) : 0.0;
    }
    // ring point of this thread (levels 2 only): rows j0-2, j0-1, j0+TJ, j0+TJ+1 (TI+2 columns each), then the two
    // side columns i0-1 and i0+TI over the TJ interior rows
    int rtr = 0, rtc = 0;
    bool ring = tid < G::RING;
    if (ring) {
        if (tid < 4 * (TI + 2)) {
            int r = tid / (TI + 2);
            rtc = tid - r * (TI + 2) - 1;
            rtr = (r < 2) ? r - 2 : TJ + r - 2;
        } else {
            int t = tid - 4 * (TI + 2);
            rtr = t >> 1;
            rtc = (t & 1) ? TI : -1;
        }
        int i = i0 + rtc, j = j0 + rtr;
        ring = i >= 0 && i < nr && j >= 0 && j < nt;
        long g = (long)j * P.pitch + i;
#pragma unroll
        for (int q = 0; q < 8; ++q) crg.c[q] = ring ? __ldg(P.coef_i + q * P.plane + g) : 0.0;
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");        // u^n (written by the previous launch) is complete
    if (tid == 0) {
        mbar_expect_tx(&bar[0], 4 * UR * UC * 8);
        tma_load_3d(us, &tm_u, i0 - 2, j0 - 4, 0, &bar[0]);
    }
    __syncthreads();
    mbar_wait(&bar[0], 0);
    mbar_wait(&bar[1], 0);

    CTile<UR, UC> ut{us, j0 - 4};
    // ---- level 1: half step of iteration 1, Eq. (13)
#pragma unroll
    for (int k = 0; k < (H1R * H1C + 255) / 256; ++k) {
        int idx = tid + k * 256;
        if (idx < H1R * H1C) {
            int tr = idx / H1C, tc = idx - tr * H1C;
            int ih = i0 - 2 + tc, jh = j0 - 3 + tr;
            if (ih >= 0 && ih <= nr - 2 && jh >= 0 && jh < nt) {
                int rm = jh - 1, rp = jh + 1;
                double sm = 1.0, sp = 1.0;
                if (rm < 0) { rm = 0; sm = P.sigma; }
                if (rp >= nt) { rp = nt - 1; sp = P.sigma; }
                R1 cjv;
                cjv.x[0] = __ldg(P.cj + jh);
                CCoef<H1R, CC> cf{chs + tr * CC + tc};
                R1 out[4];
                substep<1>(ut, jh, rm, rp, sm, sp, tc, tc + 1, cf, cjv, P.tq_half, true, out, out);
#pragma unroll
                for (int c = 0; c < 4; ++c) hs[c * H1R * H1C + tr * H1C + tc] = out[c].x[0];
            }
        }
    }
    __syncthreads();

    // ---- level 2: full step of iteration 1, Eq. (14), written over u^n in the tile; observer sample of step n+1
    {
        CTile<H1R, H1C> ht{hs, j0 - 3};
        const long ks = (P.obs_raw != nullptr) ? *P.step_base + P.step_off : 0;
#pragma unroll
        for (int k = 0; k <= KIN; ++k) {
            int tr, tc;
            bool act;
            if (k < KIN) { tr = warp + 8 * k; tc = lane; act = true; }
            else { tr = rtr; tc = rtc; act = ring; }
            int i = i0 + tc, j = j0 + tr;
            if (!act || i >= nr || j >= nt) continue;
            R1 out[4];
            if (i == 0 || i == nr - 1) {
#pragma unroll
                for (int c = 0; c < 4; ++c) out[c].x[0] = 0.0;
            } else {
                int rm = j - 1, rp = j + 1;
                double sm = 1.0, sp = 1.0;
                if (rm < 0) { rm = 0; sm = P.sigma; }
                if (rp >= nt) { rp = nt - 1; sp = P.sigma; }
                R1 bs[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) bs[c] = ut.get(c, j, tc + 2);
                R1 cjv;
                cjv.x[0] = __ldg(P.cj + j);
                if (k < KIN) substep<1>(ht, j, rm, rp, sm, sp, tc + 1, tc + 2, cin[k < KIN ? k : 0], cjv, P.tq_full, false, bs, out);
                else substep<1>(ht, j, rm, rp, sm, sp, tc + 1, tc + 2, crg, cjv, P.tq_full, false, bs, out);
            }
#pragma unroll
            for (int c = 0; c < 4; ++c) us[c * UR * UC + (tr + 4) * UC + tc + 2] = out[c].x[0];
            if (k < KIN && P.obs_raw != nullptr) {
                int di = i - P.oi, dj = j - P.oj;
                if ((di == 0 || di == 1) && (dj == 0 || dj == 1) && ks < P.obs_cap) {
                    double* o = P.obs_raw + ((ks * 4 + (dj * 2 + di)) * 4);
#pragma unroll
                    for (int c = 0; c < 4; ++c) o[c] = out[c].x[0];
                }
            }
        }
    }
    __syncthreads();

    // ---- level 3: half step of iteration 2 (coefficients: the interior of the same half-point tile)
#pragma unroll
    for (int k = 0; k < (H2R * H2C + 255) / 256; ++k) {
        int idx = tid + k * 256;
        if (idx < H2R * H2C) {
            int tr = idx / H2C, tc = idx - tr * H2C;
            int ih = i0 - 1 + tc, jh = j0 - 1 + tr;
            if (ih >= 0 && ih <= nr - 2 && jh >= 0 && jh < nt) {
                int rm = jh - 1, rp = jh + 1;
                double sm = 1.0, sp = 1.0;
                if (rm < 0) { rm = 0; sm = P.sigma; }
                if (rp >= nt) { rp = nt - 1; sp = P.sigma; }
                R1 cjv;
                cjv.x[0] = __ldg(P.cj + jh);
                CCoef<H1R, CC> cf{chs + (tr + 2) * CC + tc + 1};
                R1 out[4];
                substep<1>(ut, jh, rm, rp, sm, sp, tc + 1, tc + 2, cf, cjv, P.tq_half, true, out, out);
#pragma unroll
                for (int c = 0; c < 4; ++c) hs[c * H2R * H2C + tr * H2C + tc] = out[c].x[0];
            }
        }
    }
    __syncthreads();

    // ---- level 4: full step of iteration 2 -> global, radial Dirichlet rows, observer sample of step n+2
    {
        CTile<H2R, H2C> ht{hs, j0 - 1};
        const long ks = (P.obs_raw != nullptr) ? *P.step_base + P.step_off + 1 : 0;
#pragma unroll
        for (int k = 0; k < KIN; ++k) {
            int tr = warp + 8 * k, tc = lane;
            int i = i0 + tc, j = j0 + tr;
            if (i >= nr || j >= nt) continue;
            R1 out[4];
            if (i == 0 || i == nr - 1) {
#pragma unroll
                for (int c = 0; c < 4; ++c) out[c].x[0] = 0.0;
            } else {
                int rm = j - 1, rp = j + 1;
                double sm = 1.0, sp = 1.0;
                if (rm < 0) { rm = 0; sm = P.sigma; }
                if (rp >= nt) { rp = nt - 1; sp = P.sigma; }
                R1 bs[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) bs[c] = ut.get(c, j, tc + 2);
                R1 cjv;
                cjv.x[0] = __ldg(P.cj + j);
                substep<1>(ht, j, rm, rp, sm, sp, tc, tc + 1, cin[k], cjv, P.tq_full, false, bs, out);
            }
            long g = (long)j * P.pitch + i;
#pragma unroll
            for (int c = 0; c < 4; ++c) P.u_out[(long)c * P.plane + g] = out[c].x[0];
            if (P.obs_raw != nullptr) {
                int di = i - P.oi, dj = j - P.oj;
                if ((di == 0 || di == 1) && (dj == 0 || dj == 1) && ks < P.obs_cap) {
                    double* o = P.obs_raw + ((ks * 4 + (dj * 2 + di)) * 4);
#pragma unroll
                    for (int c = 0; c < 4; ++c) o[c] = out[c].x[0];
                }
            }
        }
    }
}

}  // namespace tk
