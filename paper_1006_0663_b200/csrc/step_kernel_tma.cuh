// fp64 step kernel for sm_100a with TMA staging (the HBM-bound precision).  Same arithmetic as
// step_kernel<1> (it calls the same substep<1>), different data movement:
//   * ONE elected thread issues three 3-D tiled TMA loads (cp.async.bulk.tensor) per block: the u^n tile
//     with its halo (4 planes), the half-point coefficient tile (8 planes) and the integer-point
//     coefficient tile (8 planes).  Out-of-range columns/rows are zero-filled by the TMA unit, which
//     supplies the radial Dirichlet halo for free; polar ghosts stay mirrored reads.
//   * all ~90 KB a block needs are in flight from its first instruction (two mbarriers: the full-step
//     coefficients may land while the half step computes), so HBM latency is paid once per block and
//     hidden by the co-resident block(s);
//   * tile sizes are compile-time, so index arithmetic folds into constants (the generic kernel spends
//     ~900 thread instructions per update, mostly integer).
#pragma once
#include <cuda.h>

#include <cstdint>
#include <type_traits>

#include "step_kernel.cuh"

namespace tk {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n"
            : "=r"(done)
            : "r"(smem_u32(bar)), "r"(parity)
            : "memory");
    } while (!done);
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int x, int y, int z, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
            smem_u32(dst)),
        "l"(reinterpret_cast<uint64_t>(map)), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar))
        : "memory");
}

template <int TI, int TJ> struct TmaGeom {
    // TMA needs a 16-byte aligned start in the innermost dimension, i.e. an EVEN first column: both haloed boxes
    // start at column i0 - 2 (one unused leading column) instead of i0 - 1.
    static constexpr int UC = TI + 4, UR = TJ + 4, HC = TI + 1, HR = TJ + 2, CC = TI + 2;
    static constexpr int a128(int v) { return (v + 127) / 128 * 128; }
    static constexpr int US_B = a128(4 * UR * UC * 8);        // u tile   [4][UR][UC], columns i0-2 .. i0+TI+1
    static constexpr int CH_B = a128(8 * HR * CC * 8);        // coef_h   [8][HR][CC], half points i0-2 .. i0+TI-1
    static constexpr int CI_B = a128(8 * TJ * TI * 8);        // coef_i   [8][TJ][TI]
    static constexpr int HS_B = a128(4 * HR * HC * 8);        // h tile   [4][HR][HC]
    static constexpr int TOTAL = US_B + CH_B + CI_B + HS_B + 128;
};

template <int ROWS, int COLS> struct CTile {       // compile-time shaped smem tile of fp64 planes
    const double* p;
    int row0;
    __device__ __forceinline__ R1 get(int c, int grow, int col) const {
        R1 r;
        r.x[0] = p[c * ROWS * COLS + (grow - row0) * COLS + col];
        return r;
    }
};
template <int ROWS, int COLS> struct CCoef {
    const double* p;     // already offset to (row, col)
    __device__ __forceinline__ R1 get(int q) const {
        R1 r;
        r.x[0] = p[q * ROWS * COLS];
        return r;
    }
};

template <int TI, int TJ>
__global__ void __launch_bounds__(256) step_kernel_f64_tma(const __grid_constant__ CUtensorMap tm_u,
                                                          const __grid_constant__ CUtensorMap tm_ch,
                                                          const __grid_constant__ CUtensorMap tm_ci, StepParams P) {
    using G = TmaGeom<TI, TJ>;
    constexpr int UC = G::UC, UR = G::UR, HC = G::HC, HR = G::HR, CC = G::CC;
    extern __shared__ __align__(128) unsigned char raw[];
    __shared__ __align__(8) uint64_t bar[3];
    unsigned char* base = raw;      // __align__(128) on the extern array is honoured; no integer round trip, so the
                                    // compiler keeps these pointers in the shared state space (LDS/STS, not generic LD/ST)
    double* us = (double*)base;
    double* chs = (double*)(base + G::US_B);
    double* cis = (double*)(base + G::US_B + G::CH_B);
    double* hs = (double*)(base + G::US_B + G::CH_B + G::CI_B);
    const int i0 = blockIdx.x * TI, j0 = blockIdx.y * TJ;
    const int nt = P.n_theta, nr = P.n_r;
    const int tid = threadIdx.x;

    // Programmatic dependent launch: let the next step's grid start as soon as SM resources free up ...
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_init(&bar[2], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        // ... and fetch the TIME-INDEPENDENT coefficient tiles before waiting for the previous step to finish
        // (the half-step tile only: the TMA unit serves requests in order, and the full-step tile must not delay u)
        mbar_expect_tx(&bar[2], 8 * HR * CC * 8);
        tma_load_3d(chs, &tm_ch, i0 - 2, j0 - 1, 0, &bar[2]);
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");        // u^n (written by the previous step) is complete and visible
    if (tid == 0) {
        mbar_expect_tx(&bar[0], 4 * UR * UC * 8);
        tma_load_3d(us, &tm_u, i0 - 2, j0 - 2, 0, &bar[0]);
        mbar_expect_tx(&bar[1], 8 * TJ * TI * 8);
        tma_load_3d(cis, &tm_ci, i0, j0, 0, &bar[1]);
    }
    __syncthreads();
    mbar_wait(&bar[0], 0);
    mbar_wait(&bar[2], 0);

    CTile<UR, UC> ut{us, j0 - 2};
    // ---- half step, Eq. (13)
#pragma unroll
    for (int k = 0; k < (HR * HC + 255) / 256; ++k) {
        int idx = tid + k * 256;
        if (idx < HR * HC) {
            int tr = idx / HC, tc = idx - tr * HC;
            int ih = i0 - 1 + tc, jh = j0 - 1 + tr;
            if (ih >= 0 && ih <= nr - 2 && jh >= 0 && jh < nt) {
                int rm = jh - 1, rp = jh + 1;
                double sm = 1.0, sp = 1.0;
                if (rm < 0) { rm = 0; sm = P.sigma; }
                if (rp >= nt) { rp = nt - 1; sp = P.sigma; }
                R1 cjv;
                cjv.x[0] = __ldg(P.cj + jh);
                CCoef<HR, CC> cf{chs + tr * CC + tc + 1};
                R1 out[4];
                substep<1>(ut, jh, rm, rp, sm, sp, tc + 1, tc + 2, cf, cjv, P.tq_half, true, out, out);
#pragma unroll
                for (int c = 0; c < 4; ++c) hs[c * HR * HC + tr * HC + tc] = out[c].x[0];
            }
        }
    }
    __syncthreads();
    mbar_wait(&bar[1], 0);

    CTile<HR, HC> ht{hs, j0 - 1};
    // ---- full step, Eq. (14), radial Dirichlet rows, observer nodes
    const int lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int k = 0; k < (TJ * TI + 255) / 256; ++k) {
        int tr, tc;
        if (TI == 32) { tr = warp + 8 * k; tc = lane; }
        else { int idx = tid + k * 256; tr = idx / TI; tc = idx - tr * TI; }
        int i = i0 + tc, j = j0 + tr;
        if (tr >= TJ || i >= nr || j >= nt) continue;
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
            CCoef<TJ, TI> cf{cis + tr * TI + tc};
            substep<1>(ht, j, rm, rp, sm, sp, tc, tc + 1, cf, cjv, P.tq_full, false, bs, out);
        }
        long g = (long)j * P.pitch + i;
#pragma unroll
        for (int c = 0; c < 4; ++c) P.u_out[(long)c * P.plane + g] = out[c].x[0];
        if (P.obs_raw != nullptr) {
            int di = i - P.oi, dj = j - P.oj;
            if ((di == 0 || di == 1) && (dj == 0 || dj == 1)) {
                long ks = *P.step_base + P.step_off;
                if (ks < P.obs_cap) {
                    double* o = P.obs_raw + ((ks * 4 + (dj * 2 + di)) * 4);
#pragma unroll
                    for (int c = 0; c < 4; ++c) o[c] = out[c].x[0];
                }
            }
        }
    }
}


// ---------------------------------------------------------------------------------------------------------------
// fp64 step kernel, SEMI-RECOMPUTE coefficient supply (H1b variant (b), see setup_kernels.cuh): same phases and
// the same substep<1> arithmetic as step_kernel_f64_tma, but the 16 coefficient planes are replaced by one
// isig = 1/Sigma plane per point family plus 1-D tables, and the 8 folded coefficients of a point are rebuilt in
// registers (17 extra flops per sub-step).  TMA loads per block: u tile, isig tile (half points), isig tile
// (integer points), r-table slab (half points, 16 x (TI+2)), r-table slab (integer points, 16 x TI).
struct RcParams {
    const double* th;      // [3][n_theta]: sin^2, cos, Tth = (m + s cos)^2 / sin^2 - s
};

template <int TI, int TJ> struct RcGeom {
    static constexpr int UC = TI + 4, UR = TJ + 4, HC = TI + 1, HR = TJ + 2, CC = TI + 2, NT = 16;
    static constexpr int a128(int v) { return (v + 127) / 128 * 128; }
    static constexpr int US_B = a128(4 * UR * UC * 8);
    static constexpr int ISH_B = a128(HR * CC * 8);
    static constexpr int ISI_B = a128(TJ * TI * 8);
    static constexpr int RTH_B = a128(NT * CC * 8);
    static constexpr int RTI_B = a128(NT * TI * 8);
    static constexpr int HS_B = a128(4 * HR * HC * 8);
    static constexpr int TOTAL = US_B + ISH_B + ISI_B + RTH_B + RTI_B + HS_B + 128;
};

// 1/sqrt(x) for variant (c): hardware rsqrt (<= 1 ulp) plus one FMA Newton step, so the result is within ~0.5 ulp like
// the stored 1/Sigma plane (the coefficient error is systematic and accumulates linearly over a long run)
__device__ __forceinline__ double rsqrt_refined(double x) {
    double y = rsqrt(x);
    double e = fma(-(x * y), y, 1.0);
    return fma(0.5 * y, e, y);
}

struct RcCoef {
    double c[8];
    __device__ __forceinline__ R1 get(int q) const { R1 r; r.x[0] = c[q]; return r; }
};
// rt: pointer to this point's column in the r-table slab, consecutive tables `stride` apart
__device__ __forceinline__ void rc_eval(RcCoef& o, double isig, const double* rt, int stride, double s2, double cs,
                                        double tth) {
    const double q = isig * isig;
    o.c[0] = rt[0] * isig;
    o.c[1] = rt[1 * stride] * q;
    o.c[2] = fma(rt[3 * stride], cs, rt[2 * stride]) * q;
    o.c[3] = q * fma(-(q * s2), rt[6 * stride], fma(rt[4 * stride], isig, rt[5 * stride]));
    o.c[4] = q * fma(fma(rt[8 * stride], cs, rt[7 * stride]), isig, rt[9 * stride]);
    o.c[5] = q * fma(rt[10 * stride], tth, rt[11 * stride]);
    o.c[6] = q * rt[12 * stride];
    o.c[7] = q * rt[13 * stride];
}

// FULL = H1b variant (c), full recompute: the 1/Sigma planes are not read either; 1/Sigma = rsqrt(R^2 - a^2 Delta sin^2 theta)
// (Eq. 7) per point and sub-step from the two spare r-tables (R^2, a^2 Delta) and sin^2 theta.  State-only
// HBM traffic: 64 B/update.  fp64 rsqrt of a sum of two rounded table entries instead of a quad-double evaluation rounded
// once: the coefficients differ from the stored planes by a few more ulps (tested), no cancellation (a^2 Delta sin^2 <= 0.06 R^2).
template <int TI, int TJ, bool FULL>
__global__ void __launch_bounds__(256) step_kernel_f64_rc(const __grid_constant__ CUtensorMap tm_u,
                                                         const __grid_constant__ CUtensorMap tm_ish,
                                                         const __grid_constant__ CUtensorMap tm_isi,
                                                         const __grid_constant__ CUtensorMap tm_rth,
                                                         const __grid_constant__ CUtensorMap tm_rti, StepParams P,
                                                         RcParams Q) {
    using G = RcGeom<TI, TJ>;
    constexpr int UC = G::UC, UR = G::UR, HC = G::HC, HR = G::HR, CC = G::CC, NT = G::NT;
    extern __shared__ __align__(128) unsigned char raw[];
    __shared__ __align__(8) uint64_t bar[3];
    __shared__ double tht[4][TJ + 2];           // cj, sin^2, cos, Tth for rows j0-1 .. j0+TJ (shared-memory, not L1, latency)
    unsigned char* base = raw;      // __align__(128) on the extern array is honoured; no integer round trip, so the
                                    // compiler keeps these pointers in the shared state space (LDS/STS, not generic LD/ST)
    double* us = (double*)base;
    double* ish = (double*)(base + G::US_B);
    double* isi = (double*)(base + G::US_B + G::ISH_B);
    double* rth = (double*)(base + G::US_B + G::ISH_B + G::ISI_B);
    double* rti = (double*)(base + G::US_B + G::ISH_B + G::ISI_B + G::RTH_B);
    double* hs = (double*)(base + G::US_B + G::ISH_B + G::ISI_B + G::RTH_B + G::RTI_B);
    const int i0 = blockIdx.x * TI, j0 = blockIdx.y * TJ;
    const int nt = P.n_theta, nr = P.n_r;
    const int tid = threadIdx.x;

    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        mbar_init(&bar[2], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(&bar[2], (FULL ? 0 : HR * CC * 8) + NT * CC * 8);
        if (!FULL) tma_load_3d(ish, &tm_ish, i0 - 2, j0 - 1, 0, &bar[2]);
        tma_load_3d(rth, &tm_rth, i0 - 2, 0, 0, &bar[2]);
    }
    if (tid < 4 * (TJ + 2)) {
        int t = tid / (TJ + 2), r = tid - t * (TJ + 2);
        int j = min(max(j0 - 1 + r, 0), P.n_theta - 1);
        tht[t][r] = (t == 0) ? __ldg(P.cj + j) : __ldg(Q.th + (t - 1) * P.n_theta + j);
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (tid == 0) {
        mbar_expect_tx(&bar[0], 4 * UR * UC * 8);
        tma_load_3d(us, &tm_u, i0 - 2, j0 - 2, 0, &bar[0]);
        mbar_expect_tx(&bar[1], (FULL ? 0 : TJ * TI * 8) + NT * TI * 8);
        if (!FULL) tma_load_3d(isi, &tm_isi, i0, j0, 0, &bar[1]);
        tma_load_3d(rti, &tm_rti, i0, 0, 0, &bar[1]);
    }
    __syncthreads();
    mbar_wait(&bar[0], 0);
    mbar_wait(&bar[2], 0);

    CTile<UR, UC> ut{us, j0 - 2};
#pragma unroll
    for (int k = 0; k < (HR * HC + 255) / 256; ++k) {
        int idx = tid + k * 256;
        if (idx < HR * HC) {
            int tr = idx / HC, tc = idx - tr * HC;
            int ih = i0 - 1 + tc, jh = j0 - 1 + tr;
            if (ih >= 0 && ih <= nr - 2 && jh >= 0 && jh < nt) {
                int rm = jh - 1, rp = jh + 1;
                double sm = 1.0, sp = 1.0;
                if (rm < 0) { rm = 0; sm = P.sigma; }
                if (rp >= nt) { rp = nt - 1; sp = P.sigma; }
                R1 cjv;
                cjv.x[0] = tht[0][tr];
                RcCoef cf;
                const double is_h = FULL ? rsqrt_refined(fma(-rth[15 * CC + tc + 1], tht[1][tr], rth[14 * CC + tc + 1])) : ish[tr * CC + tc + 1];
                rc_eval(cf, is_h, rth + tc + 1, CC, tht[1][tr], tht[2][tr], tht[3][tr]);
                R1 out[4];
                substep<1>(ut, jh, rm, rp, sm, sp, tc + 1, tc + 2, cf, cjv, P.tq_half, true, out, out);
#pragma unroll
                for (int c = 0; c < 4; ++c) hs[c * HR * HC + tr * HC + tc] = out[c].x[0];
            }
        }
    }
    __syncthreads();
    mbar_wait(&bar[1], 0);

    CTile<HR, HC> ht{hs, j0 - 1};
    const int lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int k = 0; k < (TJ * TI + 255) / 256; ++k) {
        int tr, tc;
        if (TI == 32) { tr = warp + 8 * k; tc = lane; }
        else { int idx = tid + k * 256; tr = idx / TI; tc = idx - tr * TI; }
        int i = i0 + tc, j = j0 + tr;
        if (tr >= TJ || i >= nr || j >= nt) continue;
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
            cjv.x[0] = tht[0][tr + 1];
            RcCoef cf;
            const double is_i = FULL ? rsqrt_refined(fma(-rti[15 * TI + tc], tht[1][tr + 1], rti[14 * TI + tc])) : isi[tr * TI + tc];
            rc_eval(cf, is_i, rti + tc, TI, tht[1][tr + 1], tht[2][tr + 1], tht[3][tr + 1]);
            substep<1>(ht, j, rm, rp, sm, sp, tc, tc + 1, cf, cjv, P.tq_full, false, bs, out);
        }
        long g = (long)j * P.pitch + i;
#pragma unroll
        for (int c = 0; c < 4; ++c) P.u_out[(long)c * P.plane + g] = out[c].x[0];
        if (P.obs_raw != nullptr) {
            int di = i - P.oi, dj = j - P.oj;
            if ((di == 0 || di == 1) && (dj == 0 || dj == 1)) {
                long ks = *P.step_base + P.step_off;
                if (ks < P.obs_cap) {
                    double* o = P.obs_raw + ((ks * 4 + (dj * 2 + di)) * 4);
#pragma unroll
                    for (int c = 0; c < 4; ++c) o[c] = out[c].x[0];
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// fp64 column kernel for the 10th-order theta operator (NEXT-1) with TMA staging and the semi-recompute coefficient
// supply: a block owns TI columns x all N_theta (<= 256) rows.  Five TMA loads per block (u tile, two 1/Sigma tiles,
// two r-table slabs), sig_Phi staged once in shared memory, compile-time column counts.
template <int COLS> struct RTile {              // run-time row count, compile-time column count
    const double* p;
    int rows;
    __device__ __forceinline__ R1 get(int c, int row, int col) const {
        R1 r;
        r.x[0] = p[(c * rows + row) * COLS + col];
        return r;
    }
};

template <int TI> struct ColGeom {
    static constexpr int UC = TI + 4, HC = TI + 1, CC = TI + 2, NT = 16;
    static size_t a128(size_t v) { return (v + 127) / 128 * 128; }
    static size_t total(int nt) {
        return a128((size_t)4 * nt * UC * 8) + a128((size_t)nt * CC * 8) + a128((size_t)nt * TI * 8) + a128((size_t)NT * CC * 8) +
               a128((size_t)NT * TI * 8) + a128((size_t)4 * nt * HC * 8) + a128((size_t)2 * nt * HC * 8) + 128;
    }
    static size_t total_run(int nt) {          // row-run kernel: no staged sig tile, + the four theta tables
        return a128((size_t)4 * nt * UC * 8) + a128((size_t)nt * CC * 8) + a128((size_t)nt * TI * 8) + a128((size_t)NT * CC * 8) +
               a128((size_t)NT * TI * 8) + a128((size_t)4 * nt * HC * 8) + a128((size_t)4 * nt * 8) + 128;
    }
};

template <int TI>
__global__ void __launch_bounds__(256) step_kernel_f64_col_tma(const __grid_constant__ CUtensorMap tm_u,
                                                              const __grid_constant__ CUtensorMap tm_ish,
                                                              const __grid_constant__ CUtensorMap tm_isi,
                                                              const __grid_constant__ CUtensorMap tm_rth,
                                                              const __grid_constant__ CUtensorMap tm_rti, StepParams P,
                                                              RcParams Q, ThetaWeights W) {
    using G = ColGeom<TI>;
    constexpr int UC = G::UC, HC = G::HC, CC = G::CC, NT = G::NT;
    extern __shared__ __align__(128) unsigned char raw[];
    __shared__ __align__(8) uint64_t bar[2];
    const int nt = P.n_theta, nr = P.n_r;
    auto a128 = [](size_t v) { return (v + 127) / 128 * 128; };
    unsigned char* base = raw;      // __align__(128) on the extern array is honoured; no integer round trip, so the
                                    // compiler keeps these pointers in the shared state space (LDS/STS, not generic LD/ST)
    double* us = (double*)base;                      base += a128((size_t)4 * nt * UC * 8);
    double* ish = (double*)base;                     base += a128((size_t)nt * CC * 8);
    double* isi = (double*)base;                     base += a128((size_t)nt * TI * 8);
    double* rth = (double*)base;                     base += a128((size_t)NT * CC * 8);
    double* rti = (double*)base;                     base += a128((size_t)NT * TI * 8);
    double* hs = (double*)base;                      base += a128((size_t)4 * nt * HC * 8);
    double* ss = (double*)base;
    const int i0 = blockIdx.x * TI;
    const int tid = threadIdx.x;

    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&bar[0], (4 * nt * UC + nt * CC + NT * CC) * 8);
        tma_load_3d(us, &tm_u, i0 - 2, 0, 0, &bar[0]);
        tma_load_3d(ish, &tm_ish, i0 - 2, 0, 0, &bar[0]);
        tma_load_3d(rth, &tm_rth, i0 - 2, 0, 0, &bar[0]);
        mbar_expect_tx(&bar[1], (nt * TI + NT * TI) * 8);
        tma_load_3d(isi, &tm_isi, i0, 0, 0, &bar[1]);
        tma_load_3d(rti, &tm_rti, i0, 0, 0, &bar[1]);
    }
    mbar_wait(&bar[0], 0);

    RTile<UC> ut{us, nt};
    // sig_Phi = Phi(i+1) + Phi(i) at the TI+1 half points (u tile column of half point tc: tc+1 and tc+2)
    for (int idx = tid; idx < 2 * nt * HC; idx += 256) {
        int tc = idx % HC, rest = idx / HC;
        ss[rest * HC + tc] = us[rest * UC + tc + 2] + us[rest * UC + tc + 1];
    }
    __syncthreads();
    RTile<HC> st1{ss, nt};
    for (int idx = tid; idx < nt * HC; idx += 256) {
        int tr = idx / HC, tc = idx - tr * HC;
        int ih = i0 - 1 + tc;
        if (ih < 0 || ih > nr - 2) continue;
        R1 cjv;
        cjv.x[0] = __ldg(P.cj + tr);
        RcCoef cf;
        rc_eval(cf, ish[tr * CC + tc + 1], rth + tc + 1, CC, __ldg(Q.th + tr), __ldg(Q.th + nt + tr), __ldg(Q.th + 2 * nt + tr));
        R1 out[4];
        substep_wide<1>(ut, st1, tc, tr, nt, P.sigma, tc + 1, tc + 2, cf, cjv, W, P.tq_half, true, out, out);
#pragma unroll
        for (int c = 0; c < 4; ++c) hs[(c * nt + tr) * HC + tc] = out[c].x[0];
    }
    __syncthreads();
    RTile<HC> ht{hs, nt};
    for (int idx = tid; idx < 2 * nt * TI; idx += 256) {
        int tc = idx % TI, rest = idx / TI;
        ss[rest * TI + tc] = hs[rest * HC + tc + 1] + hs[rest * HC + tc];
    }
    mbar_wait(&bar[1], 0);
    __syncthreads();
    RTile<TI> st2{ss, nt};
    for (int idx = tid; idx < nt * TI; idx += 256) {
        int tr = idx / TI, tc = idx - tr * TI;
        int i = i0 + tc, j = tr;
        if (i >= nr) continue;
        R1 out[4];
        if (i == 0 || i == nr - 1) {
#pragma unroll
            for (int c = 0; c < 4; ++c) out[c].x[0] = 0.0;
        } else {
            R1 bs[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) bs[c] = ut.get(c, j, tc + 2);
            R1 cjv;
            cjv.x[0] = __ldg(P.cj + j);
            RcCoef cf;
            rc_eval(cf, isi[tr * TI + tc], rti + tc, TI, __ldg(Q.th + j), __ldg(Q.th + nt + j), __ldg(Q.th + 2 * nt + j));
            substep_wide<1>(ht, st2, tc, j, nt, P.sigma, tc, tc + 1, cf, cjv, W, P.tq_full, false, bs, out);
        }
        long g = (long)j * P.pitch + i;
#pragma unroll
        for (int c = 0; c < 4; ++c) P.u_out[(long)c * P.plane + g] = out[c].x[0];
        if (P.obs_raw != nullptr) {
            int di = i - P.oi, dj = j - P.oj;
            if ((di == 0 || di == 1) && (dj == 0 || dj == 1)) {
                long ks = *P.step_base + P.step_off;
                if (ks < P.obs_cap) {
                    double* o = P.obs_raw + ((ks * 4 + (dj * 2 + di)) * 4);
#pragma unroll
                    for (int c = 0; c < 4; ++c) o[c] = out[c].x[0];
                }
            }
        }
    }
}


// ---------------------------------------------------------------------------------------------------------------
// Row-run variant of the 10th-order fp64 column kernel (round 2).  Same tiles, same TMA loads and the same arithmetic
// in the same order as step_kernel_f64_col_tma, but a thread owns a RUN of R consecutive theta rows of one column instead
// of single points: the 11-point stencil's window of sig_Phi (R + 10 rows x 2 components) is loaded from shared memory once
// per run and kept in registers (2 (R + 10) / R shared-memory loads per point instead of 22), and the 14 r-table entries of
// the column are loaded once per run instead of once per point.  ncu on the point-per-thread kernel: 113 shared-memory
// loads per update, shared-memory scoreboard 2.2-2.5 stalls per issued instruction.
template <int TI, int R, int NTHR, int MINB>
__global__ void __launch_bounds__(NTHR, MINB) step_kernel_f64_col_run(const __grid_constant__ CUtensorMap tm_u,
                                                               const __grid_constant__ CUtensorMap tm_ish,
                                                               const __grid_constant__ CUtensorMap tm_isi,
                                                               const __grid_constant__ CUtensorMap tm_rth,
                                                               const __grid_constant__ CUtensorMap tm_rti, StepParams P,
                                                               RcParams Q, ThetaWeights W) {
    using G = ColGeom<TI>;
    constexpr int UC = G::UC, HC = G::HC, CC = G::CC, NT = G::NT, WIN = R + 10;
    extern __shared__ __align__(128) unsigned char raw[];
    __shared__ __align__(8) uint64_t bar[2];
    const int nt = P.n_theta, nr = P.n_r;
    auto a128 = [](size_t v) { return (v + 127) / 128 * 128; };
    unsigned char* base = raw;
    double* us = (double*)base;                      base += a128((size_t)4 * nt * UC * 8);
    double* ish = (double*)base;                     base += a128((size_t)nt * CC * 8);
    double* isi = (double*)base;                     base += a128((size_t)nt * TI * 8);
    double* rth = (double*)base;                     base += a128((size_t)NT * CC * 8);
    double* rti = (double*)base;                     base += a128((size_t)NT * TI * 8);
    double* hs = (double*)base;                      base += a128((size_t)4 * nt * HC * 8);
    double* tht = (double*)base;                     // [4][nt]: cj, sin^2, cos, Tth
    const int i0 = blockIdx.x * TI;
    const int tid = threadIdx.x;
    const double sigma = P.sigma;

    if (tid == 0) {
        mbar_init(&bar[0], 1);
        mbar_init(&bar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&bar[0], (4 * nt * UC + nt * CC + NT * CC) * 8);
        tma_load_3d(us, &tm_u, i0 - 2, 0, 0, &bar[0]);
        tma_load_3d(ish, &tm_ish, i0 - 2, 0, 0, &bar[0]);
        tma_load_3d(rth, &tm_rth, i0 - 2, 0, 0, &bar[0]);
        mbar_expect_tx(&bar[1], (nt * TI + NT * TI) * 8);
        tma_load_3d(isi, &tm_isi, i0, 0, 0, &bar[1]);
        tma_load_3d(rti, &tm_rti, i0, 0, 0, &bar[1]);
    }
    for (int k = tid; k < 4 * nt; k += NTHR) tht[k] = (k < nt) ? __ldg(P.cj + k) : __ldg(Q.th + (k - nt));
    __syncthreads();
    mbar_wait(&bar[0], 0);

    // sig_Phi = Phi(i+1) + Phi(i) is formed on the fly while a run's window is loaded (no staging pass, no barrier)

    const int ngroups = (nt + R - 1) / R;
    // the window of one component: rows j0-5 .. j0+R+4 of column `col` of a [2][nt][COLS] sig tile, polar ghosts mirrored
    // with sign sigma (f_{-k} = sigma f_{k-1}, f_{N-1+k} = sigma f_{N-k})
    auto load_window = [&](const double* tile, int cols, int col, int j0, auto& win) {
        constexpr int WN = sizeof(win[0]) / sizeof(double);
#pragma unroll
        for (int w = 0; w < WN; ++w) {
            int rr = j0 - 5 + w;
            double sg = 1.0;
            if (rr < 0) { rr = -rr - 1; sg = sigma; }
            if (rr >= nt) { rr = 2 * nt - 1 - rr; sg = sigma; }
            rr = min(max(rr, 0), nt - 1);                      // rows of a partial last run that nothing uses
#pragma unroll
            for (int c = 0; c < 2; ++c) win[c][w] = sg * (tile[(c * nt + rr) * cols + col + 1] + tile[(c * nt + rr) * cols + col]);
        }
    };
    // Lambda at window position w (row j0 + w - 5 ... the centre is win[.][w]), same summation order as substep_wide
    auto lam_at = [&](const auto& win, int c, int w, double cj) {
        double s2 = W.wd[0][0] * win[c][w];
        double s1 = 0.0;
#pragma unroll
        for (int k = 1; k <= 5; ++k) {
            const double up = win[c][w + k], dn = win[c][w - k];
            s2 = s2 + W.wd[k][0] * (up + dn);
            s1 = s1 + W.wc[k - 1][0] * (up - dn);
        }
        return s2 + cj * (s1 * 2.0);
    };

    // ---- half step, Eq. (13): a task = (half-point column tc, run of RR rows starting at j0)
    auto half_task = [&](auto RRc, int tc, int j0) {
        constexpr int RR = decltype(RRc)::value;
        const int ih = i0 - 1 + tc;
        if (ih < 0 || ih > nr - 2) return;
        double win[2][RR + 10], rt[14];
        load_window(us, UC, tc + 1, j0, win);
#pragma unroll
        for (int q = 0; q < 14; ++q) rt[q] = rth[q * CC + tc + 1];
#pragma unroll
        for (int r = 0; r < RR; ++r) {
            const int j = j0 + r;
            if (j < nt) {
                R1 sg[4], dl[4], lam[2], out[4];
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const double lo = us[(c * nt + j) * UC + tc + 1], hi = us[(c * nt + j) * UC + tc + 2];
                    sg[c].x[0] = (c < 2) ? win[c][r + 5] : hi + lo;
                    dl[c].x[0] = hi - lo;
                }
                const double cj = tht[j];
#pragma unroll
                for (int c = 0; c < 2; ++c) lam[c].x[0] = lam_at(win, c, r + 5, cj);
                RcCoef cf;
                rc_eval(cf, ish[j * CC + tc + 1], rt, 1, tht[nt + j], tht[2 * nt + j], tht[3 * nt + j]);
                substep_core<1, RTile<UC>, RcCoef>(sg, dl, lam, cf, P.tq_half, true, out, out);
#pragma unroll
                for (int c = 0; c < 4; ++c) hs[(c * nt + j) * HC + tc] = out[c].x[0];
            }
        }
    };
    // as many columns as one pass of the block covers go in runs of R rows; the columns that would need a second pass
    // (the 17th half-step column of a 16-column tile at N_theta = 64) go row by row, spread over the threads again
    const int main_cols = (ngroups <= NTHR) ? min(HC, NTHR / ngroups) : 0;
    for (int task = tid; task < main_cols * ngroups; task += NTHR) {
        const int g = task / main_cols, tc = task - g * main_cols;
        half_task(std::integral_constant<int, R>{}, tc, g * R);
    }
    for (int task = tid; task < (HC - main_cols) * nt; task += NTHR) {
        const int j = task / (HC - main_cols), tc = main_cols + task - j * (HC - main_cols);
        half_task(std::integral_constant<int, 1>{}, tc, j);
    }
    mbar_wait(&bar[1], 0);
    __syncthreads();

    // ---- full step, Eq. (14), radial Dirichlet columns, observer nodes: tasks = (output column tc, run of R rows)
    for (int task = tid; task < TI * ngroups; task += NTHR) {
        const int g = task / TI, tc = task - g * TI, j0 = g * R;
        const int i = i0 + tc;
        if (i >= nr) continue;
        const bool wall = (i == 0 || i == nr - 1);
        double win[2][WIN], rt[14];
        load_window(hs, HC, tc, j0, win);
#pragma unroll
        for (int q = 0; q < 14; ++q) rt[q] = rti[q * TI + tc];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int j = j0 + r;
            if (j < nt) {
                R1 out[4];
                if (wall) {
#pragma unroll
                    for (int c = 0; c < 4; ++c) out[c].x[0] = 0.0;
                } else {
                    R1 sg[4], dl[4], lam[2], bs[4];
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const double lo = hs[(c * nt + j) * HC + tc], hi = hs[(c * nt + j) * HC + tc + 1];
                        sg[c].x[0] = (c < 2) ? win[c][r + 5] : hi + lo;
                        dl[c].x[0] = hi - lo;
                        bs[c].x[0] = us[(c * nt + j) * UC + tc + 2];
                    }
                    const double cj = tht[j];
#pragma unroll
                    for (int c = 0; c < 2; ++c) lam[c].x[0] = lam_at(win, c, r + 5, cj);
                    RcCoef cf;
                    rc_eval(cf, isi[j * TI + tc], rt, 1, tht[nt + j], tht[2 * nt + j], tht[3 * nt + j]);
                    substep_core<1, RTile<UC>, RcCoef>(sg, dl, lam, cf, P.tq_full, false, bs, out);
                }
                const long gidx = (long)j * P.pitch + i;
#pragma unroll
                for (int c = 0; c < 4; ++c) P.u_out[(long)c * P.plane + gidx] = out[c].x[0];
                if (P.obs_raw != nullptr) {
                    const int di = i - P.oi, dj = j - P.oj;
                    if ((di == 0 || di == 1) && (dj == 0 || dj == 1)) {
                        const long ks = *P.step_base + P.step_off;
                        if (ks < P.obs_cap) {
                            double* o = P.obs_raw + ((ks * 4 + (dj * 2 + di)) * 4);
#pragma unroll
                            for (int c = 0; c < 4; ++c) o[c] = out[c].x[0];
                        }
                    }
                }
            }
        }
    }
}

}  // namespace tk
