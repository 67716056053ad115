// fp64 step kernel, "column march" (round 2; the default fp64 path).  Same iteration as every other step kernel --
// half step Eq. (13) + full step Eq. (14), radial Dirichlet rows and polar ghosts,
// observer nodes in one launch -- with the SEMI-RECOMPUTE coefficient supply of H1b variant (b)
// (one 1/Sigma plane per point family + 1-D tables; 64 + 16 = 80 B of HBM traffic per update), but organised so that
// almost every instruction is arithmetic:
//   * a WARP owns a strip of 30 output columns and marches down theta; lane l holds column 30 s - 1 + l.  Rows of u and
//     of the two 1/Sigma planes stream through a private 16-row shared-memory ring, filled eleven rows ahead by 8-byte
//     asynchronous copies (cp.async, one commit group per row), so HBM latency is covered by the ring, not by
//     occupancy, and each value is read from global memory exactly once per warp (coalesced 256-byte rows);
//   * the half-step field never leaves registers: lane l computes h at (30 s - 1/2 + l, j), the full step at column
//     30 s + l takes h(i - 1/2) from itself and h(i + 1/2) from lane l + 1 by shuffle.  No barriers, warps are
//     independent;
//   * sig_Phi = Phi_hi + Phi_lo is formed once per row and kept in a four-row register window for the angular
//     operator Lambda (the tile kernels form it three times and read the tile six times per sub-step); the three
//     stages of an iteration (sums of row r, half step of row r - 2, full step of row r - 4) are mutually independent,
//     and four iterations on rows away from the poles form ONE basic block;
//   * the 28 r-only table entries of a column (rc_eval) live in registers, fetched once per work unit;
//   * the grid is persistent: a work unit is (strip, chunk of theta rows); the host picks the chunk length so that the
//     units fill the resident warps in whole rounds, and warp w takes units w, w + W, ... in chunk-major order, so
//     neighbouring strips are swept at the same time (the 32-byte sectors they share hit in L2).  A chunk that starts
//     inside a column pays a two-row theta halo (redundant half steps).
// Redundant work in r*: 32 lanes load, 31 compute half steps, 30 produce outputs.
#pragma once
#include <type_traits>

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
    int n_strips;                   // ceil(n_r / 30)
    int chunk_rows;                 // theta rows per work unit
    int n_units;                    // n_strips * ceil(n_theta / chunk_rows); unit u = chunk * n_strips + strip
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

// per-warp ring of staged rows in shared memory: [MARCH_RING rows][6 planes: u x 4, 1/Sigma half, 1/Sigma integer][32 lanes]
constexpr int MARCH_RING = 16;      // rows resident per warp (power of two: slot = row & 15)
constexpr int MARCH_PF = 11;        // rows requested ahead of the one being consumed (stage C still reads row r - 4)
constexpr int MARCH_ROW = 6 * 32;   // doubles per ring row

// (cp_async8 / cp_async_commit / cp_async_wait: step_kernel.cuh)

constexpr size_t march_smem_bytes(int n_theta) {
    return ((size_t)4 * n_theta + (size_t)MARCH_WARPS * MARCH_RING * MARCH_ROW + 8) * sizeof(double);
}

template <int MINB>                  // blocks per SM the register budget is cut for
__global__ void __launch_bounds__(32 * MARCH_WARPS, MINB) step_kernel_f64_march(StepParams P, MarchParams Q) {
    extern __shared__ double sm[];
    // programmatic dependent launch ("pdl" option): the next step's blocks may be scheduled as this step's blocks exit and
    // run their set-up (theta tables, ring clearing, r-table registers); they wait below before touching the state
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int nt = P.n_theta, nr = P.n_r;
    double* tht = sm;                                                // [4][nt]: cj, sin^2, cos, Tth
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // lane 31 reads element lane + 1 = the first element of the next plane row (or of the 8 spare doubles behind the last
    // ring): finite data that only feeds values which are never stored
    double* ring = sm + 4 * nt + warp * (MARCH_RING * MARCH_ROW) + lane;
    for (int k = threadIdx.x; k < 4 * nt; k += blockDim.x) tht[k] = (k < nt) ? __ldg(P.cj + k) : __ldg(Q.th + (k - nt));
    if (threadIdx.x < 8) sm[4 * nt + MARCH_WARPS * MARCH_RING * MARCH_ROW + threadIdx.x] = 0.0;
    for (int k = lane; k < MARCH_RING * MARCH_ROW; k += 32) ring[k - lane] = 0.0;
    __syncthreads();
    const double sigma = P.sigma;
    // 32-bit element offsets (the host checks 4 * plane < 2^31): one IMAD.WIDE per address instead of 64-bit multiplies
    const unsigned pitch = (unsigned)P.pitch, plane = (unsigned)P.plane;
    // read through lane 0 so that the compiler knows the warp's work range is warp-uniform
    const int gw = __shfl_sync(0xffffffffu, (int)(blockIdx.x * MARCH_WARPS + warp), 0);
    const int n_warps = (int)gridDim.x * MARCH_WARPS;

    for (int unit = gw; unit < Q.n_units; unit += n_warps) {
        const int chunk = unit / Q.n_strips;
        const int s = unit - chunk * Q.n_strips;
        const int ja = chunk * Q.chunk_rows;
        const int jb = min(nt, ja + Q.chunk_rows);

        const int cu = MARCH_W * s - 1 + lane;                      // this lane's column (lo of its half point)
        const int ci = cu + 1;                                      // its output column (lanes 0..29)
        const bool lo_ok = cu >= 0 && cu < nr;
        const bool h_ok = cu >= 0 && ci < nr;                       // half point (cu, cu + 1) exists
        const bool c_ok = ci < nr;
        const bool i_ok = c_ok && lane < MARCH_W;
        const bool interior = i_ok && ci > 0 && ci < nr - 1;
        const int cuc = min(max(cu, 0), nr - 1), cic = min(ci, nr - 1);       // clamped: a valid address for the masked copies
        // warp-uniform: this strip holds an observer column
        const bool obs_strip = P.obs_raw != nullptr && P.oi + 1 >= MARCH_W * s && P.oi < MARCH_W * (s + 1);
        // r-only table entries of this lane's half point and output column (registers, fetched once per unit)
        double rth[MARCH_NRT], rti[MARCH_NRT];
#pragma unroll
        for (int q = 0; q < MARCH_NRT; ++q) {
            rth[q] = h_ok ? __ldg(Q.rt + ((16 + q) * pitch + cuc)) : 0.0;
            rti[q] = c_ok ? __ldg(Q.rt + (q * pitch + cic)) : 0.0;
        }

        const int ha = max(ja - 1, 0), hb = min(jb + 1, nt);        // half-step rows
        const int ua = max(ha - 1, 0), ub = min(hb + 1, nt);        // u rows
        __syncwarp();                                               // the previous unit's ring reads are done
        // request row r into ring slot r & 15: six 8-byte asynchronous copies per lane (masked beyond the last row needed
        // and outside the grid), one commit group per row
        auto request = [&](int r) {
            const bool inr = r < ub;
            double* dst = ring + (r & (MARCH_RING - 1)) * MARCH_ROW;
            const unsigned row = (unsigned)min(r, nt - 1) * pitch;
#pragma unroll
            for (int c = 0; c < 4; ++c) cp_async8(dst + c * 32, P.u_in + (row + (unsigned)cuc + c * plane), inr && lo_ok);
            cp_async8(dst + 4 * 32, Q.isig_h + (row + (unsigned)cuc), inr && h_ok);
            cp_async8(dst + 5 * 32, Q.isig_i + (row + (unsigned)cic), inr && c_ok);
            cp_async_commit();
        };
        asm volatile("griddepcontrol.wait;" ::: "memory");          // u^n (written by the previous step) is complete and visible
#pragma unroll 1
        for (int r = ua; r < ua + MARCH_PF; ++r) request(r);

        // rolling register windows, slot = (row - ua) mod 4
        double SU[4][2];                                             // sig_Phi of u
        double SH[4][2], SHP[4][2], DH[4][4];                        // sig_Phi, sig_Pi, del of the half-step field
#pragma unroll
        for (int a = 0; a < 4; ++a) {
#pragma unroll
            for (int c = 0; c < 4; ++c) DH[a][c] = 0.0;
#pragma unroll
            for (int c = 0; c < 2; ++c) SU[a][c] = SH[a][c] = SHP[a][c] = 0.0;
        }
        // ---- A: sig_Phi of row r
        auto stage_a = [&](int k, int r) {
            const double* w = ring + (r & (MARCH_RING - 1)) * MARCH_ROW;
#pragma unroll
            for (int c = 0; c < 2; ++c) SU[k][c] = w[c * 32 + 1] + w[c * 32];
        };
        // ---- B: half step at row q = r - 2, Eq. (13); slots: q - 1 -> k + 1, q -> k + 2, q + 1 -> k + 3 (mod 4).
        //      fast = the row is known (at compile time of this call) to lie away from the poles
        auto stage_b = [&](auto fast, int k, int q) {
            const double* w = ring + (q & (MARCH_RING - 1)) * MARCH_ROW;
            double sg[4], dl[4], lam[2], base[4], h[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const double lo = w[c * 32], hi = w[c * 32 + 1];
                sg[c] = hi + lo;
                dl[c] = hi - lo;
                base[c] = 0.5 * sg[c];
            }
            const double cjq = tht[q];
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                double dn = SU[(k + 1) % 4][c], up = SU[(k + 3) % 4][c];
                if (!decltype(fast)::value) {                        // polar ghosts f_{-1} = sigma f_0, f_N = sigma f_{N-1}
                    if (q == 0) dn = sigma * sg[c];
                    if (q + 1 == nt) up = sigma * sg[c];
                }
                lam[c] = lam_op(up, dn, sg[c], cjq);
            }
            RcCoef cf;
            rc_eval(cf, w[4 * 32], rth, 1, tht[nt + q], tht[2 * nt + q], tht[3 * nt + q]);
            march_core(sg, dl, lam, cf, P.tq_half, base, h);
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const double hn = shfl_down1(h[c]);                  // h at (ci + 1/2, q)
                DH[(k + 2) % 4][c] = hn - h[c];
                if (c < 2) SH[(k + 2) % 4][c] = hn + h[c]; else SHP[(k + 2) % 4][c - 2] = hn + h[c];
            }
        };
        // ---- C: full step at row q2 = r - 4, Eq. (14); radial Dirichlet columns; observer nodes
        //      slots: q2 - 1 -> k + 3, q2 -> k, q2 + 1 -> k + 1 (mod 4)
        auto stage_c = [&](auto fast, int k, int q2) {
            const double* w = ring + (q2 & (MARCH_RING - 1)) * MARCH_ROW;
            double sg[4] = {SH[k][0], SH[k][1], SHP[k][0], SHP[k][1]};
            double lam[2], out[4], base[4];
            const double cjq = tht[q2];
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                double dn = SH[(k + 3) % 4][c], up = SH[(k + 1) % 4][c];
                if (!decltype(fast)::value) {
                    if (q2 == 0) dn = sigma * sg[c];
                    if (q2 + 1 == nt) up = sigma * sg[c];
                }
                lam[c] = lam_op(up, dn, sg[c], cjq);
            }
#pragma unroll
            for (int c = 0; c < 4; ++c) base[c] = w[c * 32 + 1];    // u^n at column ci
            RcCoef cf;
            rc_eval(cf, w[5 * 32], rti, 1, tht[nt + q2], tht[2 * nt + q2], tht[3 * nt + q2]);
            march_core(sg, DH[k], lam, cf, P.tq_full, base, out);
            const unsigned go = (unsigned)q2 * pitch + (unsigned)cic;
            if (decltype(fast)::value) {                             // interior strip: every output column is an interior column
                if (lane < MARCH_W) {
#pragma unroll
                    for (int c = 0; c < 4; ++c) P.u_out[go + c * plane] = out[c];
                }
            } else {
                if (interior) {
#pragma unroll
                    for (int c = 0; c < 4; ++c) P.u_out[go + c * plane] = out[c];
                } else if (i_ok) {                                   // radial Dirichlet columns
#pragma unroll
                    for (int c = 0; c < 4; ++c) P.u_out[go + c * plane] = out[c] = 0.0;
                }
                if (obs_strip && (unsigned)(q2 - P.oj) < 2u) {       // warp-uniform, rare
                    const int di = ci - P.oi, dj = q2 - P.oj;
                    const long ks = *P.step_base + P.step_off;
                    if (i_ok && (di == 0 || di == 1) && ks < P.obs_cap) {
                        double* o = P.obs_raw + ((ks * 4 + (dj * 2 + di)) * 4);
#pragma unroll
                        for (int c = 0; c < 4; ++c) o[c] = out[c];
                    }
                }
            }
        };

        // interior strip without observer columns: all 32 lanes hold grid columns, outputs are interior columns
        const bool strip_fast = !obs_strip && s >= 1 && MARCH_W * s + 31 <= nr - 1;
        for (int rb = ua; rb <= jb + 3; rb += 4) {
            // the four iterations of this block run all three stages on rows away from the poles: ONE basic block, so
            // the scheduler overlaps the (independent) stages; anything else takes the general path
            const bool fast = strip_fast && rb + 3 < ub && rb - 2 >= max(ha, 1) && rb + 1 <= min(hb - 1, nt - 2) &&
                              rb - 4 >= max(ja, 1) && rb - 1 <= min(jb - 1, nt - 2);
            if (fast) {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int r = rb + k;
                    cp_async_wait<MARCH_PF - 1>();                   // row r has landed (for this lane) ...
                    __syncwarp();                                    // ... and for its neighbour; every lane is done with row r - 5
                    request(r + MARCH_PF);                           // reuses the slot of row r - 5
                    stage_a(k, r);
                    stage_b(std::true_type{}, k, r - 2);
                    stage_c(std::true_type{}, k, r - 4);
                }
            } else {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int r = rb + k;
                    cp_async_wait<MARCH_PF - 1>();
                    __syncwarp();
                    request(r + MARCH_PF);
                    if (r < ub) stage_a(k, r);
                    if (r - 2 >= ha && r - 2 < hb) stage_b(std::false_type{}, k, r - 2);
                    if (r - 4 >= ja && r - 4 < jb) stage_c(std::false_type{}, k, r - 4);
                }
            }
        }
        cp_async_wait<0>();
    }
}

}  // namespace tk
