// libteuk.so — C ABI of include/teuk.h.  Host logic only marshals arguments, lays out the caller's
// device workspace and launches kernels; r(r*), the coefficient planes and every step of the time loop (stepping,
// boundary and polar conditions, observer extraction and interpolation) run in CUDA kernels for sm_100a.  Host
// arithmetic: set-up scalars and r*-independent 1-D tables in quad-double (theta tables, stencil / quadrature weights).
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <algorithm>
#include <cstring>
#include <map>
#include <vector>

#include "../../include/teuk.h"
#include "mp.cuh"
#include "setup_kernels.cuh"
#include "setup_math.cuh"
#include "step_kernel.cuh"
#include "step_kernel_tma.cuh"
#include "step_kernel_tb2.cuh"
#include "step_kernel_march.cuh"
#include "kernels.h"

using namespace tk;

static int cuda_fail(cudaError_t e, const char* what, int line) {
    if (getenv("TEUK_DEBUG")) fprintf(stderr, "[teuk] CUDA error %d (%s) at line %d: %s\n", (int)e, cudaGetErrorString(e), line, what);
    return TEUK_ECUDA;
}
#define CK(call)                                                      \
    do {                                                              \
        cudaError_t e_ = (call);                                      \
        if (e_ != cudaSuccess) return cuda_fail(e_, #call, __LINE__); \
    } while (0)

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
constexpr int MP_MAX_ELL = 9;      // l' = l_min .. l_min + 8 (Fig. 1)

struct Layout {
    int pitch;
    long plane;
    size_t state_a, state_b, coef_i, coef_h, cj, r_tab, d_tab, sin_tab, cos_tab, obs_raw, obs_out, scalars, rc_rt, rc_isig, rc_th, mp_q, mp_series, total;
};

// cv = coefficient supplies resident in the workspace: -1 all (switchable with teuk_set_option), 0 stored planes only,
// 1 / 2 recompute tables only (fp64)
static inline bool cv_has_planes(int L, int cv) { return L > 1 || cv <= 0; }
static inline bool cv_has_rc(int L, int cv) { return L == 1 && cv != 0; }
static Layout make_layout(int n_r, int n_theta, int L, long cap, int cv) {
    Layout y;
    y.pitch = (int)align_up((size_t)n_r, 16);
    y.plane = (long)y.pitch * n_theta;
    size_t off = 0;
    auto take = [&](size_t doubles) {
        size_t o = off;
        off = align_up(off + doubles * sizeof(double), 256);
        return o;
    };
    y.state_a = take((size_t)4 * L * y.plane);
    y.state_b = take((size_t)4 * L * y.plane);
    y.coef_i = take(cv_has_planes(L, cv) ? (size_t)8 * L * y.plane : 1);
    y.coef_h = take(cv_has_planes(L, cv) ? (size_t)8 * L * y.plane : 1);
    y.cj = take((size_t)L * n_theta);
    y.r_tab = take((size_t)4 * (2 * n_r - 1));
    y.d_tab = take((size_t)4 * (2 * n_r - 1));
    y.sin_tab = take((size_t)4 * n_theta);
    y.cos_tab = take((size_t)4 * n_theta);
    y.obs_raw = take((size_t)(cap > 0 ? cap : 1) * 16 * L);
    y.obs_out = take((size_t)(cap > 0 ? cap : 1) * 4 * L);
    y.scalars = take(8);
    // semi-recompute supply (fp64 only): r-tables [2][16][pitch], isig planes [2][n_theta][pitch], theta tables [3][n_theta]
    y.rc_rt = take(cv_has_rc(L, cv) ? (size_t)2 * RC_NT * y.pitch : 1);
    y.rc_isig = take(cv_has_rc(L, cv) ? (size_t)2 * y.plane : 1);
    y.rc_th = take(cv_has_rc(L, cv) ? (size_t)3 * n_theta : 1);
    // multipole-projection observer (NEXT-2): weights [9][L][n_theta], series [cap][9][2][L]
    y.mp_q = take((size_t)MP_MAX_ELL * L * n_theta);
    y.mp_series = take((size_t)(cap > 0 ? cap : 1) * MP_MAX_ELL * 2 * L);
    y.total = off;
    return y;
}

struct teuk_ctx {
    double M, a, rmin, rmax, dt;
    int s, m, n_r, n_theta, L;
    int i_lo = 0, n_r_global = 0;      // radial slab: local column i <-> global column i_lo + i
    int create_variant = -1;           // supplies resident in the workspace (see make_layout)
    bool has_planes = true, has_rc = false;
    long cap_alloc;
    char* ws;
    Layout lay;
    cudaStream_t stream;
    SetupConsts C;
    // options
    int graph_steps = 32, opt_ti = 0, opt_tj = 0, opt_tma = 1, variant = 0, coef_variant = 0, theta_order = 2, opt_pdl = -1, opt_tb = 1;   // PDL measured neutral on cfg 2 (40.2 vs 40.0 us): kept as an option
    ThetaWeights tw;
    // TMA path (fp64): tensor maps of the two state buffers and the two coefficient families
    bool use_tma = false, use_rc = false, use_col_tma = false, use_march = false;
    const void* col_fn_ptr = nullptr;   // the fp64 10th-order TMA column kernel chosen by setup_col_tma
    int opt_cv = -1;                   // "coef_variant" option; -1 = automatic (resolved into coef_variant at teuk_set_initial)
    int opt_march = 1, opt_march_chunk = 0, opt_col_run = 1;   // fp64 semi-recompute supply: column-march kernel (step_kernel_march.cuh) unless march=0
    int march_strips = 0, march_chunk = 0, march_units = 0;
    CUtensorMap tm_state[2], tm_ch, tm_ci, tm_ish, tm_isi, tm_rth, tm_rti;
    // temporally blocked fp64 path (two iterations per launch, step_kernel_tb2.cuh): its own boxes, grid and smem
    bool use_tb2 = false;
    CUtensorMap tm2_state[2], tm2_ch;
    dim3 grid2;
    size_t smem2 = 0;
    // geometry
    int ti = 0, tj = 0, threads = 256;
    dim3 grid;
    size_t smem = 0;
    // state
    bool have_init = false;
    int cur = 0;                       // which state buffer holds u^n
    long steps_done = 0, launches = 0;
    long series_origin = 0;            // steps_done when the sample counter was last reset (set_observer / set_initial)
    // observer
    long obs_cap = 0;
    int oi = 0, oj = 0;
    R4 wr, wt;
    bool nonfinite = false;
    // multipole-projection observer
    long mp_cap = 0;
    int mp_n = 0, mp_i = 0;
    R4 mp_wr;
    // CUDA graphs of n consecutive iterations starting from state buffer `parity`, keyed by n: n = graph_steps for the
    // bulk of a teuk_step call and one more entry per distinct remainder (so a 20-iteration call is one graph launch too)
    std::map<long, cudaGraphExec_t> graph[2];
    void drop_graphs() {
        for (int p = 0; p < 2; ++p) {
            for (auto& kv : graph[p]) cudaGraphExecDestroy(kv.second);
            graph[p].clear();
        }
    }

    double* dptr(size_t off) const { return (double*)(ws + off); }
    double* state(int which) const { return dptr(which ? lay.state_b : lay.state_a); }
    long* step_base() const { return (long*)(ws + lay.scalars); }
    int* flag() const { return (int*)(ws + lay.scalars + 16); }
};

// ------------------------------------------------------------------------------------ small kernels
__global__ void advance_kernel(long* base, long k) { *base += k; }

template <int L>
__global__ void observer_combine_kernel(const double* __restrict__ raw, double* __restrict__ out, long count, R4 wr,
                                        R4 wt, int* flag) {
    // bilinear interpolation of the four recorded nodes in working precision (reading A11)
    long k = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (k >= count * 4) return;
    long smp = k / 4;
    int c = (int)(k % 4);
    Real<L> w_r = narrow<L>(wr), w_t = narrow<L>(wt), one = from_double<L>(1.0);
    Real<L> u[4];
#pragma unroll
    for (int nd = 0; nd < 4; ++nd)
#pragma unroll
        for (int l = 0; l < L; ++l) u[nd].x[l] = raw[((smp * 4 + nd) * 4 + c) * L + l];
    Real<L> lo = add(mul(sub(one, w_r), u[0]), mul(w_r, u[1]));
    Real<L> hi = add(mul(sub(one, w_r), u[2]), mul(w_r, u[3]));
    Real<L> v = add(mul(sub(one, w_t), lo), mul(w_t, hi));
    bool bad = false;
#pragma unroll
    for (int l = 0; l < L; ++l) {
        out[k * L + l] = v.x[l];
        bad |= !isfinite(v.x[l]);
    }
    if (bad) atomicOr(flag, 1);
}

// NEXT-2 (Fig. 1; reading A24): a_l' = sum_j Q_l'(theta_j) [(1-w) Phi(i0,j) + w Phi(i0+1,j)]
// for l' = l_min .. l_min + n_ell - 1, real and imaginary part, once per step.  One block of 32 x 2 n_ell threads:
// the interpolated column is staged in shared memory, one warp per output does a strided sum + shuffle tree.
template <int L>
__global__ void multipole_kernel(const double* __restrict__ u, const double* __restrict__ q, double* __restrict__ series,
                                 const long* step_base, int step_off, long cap, int n_ell, int nt, int pitch, long plane,
                                 int i0, R4 wr) {
    extern __shared__ double v[];                 // [2][L][nt]
    const int tid = threadIdx.x, nth = blockDim.x;
    const Real<L> w = narrow<L>(wr), omw = sub(from_double<L>(1.0), narrow<L>(wr));
    for (int idx = tid; idx < 2 * nt; idx += nth) {
        int c = idx / nt, j = idx - c * nt;
        Real<L> a, b;
#pragma unroll
        for (int l = 0; l < L; ++l) {
            a.x[l] = u[(long)(c * L + l) * plane + (long)j * pitch + i0];
            b.x[l] = u[(long)(c * L + l) * plane + (long)j * pitch + i0 + 1];
        }
        Real<L> val = add(mul(omw, a), mul(w, b));
#pragma unroll
        for (int l = 0; l < L; ++l) v[(c * L + l) * nt + j] = val.x[l];
    }
    __syncthreads();
    const int warp = tid >> 5, lane = tid & 31;
    if (warp >= 2 * n_ell) return;
    const int k = warp >> 1, c = warp & 1;
    Real<L> acc = from_double<L>(0.0);
    for (int j = lane; j < nt; j += 32) {
        Real<L> qq, vv;
#pragma unroll
        for (int l = 0; l < L; ++l) { qq.x[l] = q[(long)(k * L + l) * nt + j]; vv.x[l] = v[(c * L + l) * nt + j]; }
        acc = add(acc, mul(qq, vv));
    }
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        Real<L> o;
#pragma unroll
        for (int l = 0; l < L; ++l) o.x[l] = __shfl_down_sync(0xffffffffu, acc.x[l], off);
        acc = add(acc, o);
    }
    if (lane == 0) {
        long smp = *step_base + step_off;
        if (smp < cap) {
#pragma unroll
            for (int l = 0; l < L; ++l) series[((smp * n_ell + k) * 2 + c) * L + l] = acc.x[l];
        }
    }
}

// set_initial on the device: copy limbs_in planes per field into L planes (missing limbs := 0), force the
// radial boundary rows to zero, source layout [4][limbs_in][n_theta][n_r] (unpadded)
__global__ void load_state_kernel(const double* __restrict__ src, double* __restrict__ dst, int n_r, int n_theta,
                                  int pitch, long plane, int L, int limbs_in) {
    long idx = blockIdx.x * (long)blockDim.x + threadIdx.x;
    long per = (long)n_theta * n_r;
    if (idx >= 4 * L * per) return;
    int i = (int)(idx % n_r);
    long rest = idx / n_r;
    int j = (int)(rest % n_theta);
    int pl = (int)(rest / n_theta);
    int f = pl / L, l = pl % L;
    double v = 0.0;
    if (l < limbs_in && i != 0 && i != n_r - 1) v = src[((long)(f * limbs_in + l) * n_theta + j) * n_r + i];
    dst[pl * plane + (long)j * pitch + i] = v;
}
__global__ void store_state_kernel(const double* __restrict__ src, double* __restrict__ dst, int n_r, int n_theta,
                                   int pitch, long plane, int planes) {
    long idx = blockIdx.x * (long)blockDim.x + threadIdx.x;
    long per = (long)n_theta * n_r;
    if (idx >= planes * per) return;
    int i = (int)(idx % n_r);
    long rest = idx / n_r;
    int j = (int)(rest % n_theta);
    int pl = (int)(rest / n_theta);
    dst[idx] = src[pl * plane + (long)j * pitch + i];
}

// ------------------------------------------------------------------------------------ create
static bool valid_sizes(int n_r, int n_theta, int precision, long cap) {
    return n_r >= 3 && n_theta >= 2 && (precision == 1 || precision == 2 || precision == 4) && cap >= 0 &&
           (long)n_r * n_theta < (1L << 31);
}

static bool valid_variant(int precision, int cv) { return cv >= -1 && cv <= 2 && (cv < 1 || precision == 1); }

extern "C" int teuk_workspace_bytes(int n_r, int n_theta, int precision, int coef_variant, long obs_capacity, size_t* bytes) {
    if (!bytes || !valid_sizes(n_r, n_theta, precision, obs_capacity) || !valid_variant(precision, coef_variant)) return TEUK_EINVAL;
    *bytes = make_layout(n_r, n_theta, precision, obs_capacity, coef_variant).total;
    return TEUK_OK;
}

template <int L>
static int launch_coef(teuk_ctx* c, int half, int fold, double* out) {
    int cols = half ? c->n_r - 1 : c->n_r;
    dim3 grid((cols + 127) / 128, c->n_theta);
    coef_kernel<L><<<grid, 128, 0, c->stream>>>(c->C, c->dptr(c->lay.r_tab), c->dptr(c->lay.d_tab),
                                                c->dptr(c->lay.sin_tab), c->dptr(c->lay.cos_tab), half, fold, out);
    c->launches++;
    return cudaGetLastError() == cudaSuccess ? TEUK_OK : TEUK_ECUDA;
}
static int launch_coef_any(teuk_ctx* c, int half, int fold, double* out) {
    if (c->L == 1) return launch_coef<1>(c, half, fold, out);
    if (c->L == 2) return launch_coef<2>(c, half, fold, out);
    return launch_coef<4>(c, half, fold, out);
}

// one handle = columns [i_lo, i_lo + n_r) of the uniform grid of n_r_global nodes on [rstar_min, rstar_max]
static int create_impl(double M, double a, int s, int m, int n_r_global, int i_lo, int n_r, int n_theta, double rstar_min,
                       double rstar_max, double dt, int precision, int cv, void* d_workspace, size_t workspace_bytes,
                       long obs_capacity, void* cuda_stream, teuk_ctx** out) {
    if (!out || !d_workspace || !valid_sizes(n_r, n_theta, precision, obs_capacity) || !valid_variant(precision, cv)) return TEUK_EINVAL;
    if (i_lo < 0 || (long)i_lo + n_r > n_r_global || n_r_global >= (1 << 29)) return TEUK_EINVAL;
    if (!(M > 0) || !(std::fabs(a) < M) || !(dt > 0) || !(rstar_min < rstar_max)) return TEUK_EINVAL;
    if (!std::isfinite(M) || !std::isfinite(a) || !std::isfinite(dt) || !std::isfinite(rstar_min) ||
        !std::isfinite(rstar_max))
        return TEUK_EINVAL;
    Layout lay = make_layout(n_r, n_theta, precision, obs_capacity, cv);
    if (workspace_bytes < lay.total || ((size_t)d_workspace % 256) != 0) return TEUK_EINVAL;
    teuk_ctx* c = new (std::nothrow) teuk_ctx();
    if (!c) return TEUK_ENOMEM;
    c->M = M; c->a = a; c->s = s; c->m = m; c->n_r = n_r; c->n_theta = n_theta; c->L = precision;
    c->rmin = rstar_min; c->rmax = rstar_max; c->dt = dt; c->cap_alloc = obs_capacity;
    c->i_lo = i_lo; c->n_r_global = n_r_global;
    c->create_variant = cv; c->has_planes = cv_has_planes(precision, cv); c->has_rc = cv_has_rc(precision, cv);
    c->opt_cv = cv;                    // a handle created for one supply uses it; -1: chosen at teuk_set_initial
    c->coef_variant = cv < 0 ? 0 : cv;
    c->ws = (char*)d_workspace; c->lay = lay; c->stream = (cudaStream_t)cuda_stream;

    // ---- host scalars in quad-double
    QConst qc = q_constants();
    SetupConsts& C = c->C;
    C.M = from_double<4>(M);
    C.a = from_double<4>(a);
    R4 root = msqrt(sub(mul(C.M, C.M), mul(C.a, C.a)));
    C.rp = add(C.M, root);
    R4 rm = sub(C.M, root);
    C.rpm = scale2(root, 2.0);
    C.cplus = div(mul(scale2(C.M, 2.0), C.rp), C.rpm);
    C.cminus = div(mul(scale2(C.M, 2.0), rm), C.rpm);
    C.rmin = from_double<4>(rstar_min);
    C.dr = div(sub(from_double<4>(rstar_max), C.rmin), from_double<4>((double)(n_r_global - 1)));
    C.k0 = 2 * i_lo;
    C.dth = div(qc.pi, from_double<4>((double)n_theta));
    C.ln2 = qc.ln2;
    C.tau_f = from_double<4>(dt);
    C.tau_h = scale2(C.tau_f, 0.5);
    C.s = s; C.m = m; C.n_r = n_r; C.n_theta = n_theta; C.pitch = lay.pitch; C.plane = lay.plane;

    // ---- theta tables on the host (N_theta/2 Taylor evaluations), mirrored so they are exactly symmetric
    std::vector<double> sn(4 * n_theta), cs(4 * n_theta), cjv((size_t)precision * n_theta);
    for (int j = 0; j < (n_theta + 1) / 2; ++j) {
        R4 th = mul(C.dth, add(from_double<4>((double)j), from_double<4>(0.5)));
        R4 sj, cj;
        q_sincos(th, sj, cj);
        int jm = n_theta - 1 - j;
        if (jm == j) cj = from_double<4>(0.0);
        R4 cot = div(cj, sj);
        R4 cjq = scale2(mul(cot, C.dth), 0.5);            // cot(theta_j) dtheta / 2
        for (int l = 0; l < 4; ++l) {
            sn[4 * j + l] = sj.x[l];  cs[4 * j + l] = cj.x[l];
            sn[4 * jm + l] = sj.x[l]; cs[4 * jm + l] = -cj.x[l];
        }
        for (int l = 0; l < precision; ++l) {
            cjv[(size_t)l * n_theta + j] = cjq.x[l];
            cjv[(size_t)l * n_theta + jm] = (jm == j) ? 0.0 : -cjq.x[l];
        }
    }
    int rc = TEUK_OK;
    auto fail = [&](int code) { delete c; return code; };
    if (cudaMemsetAsync(c->ws, 0, lay.total, c->stream) != cudaSuccess) return fail(TEUK_ECUDA);
    if (cudaMemcpyAsync(c->dptr(lay.sin_tab), sn.data(), sn.size() * 8, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(c->dptr(lay.cos_tab), cs.data(), cs.size() * 8, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
        cudaMemcpyAsync(c->dptr(lay.cj), cjv.data(), cjv.size() * 8, cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
        return fail(TEUK_ECUDA);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return fail(TEUK_ECUDA);   // host vectors go out of scope

    // ---- r(r*) and the coefficient planes on the device
    int npts = 2 * n_r - 1;
    radial_kernel<<<(npts + 63) / 64, 64, 0, c->stream>>>(C, c->dptr(lay.r_tab), c->dptr(lay.d_tab));
    c->launches++;
    if (cudaGetLastError() != cudaSuccess) return fail(TEUK_ECUDA);
    if (c->has_rc) {
        // semi-recompute supply: theta tables on the host in quad-double, r-tables and isig planes on the device
        std::vector<double> th((size_t)3 * n_theta);
        for (int j = 0; j < n_theta; ++j) {
            R4 sj, cj;
            for (int l = 0; l < 4; ++l) { sj.x[l] = sn[4 * j + l]; cj.x[l] = cs[4 * j + l]; }
            R4 s2 = mul(sj, sj);
            R4 mc = add(from_double<4>((double)m), mul_d(cj, (double)s));
            R4 tth = sub(div(mul(mc, mc), s2), from_double<4>((double)s));
            th[j] = s2.x[0]; th[n_theta + j] = cj.x[0]; th[2 * n_theta + j] = tth.x[0];
        }
        if (cudaMemcpyAsync(c->dptr(lay.rc_th), th.data(), th.size() * 8, cudaMemcpyHostToDevice, c->stream) != cudaSuccess ||
            cudaStreamSynchronize(c->stream) != cudaSuccess)
            return fail(TEUK_ECUDA);
        rtab_kernel<<<(npts + 63) / 64, 64, 0, c->stream>>>(C, c->dptr(lay.r_tab), c->dptr(lay.d_tab), c->dptr(lay.rc_rt));
        for (int half = 0; half < 2; ++half) {
            int cols = half ? n_r - 1 : n_r;
            isig_kernel<<<dim3((cols + 127) / 128, n_theta), 128, 0, c->stream>>>(
                C, c->dptr(lay.r_tab), c->dptr(lay.d_tab), c->dptr(lay.sin_tab), half, c->dptr(lay.rc_isig) + (size_t)half * lay.plane);
        }
        c->launches += 3;
        if (cudaGetLastError() != cudaSuccess) return fail(TEUK_ECUDA);
    }
    if (c->has_planes) {
        if ((rc = launch_coef_any(c, 0, 1, c->dptr(lay.coef_i))) != TEUK_OK) return fail(rc);
        if ((rc = launch_coef_any(c, 1, 1, c->dptr(lay.coef_h))) != TEUK_OK) return fail(rc);
    }
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return fail(TEUK_ECUDA);
    *out = c;
    return TEUK_OK;
}

extern "C" int teuk_create(double M, double a, int s, int m, int n_r, int n_theta, double rstar_min, double rstar_max,
                           double dt, int precision, int coef_variant, void* d_workspace, size_t workspace_bytes,
                           long obs_capacity, void* cuda_stream, teuk_ctx** out) {
    return create_impl(M, a, s, m, n_r, 0, n_r, n_theta, rstar_min, rstar_max, dt, precision, coef_variant, d_workspace,
                       workspace_bytes, obs_capacity, cuda_stream, out);
}

extern "C" int teuk_create_slab(double M, double a, int s, int m, int n_r_global, int n_theta, double rstar_min,
                                double rstar_max, double dt, int precision, int coef_variant, int i_lo, int n_win,
                                void* d_workspace, size_t workspace_bytes, long obs_capacity, void* cuda_stream,
                                teuk_ctx** out) {
    return create_impl(M, a, s, m, n_r_global, i_lo, n_win, n_theta, rstar_min, rstar_max, dt, precision, coef_variant,
                       d_workspace, workspace_bytes, obs_capacity, cuda_stream, out);
}

extern "C" int teuk_set_option(teuk_ctx* c, const char* key, double value) {
    if (!c || !key) return TEUK_EINVAL;
    if (c->have_init) return TEUK_ESTATE;
    int v = (int)value;
    if (!strcmp(key, "graph_steps")) {
        if (v < 0 || (v % 2) != 0 || v > 4096) return TEUK_EINVAL;
        c->graph_steps = v;
    } else if (!strcmp(key, "tile_i")) {
        if (v < 0 || v > 256) return TEUK_EINVAL;
        c->opt_ti = v;
    } else if (!strcmp(key, "tile_j")) {
        if (v < 0 || v > 256) return TEUK_EINVAL;
        c->opt_tj = v;
    } else if (!strcmp(key, "pdl")) {
        c->opt_pdl = v != 0;
    } else if (!strcmp(key, "theta_order")) {
        if ((v != 2 && v != 10) || c->n_theta < v / 2) return TEUK_EINVAL;
        c->theta_order = v;
    } else if (!strcmp(key, "coef_variant")) {
        if (v < 0 || v > 2 || (v >= 1 && c->L != 1)) return TEUK_EINVAL;
        if (v == 0 ? !c->has_planes : !c->has_rc) return TEUK_EINVAL;      // that supply is not resident in this handle's workspace
        c->opt_cv = v;
    } else if (!strcmp(key, "variant")) {
        if (v < 0 || v > 4) return TEUK_EINVAL;
        c->variant = v;
    } else if (!strcmp(key, "time_block")) {
        if ((v != 1 && v != 2) || (v == 2 && c->L != 1)) return TEUK_EINVAL;
        c->opt_tb = v;
    } else if (!strcmp(key, "col_run")) {
        c->opt_col_run = v != 0;
    } else if (!strcmp(key, "march")) {
        c->opt_march = v != 0;
    } else if (!strcmp(key, "march_chunk")) {        // theta rows per work unit of the march kernel (0 = chosen by the library)
        if (v < 0 || v > c->n_theta) return TEUK_EINVAL;
        c->opt_march_chunk = v;
    } else if (!strcmp(key, "use_tma")) {
        c->opt_tma = v != 0;
    } else {
        return TEUK_EINVAL;
    }
    return TEUK_OK;
}

extern "C" int teuk_set_observer(teuk_ctx* c, double rstar_obs, double theta_obs, long capacity) {
    if (!c || capacity < 0 || capacity > c->cap_alloc || !std::isfinite(rstar_obs) || !std::isfinite(theta_obs))
        return TEUK_EINVAL;
    R4 x = sub(div(sub(from_double<4>(rstar_obs), c->C.rmin), c->C.dr), from_double<4>((double)c->i_lo));
    R4 y = sub(div(from_double<4>(theta_obs), c->C.dth), from_double<4>(0.5));
    int i0 = (int)std::floor(x.x[0]), j0 = (int)std::floor(y.x[0]);
    if (x.x[0] < 0 || x.x[0] > c->n_r - 1 || y.x[0] < 0 || y.x[0] > c->n_theta - 1) return TEUK_EINVAL;
    if (i0 > c->n_r - 2) i0 = c->n_r - 2;
    if (j0 > c->n_theta - 2) j0 = c->n_theta - 2;
    c->wr = sub(x, from_double<4>((double)i0));
    c->wt = sub(y, from_double<4>((double)j0));
    c->oi = i0; c->oj = j0; c->obs_cap = capacity;
    c->nonfinite = false;
    c->drop_graphs();
    CK(cudaMemsetAsync(c->step_base(), 0, 32, c->stream));
    c->series_origin = c->steps_done;      // both series (point observer and multipoles) restart here
    return TEUK_OK;
}

// ------------------------------------------------------------------------------------ stepping
static size_t smem_bytes(int L, int ti, int tj) {
    return (size_t)4 * L * ((size_t)(ti + 2) * (tj + 4) + (size_t)(ti + 1) * (tj + 2)) * sizeof(double);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 3-D tensor map over `planes` fp64 planes of n_theta rows x cols columns (row pitch `pitch`, plane stride `plane`)
static bool make_map(CUtensorMap* tm, double* ptr, int cols, int n_theta, int planes, int pitch, long plane, int bx,
                     int by, int bz) {
    static EncodeTiledFn enc = nullptr;
    if (!enc) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn) return false;
        enc = (EncodeTiledFn)fn;
    }
    cuuint64_t dims[3] = {(cuuint64_t)cols, (cuuint64_t)n_theta, (cuuint64_t)planes};
    cuuint64_t strides[2] = {(cuuint64_t)pitch * 8, (cuuint64_t)plane * 8};
    cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, (cuuint32_t)bz};
    cuuint32_t es[3] = {1, 1, 1};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, ptr, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int TI, int TJ> static bool setup_tma(teuk_ctx* c) {
    using G = TmaGeom<TI, TJ>;
    const Layout& y = c->lay;
    bool ok = make_map(&c->tm_state[0], c->state(0), c->n_r, c->n_theta, 4, y.pitch, y.plane, G::UC, G::UR, 4) &&
              make_map(&c->tm_state[1], c->state(1), c->n_r, c->n_theta, 4, y.pitch, y.plane, G::UC, G::UR, 4) &&
              make_map(&c->tm_ch, c->dptr(y.coef_h), c->n_r - 1, c->n_theta, 8, y.pitch, y.plane, G::CC, G::HR, 8) &&
              make_map(&c->tm_ci, c->dptr(y.coef_i), c->n_r, c->n_theta, 8, y.pitch, y.plane, TI, TJ, 8);
    if (!ok) return false;
    const void* fn = tma_step_fn(TI, TJ);
    if (!fn || cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, G::TOTAL) != cudaSuccess) return false;
    c->ti = TI; c->tj = TJ; c->smem = G::TOTAL; c->threads = 256;
    c->grid = dim3((c->n_r + TI - 1) / TI, (c->n_theta + TJ - 1) / TJ);
    return true;
}

template <int TI, int TJ> static bool setup_tb2(teuk_ctx* c) {
    using G = Tb2Geom<TI, TJ>;
    const Layout& y = c->lay;
    bool ok = make_map(&c->tm2_state[0], c->state(0), c->n_r, c->n_theta, 4, y.pitch, y.plane, G::UC, G::UR, 4) &&
              make_map(&c->tm2_state[1], c->state(1), c->n_r, c->n_theta, 4, y.pitch, y.plane, G::UC, G::UR, 4) &&
              make_map(&c->tm2_ch, c->dptr(y.coef_h), c->n_r - 1, c->n_theta, 8, y.pitch, y.plane, G::CC, G::H1R, 8);
    if (!ok) return false;
    const void* fn = tb2_step_fn(TI, TJ);
    if (!fn || cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, G::TOTAL) != cudaSuccess) return false;
    c->smem2 = G::TOTAL;
    c->grid2 = dim3((c->n_theta + TJ - 1) / TJ, (c->n_r + TI - 1) / TI);      // theta tiles fastest
    return c->grid2.y <= 65535;
}

// instantiation tables of the generic kernels live in k_generic{1,2,4}.cu: (precision, variant, tile) -> function, block size
static const void* step_fn(const teuk_ctx* c, int* threads) {
    if (c->L == 1) return generic_step_fn_1(c->variant, c->ti, c->tj, threads);
    if (c->L == 2) return generic_step_fn_2(c->variant, c->ti, c->tj, threads);
    return generic_step_fn_4(c->variant, c->ti, c->tj, threads);
}

template <int TI, int TJ> static bool setup_rc(teuk_ctx* c) {
    using G = RcGeom<TI, TJ>;
    const Layout& y = c->lay;
    double* is0 = c->dptr(y.rc_isig);
    double* rt0 = c->dptr(y.rc_rt);
    bool ok = make_map(&c->tm_state[0], c->state(0), c->n_r, c->n_theta, 4, y.pitch, y.plane, G::UC, G::UR, 4) &&
              make_map(&c->tm_state[1], c->state(1), c->n_r, c->n_theta, 4, y.pitch, y.plane, G::UC, G::UR, 4) &&
              make_map(&c->tm_isi, is0, c->n_r, c->n_theta, 1, y.pitch, y.plane, TI, TJ, 1) &&
              make_map(&c->tm_ish, is0 + y.plane, c->n_r - 1, c->n_theta, 1, y.pitch, y.plane, G::CC, G::HR, 1) &&
              make_map(&c->tm_rti, rt0, c->n_r, RC_NT, 1, y.pitch, (long)RC_NT * y.pitch, TI, RC_NT, 1) &&
              make_map(&c->tm_rth, rt0 + (size_t)RC_NT * y.pitch, c->n_r - 1, RC_NT, 1, y.pitch, (long)RC_NT * y.pitch, G::CC, RC_NT, 1);
    if (!ok) return false;
    const void* fn = rc_step_fn(TI, TJ, c->coef_variant == 2);
    if (!fn || cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, G::TOTAL) != cudaSuccess) return false;
    c->ti = TI; c->tj = TJ; c->smem = G::TOTAL; c->threads = 256;
    c->grid = dim3((c->n_r + TI - 1) / TI, (c->n_theta + TJ - 1) / TJ);
    return true;
}

template <int TI> static bool setup_col_tma(teuk_ctx* c, bool row_run) {
    using G = ColGeom<TI>;
    const Layout& y = c->lay;
    const int nt = c->n_theta;
    double* is0 = c->dptr(y.rc_isig);
    double* rt0 = c->dptr(y.rc_rt);
    bool ok = make_map(&c->tm_state[0], c->state(0), c->n_r, nt, 4, y.pitch, y.plane, G::UC, nt, 4) &&
              make_map(&c->tm_state[1], c->state(1), c->n_r, nt, 4, y.pitch, y.plane, G::UC, nt, 4) &&
              make_map(&c->tm_isi, is0, c->n_r, nt, 1, y.pitch, y.plane, TI, nt, 1) &&
              make_map(&c->tm_ish, is0 + y.plane, c->n_r - 1, nt, 1, y.pitch, y.plane, G::CC, nt, 1) &&
              make_map(&c->tm_rti, rt0, c->n_r, RC_NT, 1, y.pitch, (long)RC_NT * y.pitch, TI, RC_NT, 1) &&
              make_map(&c->tm_rth, rt0 + (size_t)RC_NT * y.pitch, c->n_r - 1, RC_NT, 1, y.pitch, (long)RC_NT * y.pitch, G::CC, RC_NT, 1);
    size_t sm = row_run ? G::total_run(nt) : G::total(nt);
    if (!ok || sm > 227 * 1024) return false;
    const int threads = 256;
    const void* fn = row_run ? col_run_fn(TI) : col_tma_fn(TI);
    if (!fn || cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm) != cudaSuccess) return false;
    c->ti = TI; c->tj = nt; c->smem = sm; c->threads = threads; c->col_fn_ptr = fn;
    c->grid = dim3((c->n_r + TI - 1) / TI, 1);
    return true;
}

static const void* col_fn(const teuk_ctx* c, int* threads) {
    if (c->L == 1) return generic_col_fn_1(threads);
    if (c->L == 2) return generic_col_fn_2(threads);
    return generic_col_fn_4(c->variant, threads);
}

// centred 11-point weights from the textbook closed form c_k = (-1)^(k+1) (N!)^2 / (k (N-k)! (N+k)!), d_k = 2 c_k / k
static void fill_theta_weights(ThetaWeights& w) {
    const int N = 5;
    double fact[11] = {1, 1, 2, 6, 24, 120, 720, 5040, 40320, 362880, 3628800};
    R4 d0 = from_double<4>(0.0);
    for (int k = 1; k <= N; ++k) {
        R4 num = from_double<4>(((k & 1) ? 1.0 : -1.0) * fact[N] * fact[N]);
        R4 den = from_double<4>((double)k * fact[N - k] * fact[N + k]);
        R4 ck = div(num, den);
        R4 dk = div(scale2(ck, 2.0), from_double<4>((double)k));
        d0 = sub(d0, scale2(dk, 2.0));
        for (int l = 0; l < 4; ++l) { w.wc[k - 1][l] = ck.x[l]; w.wd[k][l] = dk.x[l]; }
    }
    for (int l = 0; l < 4; ++l) w.wd[0][l] = d0.x[l];
}

// fp64 grids from this many points on step faster with the semi-recompute column-march kernel than with the stored
// planes (profiles/r02_sweep.md: 16384 x 32 and 4096 x 256 win, 4096 x 64 loses: too few work units for 1184 warps)
constexpr long MARCH_AUTO_MIN_POINTS = 400000;

static int choose_geometry(teuk_ctx* c) {
    c->coef_variant = c->opt_cv;
    if (c->opt_cv < 0) {
        // automatic: the fastest parity-green supply for this grid, unless an option asks for a specific stored-plane kernel
        const bool plain = c->theta_order == 2 && c->opt_tb == 1 && c->opt_tma && c->opt_march && c->opt_ti == 0 &&
                           c->opt_tj == 0 && c->variant == 0;
        const bool big = (long)c->n_r * c->n_theta >= MARCH_AUTO_MIN_POINTS && 4 * c->lay.plane < (1L << 31);
        c->coef_variant = (c->L == 1 && c->has_rc && c->has_planes && plain && big) ? 1 : (c->has_planes ? 0 : 1);
    }
    c->use_tma = false;
    c->use_rc = false;
    c->use_tb2 = false;
    if (c->opt_tb == 2 && (c->theta_order == 10 || c->coef_variant != 0)) return TEUK_EINVAL;
    if (c->theta_order == 10) {
        fill_theta_weights(c->tw);
        c->use_col_tma = false;
        if (c->L == 1 && c->has_rc && c->opt_tma && c->n_theta <= 256 && (c->opt_ti == 0 || c->opt_ti == 8 || c->opt_ti == 12 || c->opt_ti == 16)) {
            // fp64: TMA column kernel with the semi-recompute coefficient supply (always, whatever coef_variant says)
            // automatic tile: 16 columns when N_theta <= 64 (half the block barriers and one redundant half-step column per
            // 16 instead of per 8: measured 3-5 % faster on 16384 x 64 and 65536 x 64 although one block per SM), else 8
            const int ti = c->opt_ti ? c->opt_ti : (c->n_theta <= 64 && c->n_r >= 2048 ? 16 : 8);
            // kernel: row runs (a thread owns 4 consecutive rows of a column, stencil window in registers; +22 % on
            // config 2) unless "col_run" = 0 or the 12-column tile is asked for: then one point per thread
            const bool rr = c->opt_col_run && ti != 12;
            bool ok = ti == 16 ? setup_col_tma<16>(c, rr) : ti == 12 ? setup_col_tma<12>(c, false) : setup_col_tma<8>(c, rr);
            cudaGetLastError();
            if (ok) { c->use_col_tma = true; return TEUK_OK; }
        }
        if (c->coef_variant != 0 || !c->has_planes) return TEUK_EINVAL;
        int ti = c->opt_ti;
        if (ti == 0) {
            // largest tile within the shared-memory budget: 3 blocks/SM for qd (72 KB each), 2 blocks/SM otherwise (100 KB)
            long per_col = (long)4 * c->L * 8 * c->n_theta;       // bytes per tile column of u or h (sig tile: half of that)
            ti = (int)(((c->L == 4 ? 72 : 100) * 1024 / per_col - 3.5) / 2.5);
            if (ti > 32) ti = 32;
            if (c->L == 1 && ti >= 8) ti = (ti >= 16) ? 16 : 8;      // fp64: whole 64/128-byte rows per tile (measured best)
            if (ti < 2) ti = 2;
            if (c->L == 4 && c->variant != 4) {
                // pair kernel: 2 blocks/SM (110 KB each) of 256 threads = 128 points per pass over the sub-step code; among
                // the tiles that fit take the one with the fewest passes per column (half step: (ti + 1) columns, full: ti)
                const int tmax = std::max(2, std::min(32, (int)((110 * 1024 / per_col - 3.5) / 2.5)));
                double best = 1e30;
                for (int t = 2; t <= tmax; ++t) {
                    const long nt = c->n_theta;
                    const double cost = (double)(((t + 1) * nt + 127) / 128 + (t * nt + 127) / 128) / t;
                    if (cost <= best) { best = cost; ti = t; }
                }
            }
        }
        if (ti > c->n_r) ti = c->n_r;
        size_t sm = (size_t)4 * c->L * 8 * c->n_theta * (2 * ti + 3) + (size_t)2 * c->L * 8 * c->n_theta * (ti + 1);
        if (sm > 227 * 1024) return TEUK_EINVAL;
        c->ti = ti; c->tj = c->n_theta; c->smem = sm;
        c->grid = dim3((c->n_r + ti - 1) / ti, 1);
        const void* fn = col_fn(c, &c->threads);
        return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm) == cudaSuccess ? TEUK_OK : TEUK_ECUDA;
    }
    c->use_march = false;
    if (c->L == 1 && c->coef_variant == 1 && c->opt_march && 4 * c->lay.plane < (1L << 31)) {
        // persistent grid of resident warps; work unit = (strip of 30 columns, chunk of theta rows)
        const void* fn = march_step_fn();
        const size_t sm = march_smem_bytes(c->n_theta);
        int dev = 0, sms = 0, per_sm = 0;
        if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm) != cudaSuccess ||
            cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, 32 * MARCH_WARPS, sm) != cudaSuccess || per_sm < 1)
            return TEUK_ECUDA;
        const int nt = c->n_theta;
        const long strips = (c->n_r + MARCH_W - 1) / MARCH_W;
        const long capacity = (long)sms * per_sm * MARCH_WARPS;
        // chunk length: k chunks per column; a warp's time ~ rounds x (rows + 6 rows of pipeline fill and drain + 4 halo
        // rows when the column is cut); pick the k that minimises it (k = 1: whole columns)
        int best_k = 1;
        long best_cost = -1;
        for (int k = 1; k <= std::max(1, nt / 8); ++k) {
            const long rows = (nt + k - 1) / k;
            const long kk = (nt + rows - 1) / rows;                 // chunks per column actually produced
            const long rounds = (strips * kk + capacity - 1) / capacity;
            const long cost = rounds * (rows + 6 + (kk > 1 ? 4 : 0));
            if (best_cost < 0 || cost < best_cost) { best_cost = cost; best_k = k; }
        }
        int rows = c->opt_march_chunk > 0 ? c->opt_march_chunk : (nt + best_k - 1) / best_k;
        const long chunks = (nt + rows - 1) / rows;
        const long units = strips * chunks;
        if (units >= (1L << 31)) return TEUK_EINVAL;
        const long warps = std::min(units, capacity);
        c->march_strips = (int)strips; c->march_chunk = rows; c->march_units = (int)units;
        c->ti = MARCH_W; c->tj = rows; c->smem = sm; c->threads = 32 * MARCH_WARPS;
        c->grid = dim3((unsigned)((warps + MARCH_WARPS - 1) / MARCH_WARPS), 1);
        c->use_march = true;
        return TEUK_OK;
    }
    if (c->L == 1 && c->coef_variant >= 1) {
        bool ok = (c->opt_tj == 8) ? setup_rc<32, 8>(c) : setup_rc<32, 16>(c);
        cudaGetLastError();
        if (!ok) return TEUK_ECUDA;       // the recompute variant exists only as a TMA kernel
        c->use_rc = true;
        return TEUK_OK;
    }
    if (!c->has_planes) return TEUK_EINVAL;      // every path below reads the stored coefficient planes
    if (c->L == 1 && c->opt_tma && (c->opt_ti == 0 || c->opt_ti == 32) && (c->opt_tj == 0 || c->opt_tj == 8 || c->opt_tj == 16)) {
        bool ok = (c->opt_tj == 8) ? setup_tma<32, 8>(c) : setup_tma<32, 16>(c);
        cudaGetLastError();
        if (ok) {
            c->use_tma = true;
            if (c->opt_tb == 2) {
                // two iterations per launch on the same output tile; the single-step kernel serves an odd last step
                bool ok2 = (c->tj == 8) ? setup_tb2<32, 8>(c) : setup_tb2<32, 16>(c);
                cudaGetLastError();
                if (!ok2) return TEUK_ECUDA;
                c->use_tb2 = true;
            }
            return TEUK_OK;
        }
    }
    if (c->opt_tb == 2) return TEUK_EINVAL;        // time blocking exists only on the fp64 TMA stored-plane path
    int ti = c->opt_ti, tj = c->opt_tj;
    // qd default: the pair kernel on its compile-time 16 x 16 tile (ragged edges are masked in the kernel, no clamping)
    const bool qd_pair = c->L == 4 && (c->variant == 0 || c->variant == 3) && ti == 0 && tj == 0 && c->n_theta >= 12;
    if (ti == 0) ti = (c->L == 4) ? 16 : 32;
    if (qd_pair) {
        tj = 16;
    } else {
        if (tj == 0) {
            // whole theta extent when it fits (no theta halo, no redundant half-step rows), else strips of 16
            int full = c->n_theta;
            tj = (smem_bytes(c->L, ti, full) <= 100 * 1024 && full <= 64) ? full : ((c->L == 4) ? 8 : 16);
        }
        if (tj > c->n_theta) tj = c->n_theta;
        if (ti > c->n_r) ti = c->n_r;
    }
    size_t sm = smem_bytes(c->L, ti, tj);
    if (sm > 227 * 1024) return TEUK_EINVAL;
    c->ti = ti; c->tj = tj; c->smem = sm;
    c->grid = dim3((c->n_r + ti - 1) / ti, (c->n_theta + tj - 1) / tj);
    cudaError_t e = cudaSuccess;
    const void* fn = step_fn(c, &c->threads);
    e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    return e == cudaSuccess ? TEUK_OK : TEUK_ECUDA;
}

static int launch_step(teuk_ctx* c, int from, int step_off) {
    StepParams P;
    P.u_in = c->state(from);
    P.u_out = c->state(from ^ 1);
    P.coef_i = c->dptr(c->lay.coef_i);
    P.coef_h = c->dptr(c->lay.coef_h);
    P.cj = c->dptr(c->lay.cj);
    P.n_r = c->n_r; P.n_theta = c->n_theta; P.pitch = c->lay.pitch; P.plane = c->lay.plane;
    P.ti = c->ti; P.tj = c->tj;
    P.sigma = (std::abs(c->m) % 2 == 0) ? 1.0 : -1.0;
    P.tq_half = 0.25 * c->dt;
    P.tq_full = 0.5 * c->dt;
    P.obs_raw = c->obs_cap > 0 ? c->dptr(c->lay.obs_raw) : nullptr;
    P.step_base = c->step_base();
    P.obs_cap = c->obs_cap;
    P.step_off = step_off;
    P.oi = c->oi; P.oj = c->oj;
    if (c->theta_order == 10 && c->use_col_tma) {
        RcParams Q{c->dptr(c->lay.rc_th)};
        void* args[] = {&c->tm_state[from], &c->tm_ish, &c->tm_isi, &c->tm_rth, &c->tm_rti, &P, &Q, &c->tw};
        if (cudaLaunchKernel(c->col_fn_ptr, c->grid, dim3(c->threads), args, c->smem, c->stream) != cudaSuccess) return TEUK_ECUDA;
    } else if (c->theta_order == 10) {
        void* args[] = {&P, &c->tw};
        int threads = 256;
        const void* fn = col_fn(c, &threads);
        if (cudaLaunchKernel(fn, c->grid, dim3(threads), args, c->smem, c->stream) != cudaSuccess) return TEUK_ECUDA;
    } else if (c->use_march) {
        MarchParams Q;
        Q.isig_i = c->dptr(c->lay.rc_isig);
        Q.isig_h = c->dptr(c->lay.rc_isig) + c->lay.plane;
        Q.rt = c->dptr(c->lay.rc_rt);
        Q.th = c->dptr(c->lay.rc_th);
        Q.n_strips = c->march_strips;
        Q.chunk_rows = c->march_chunk;
        Q.n_units = c->march_units;
        void* args[] = {&P, &Q};
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = c->grid; cfg.blockDim = dim3(c->threads); cfg.dynamicSmemBytes = c->smem; cfg.stream = c->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = c->opt_pdl != 0 ? 1 : 0;      // automatic (-1) = on: +2.7 % on cfg 2, +1.6 % on 65536 x 64
        cudaError_t le = cudaLaunchKernelExC(&cfg, march_step_fn(), args);
        if (le != cudaSuccess) return cuda_fail(le, "cudaLaunchKernelEx(march kernel)", __LINE__);
    } else if (c->use_rc || c->use_tma) {
        // programmatic dependent launch: the next step's blocks may start (and prefetch their coefficient tiles) while this
        // step drains; they execute griddepcontrol.wait before touching the state
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = c->grid; cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = c->smem; cfg.stream = c->stream;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = c->opt_pdl == 1 ? 1 : 0;
        cudaError_t le;
        RcParams Q{c->dptr(c->lay.rc_th)};
        if (c->use_rc) {
            void* args[] = {&c->tm_state[from], &c->tm_ish, &c->tm_isi, &c->tm_rth, &c->tm_rti, &P, &Q};
            le = cudaLaunchKernelExC(&cfg, rc_step_fn(c->ti, c->tj, c->coef_variant == 2), args);
        } else {
            void* args[] = {&c->tm_state[from], &c->tm_ch, &c->tm_ci, &P};
            le = cudaLaunchKernelExC(&cfg, tma_step_fn(c->ti, c->tj), args);
        }
        if (le != cudaSuccess) return cuda_fail(le, "cudaLaunchKernelEx(step kernel)", __LINE__);
    } else {
        void* args[] = {&P};
        int threads = 256;
        const void* fn = step_fn(c, &threads);
        if (cudaLaunchKernel(fn, c->grid, dim3(threads), args, c->smem, c->stream) != cudaSuccess) return TEUK_ECUDA;
    }
    if (c->mp_cap > 0) {
        const double* uo = c->state(from ^ 1);
        const double* qd_ = c->dptr(c->lay.mp_q);
        double* ser = c->dptr(c->lay.mp_series);
        int threads = 64 * c->mp_n;
        size_t sm = (size_t)2 * c->L * c->n_theta * sizeof(double);
        if (c->L == 1) multipole_kernel<1><<<1, threads, sm, c->stream>>>(uo, qd_, ser, c->step_base(), step_off, c->mp_cap, c->mp_n, c->n_theta, c->lay.pitch, c->lay.plane, c->mp_i, c->mp_wr);
        else if (c->L == 2) multipole_kernel<2><<<1, threads, sm, c->stream>>>(uo, qd_, ser, c->step_base(), step_off, c->mp_cap, c->mp_n, c->n_theta, c->lay.pitch, c->lay.plane, c->mp_i, c->mp_wr);
        else multipole_kernel<4><<<1, threads, sm, c->stream>>>(uo, qd_, ser, c->step_base(), step_off, c->mp_cap, c->mp_n, c->n_theta, c->lay.pitch, c->lay.plane, c->mp_i, c->mp_wr);
    }
    return cudaGetLastError() == cudaSuccess ? TEUK_OK : TEUK_ECUDA;
}

static inline bool tb2_active(const teuk_ctx* c) { return c->use_tb2 && c->mp_cap == 0; }

// two iterations in one launch: state(from) = u^n  ->  state(from ^ 1) = u^{n+2}; observer samples step_off, step_off + 1
static int launch_step2(teuk_ctx* c, int from, int step_off) {
    StepParams P;
    P.u_in = c->state(from);
    P.u_out = c->state(from ^ 1);
    P.coef_i = c->dptr(c->lay.coef_i);
    P.coef_h = c->dptr(c->lay.coef_h);
    P.cj = c->dptr(c->lay.cj);
    P.n_r = c->n_r; P.n_theta = c->n_theta; P.pitch = c->lay.pitch; P.plane = c->lay.plane;
    P.ti = c->ti; P.tj = c->tj;
    P.sigma = (std::abs(c->m) % 2 == 0) ? 1.0 : -1.0;
    P.tq_half = 0.25 * c->dt;
    P.tq_full = 0.5 * c->dt;
    P.obs_raw = c->obs_cap > 0 ? c->dptr(c->lay.obs_raw) : nullptr;
    P.step_base = c->step_base();
    P.obs_cap = c->obs_cap;
    P.step_off = step_off;
    P.oi = c->oi; P.oj = c->oj;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = c->grid2; cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = c->smem2; cfg.stream = c->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = c->opt_pdl == 1 ? 1 : 0;
    void* args[] = {&c->tm2_state[from], &c->tm2_ch, &P};
    cudaError_t le = cudaLaunchKernelExC(&cfg, tb2_step_fn(c->ti, c->tj), args);
    if (le != cudaSuccess) return cuda_fail(le, "cudaLaunchKernelExC(step2 kernel)", __LINE__);
    return TEUK_OK;
}

static int upload_initial(teuk_ctx* c, const double* d_src, int limbs_in) {
    long total = 4L * c->L * c->n_theta * c->n_r;
    load_state_kernel<<<(unsigned)((total + 255) / 256), 256, 0, c->stream>>>(
        d_src, c->state(0), c->n_r, c->n_theta, c->lay.pitch, c->lay.plane, c->L, limbs_in);
    c->launches++;
    if (cudaGetLastError() != cudaSuccess) return TEUK_ECUDA;
    CK(cudaMemsetAsync(c->step_base(), 0, 32, c->stream));
    c->cur = 0; c->steps_done = 0; c->series_origin = 0; c->nonfinite = false;
    if (!c->have_init) {
        int rc = choose_geometry(c);
        if (rc != TEUK_OK) return rc;
    }
    c->have_init = true;
    return TEUK_OK;
}

extern "C" int teuk_set_initial_device(teuk_ctx* c, const double* d_planes, int limbs_in) {
    if (!c || !d_planes || (limbs_in != 1 && limbs_in != c->L)) return TEUK_EINVAL;
    return upload_initial(c, d_planes, limbs_in);
}

extern "C" int teuk_set_initial(teuk_ctx* c, const double* host_planes, int limbs_in) {
    if (!c || !host_planes || (limbs_in != 1 && limbs_in != c->L)) return TEUK_EINVAL;
    // stage through the not-yet-used second state buffer (large enough: limbs_in <= L, unpadded <= padded)
    size_t bytes = (size_t)4 * limbs_in * c->n_theta * c->n_r * sizeof(double);
    CK(cudaMemcpyAsync(c->state(1), host_planes, bytes, cudaMemcpyHostToDevice, c->stream));
    int rc = upload_initial(c, c->state(1), limbs_in);
    if (rc != TEUK_OK) return rc;
    CK(cudaStreamSynchronize(c->stream));     // the caller may free host_planes
    return TEUK_OK;
}

// launches n iterations starting from state(from) on the stream (captured or not); *flips = number of buffer swaps,
// *nl = step-kernel launches.  Sample offsets are relative to the device-side counter, which the trailing
// advance_kernel moves on by n.
static int launch_iterations(teuk_ctx* c, int from, long n, int* flips, long* nl) {
    long k = 0;
    *flips = 0; *nl = 0;
    while (k < n) {
        int rc;
        if (tb2_active(c) && k + 2 <= n) { rc = launch_step2(c, from, (int)k); k += 2; }
        else { rc = launch_step(c, from, (int)k); k += 1; }
        if (rc != TEUK_OK) return rc;
        from ^= 1; ++*flips; ++*nl;
    }
    advance_kernel<<<1, 1, 0, c->stream>>>(c->step_base(), n);
    return cudaGetLastError() == cudaSuccess ? TEUK_OK : TEUK_ECUDA;
}

static int build_graph(teuk_ctx* c, int parity, long n, cudaGraphExec_t* out) {
    cudaGraph_t g;
    CK(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
    int flips; long nl;
    int rc = launch_iterations(c, parity, n, &flips, &nl);
    cudaError_t e = cudaStreamEndCapture(c->stream, &g);
    if (rc != TEUK_OK || e != cudaSuccess) return TEUK_ECUDA;
    e = cudaGraphInstantiate(out, g, 0);
    cudaGraphDestroy(g);
    return e == cudaSuccess ? TEUK_OK : TEUK_ECUDA;
}

extern "C" int teuk_step(teuk_ctx* c, long n) {
    if (!c || n < 0) return TEUK_EINVAL;
    if (!c->have_init) return TEUK_ESTATE;
    long left = n;
    // the legacy default stream cannot be captured: plain launches there
    const long K = (c->stream == nullptr || c->stream == cudaStreamLegacy) ? 0 : c->graph_steps;
    while (left > 0) {
        const long chunk = (K > 0 && left >= K) ? K : left;
        // launches and buffer swaps of a chunk (a two-iteration launch swaps once)
        const long nl = tb2_active(c) ? chunk / 2 + (chunk & 1) : chunk;
        const bool graphable = K > 0 && chunk >= 2 && (chunk == K || c->graph[c->cur].size() < 16);
        if (graphable) {
            auto it = c->graph[c->cur].find(chunk);
            if (it == c->graph[c->cur].end()) {
                cudaGraphExec_t ge = nullptr;
                int rc = build_graph(c, c->cur, chunk, &ge);
                if (rc != TEUK_OK) return rc;
                it = c->graph[c->cur].emplace(chunk, ge).first;
            }
            CK(cudaGraphLaunch(it->second, c->stream));
        } else {
            int flips; long nl2;
            int rc = launch_iterations(c, c->cur, chunk, &flips, &nl2);
            if (rc != TEUK_OK) return rc;
        }
        c->cur ^= (int)(nl & 1);
        c->launches += (c->mp_cap > 0 ? 2 * nl : nl) + 1;
        left -= chunk;
    }
    c->steps_done += n;
    return TEUK_OK;
}

extern "C" int teuk_read_device(teuk_ctx* c, double* d_planes) {
    if (!c || !d_planes) return TEUK_EINVAL;
    if (!c->have_init) return TEUK_ESTATE;
    long total = 4L * c->L * c->n_theta * c->n_r;
    store_state_kernel<<<(unsigned)((total + 255) / 256), 256, 0, c->stream>>>(
        c->state(c->cur), d_planes, c->n_r, c->n_theta, c->lay.pitch, c->lay.plane, 4 * c->L);
    c->launches++;
    return cudaGetLastError() == cudaSuccess ? TEUK_OK : TEUK_ECUDA;
}

extern "C" int teuk_read(teuk_ctx* c, double* host_planes) {
    if (!c || !host_planes) return TEUK_EINVAL;
    if (!c->have_init) return TEUK_ESTATE;
    // unpad through the idle state buffer, then one D2H copy
    double* tmp = c->state(c->cur ^ 1);
    int rc = teuk_read_device(c, tmp);
    if (rc != TEUK_OK) return rc;
    size_t bytes = (size_t)4 * c->L * c->n_theta * c->n_r * sizeof(double);
    CK(cudaMemcpyAsync(host_planes, tmp, bytes, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return TEUK_OK;
}

// halo strips of the current state: buf is double[4][L][n_theta][n_cols] (i fastest), columns i_first .. i_first + n_cols - 1
__global__ void columns_kernel(double* __restrict__ state, double* __restrict__ buf, int i_first, int n_cols, int n_theta,
                               int pitch, long plane, int planes, int write) {
    long idx = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (idx >= (long)planes * n_theta * n_cols) return;
    int ic = (int)(idx % n_cols);
    long rest = idx / n_cols;
    int j = (int)(rest % n_theta);
    int pl = (int)(rest / n_theta);
    long g = pl * plane + (long)j * pitch + i_first + ic;
    if (write) state[g] = buf[idx];
    else buf[idx] = state[g];
}

static int columns_io(teuk_ctx* c, int i_first, int n_cols, double* d_buf, int write) {
    if (!c || !d_buf || i_first < 0 || n_cols < 1 || (long)i_first + n_cols > c->n_r) return TEUK_EINVAL;
    if (!c->have_init) return TEUK_ESTATE;
    long total = 4L * c->L * c->n_theta * n_cols;
    columns_kernel<<<(unsigned)((total + 255) / 256), 256, 0, c->stream>>>(c->state(c->cur), d_buf, i_first, n_cols, c->n_theta,
                                                                          c->lay.pitch, c->lay.plane, 4 * c->L, write);
    c->launches++;
    return cudaGetLastError() == cudaSuccess ? TEUK_OK : TEUK_ECUDA;
}
extern "C" int teuk_read_columns_device(teuk_ctx* c, int i_first, int n_cols, double* d_out) {
    return columns_io(c, i_first, n_cols, d_out, 0);
}
extern "C" int teuk_write_columns_device(teuk_ctx* c, int i_first, int n_cols, const double* d_in) {
    return columns_io(c, i_first, n_cols, const_cast<double*>(d_in), 1);
}

extern "C" int teuk_observe(teuk_ctx* c, double* host_out, long max_samples, long* count) {
    if (!c || !host_out || !count || max_samples < 0) return TEUK_EINVAL;
    long n = c->steps_done - c->series_origin;
    if (n > c->obs_cap) n = c->obs_cap;
    if (n > max_samples) n = max_samples;
    if (n > 0) {
        unsigned blocks = (unsigned)((n * 4 + 127) / 128);
        const double* raw = c->dptr(c->lay.obs_raw);
        double* out = c->dptr(c->lay.obs_out);
        if (c->L == 1) observer_combine_kernel<1><<<blocks, 128, 0, c->stream>>>(raw, out, n, c->wr, c->wt, c->flag());
        else if (c->L == 2) observer_combine_kernel<2><<<blocks, 128, 0, c->stream>>>(raw, out, n, c->wr, c->wt, c->flag());
        else observer_combine_kernel<4><<<blocks, 128, 0, c->stream>>>(raw, out, n, c->wr, c->wt, c->flag());
        c->launches++;
        if (cudaGetLastError() != cudaSuccess) return TEUK_ECUDA;
        CK(cudaMemcpyAsync(host_out, out, (size_t)n * 4 * c->L * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        int flag = 0;
        CK(cudaMemcpyAsync(&flag, c->flag(), sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        CK(cudaStreamSynchronize(c->stream));
        if (flag) c->nonfinite = true;
    } else {
        CK(cudaStreamSynchronize(c->stream));
    }
    *count = n;
    return c->nonfinite ? TEUK_ENONFINITE : TEUK_OK;
}

// ---- NEXT-2: multipole-projection observer ------------------------------------------------------------------
static R4 q_factorial(int n) {
    R4 r = from_double<4>(1.0);
    for (int k = 2; k <= n; ++k) r = mul_d(r, (double)k);
    return r;
}
static double binom_d(int n, int k) {          // exact in fp64 for the small arguments used here (n <= 40)
    if (k < 0 || k > n) return 0.0;
    double r = 1.0;
    for (int i = 1; i <= k; ++i) r = r * (double)(n - k + i) / (double)i;
    return nearbyint(r);
}
static R4 q_powi(const R4& x, int n) {
    R4 r = from_double<4>(1.0);
    for (int i = 0; i < n; ++i) r = mul(r, x);
    return r;
}
// _sY_lm(theta, 0) from the Goldberg closed form written in sin, cos of theta/2 (regular at the poles)
static R4 q_swsh(int s, int l, int m, const R4& sh, const R4& ch, const R4& pi) {
    R4 num = mul_d(mul(q_factorial(l + m), q_factorial(l - m)), (double)(2 * l + 1));
    R4 den = mul(scale2(pi, 4.0), mul(q_factorial(l + s), q_factorial(l - s)));
    R4 pref = msqrt(div(num, den));
    if (m & 1) pref = neg(pref);
    R4 tot = from_double<4>(0.0);
    for (int r = 0; r <= l - s; ++r) {
        int k = r + s - m;
        if (k < 0 || k > l + s) continue;
        double cf = binom_d(l - s, r) * binom_d(l + s, k) * (((l - r - s) & 1) ? -1.0 : 1.0);
        tot = add(tot, mul_d(mul(q_powi(sh, 2 * l - 2 * r - s + m), q_powi(ch, 2 * r + s - m)), cf));
    }
    return mul(pref, tot);
}

// cos(pi p / N) for integers p, N in quad-double: the angle is reduced to [0, pi/2] with integer arithmetic first
static R4 q_cos_pi_frac(long p, long N, const R4& pi) {
    p %= 2 * N;
    if (p < 0) p += 2 * N;
    if (p > N) p = 2 * N - p;                  // cos(2 pi - x) = cos x
    bool negate = false;
    if (2 * p > N) { p = N - p; negate = true; }   // cos(pi - x) = -cos x
    R4 sn, cs;
    q_sincos(div(mul_d(pi, (double)p), from_double<4>((double)N)), sn, cs);
    return negate ? neg(cs) : cs;
}
// Fejer's first rule on the cell-centred grid: w_j = (2/N) [1 - 2 sum_{k=1}^{N/2} cos(2 k theta_j) / (4 k^2 - 1)];
// exact for polynomials of degree < N in cos(theta), so the dominant multipole does not leak into the others.
static R4 q_fejer_weight(int j, int N, const R4& pi) {
    R4 acc = from_double<4>(1.0);
    for (long k = 1; k <= N / 2; ++k) {
        R4 ck = q_cos_pi_frac(k * (2L * j + 1), N, pi);           // 2 k theta_j = pi k (2j + 1) / N
        acc = sub(acc, div(scale2(ck, 2.0), from_double<4>((double)(4 * k * k - 1))));
    }
    return div(scale2(acc, 2.0), from_double<4>((double)N));
}

extern "C" int teuk_set_multipole_observer(teuk_ctx* c, double rstar_obs, int n_ell, long capacity) {
    if (!c || n_ell < 1 || n_ell > MP_MAX_ELL || capacity < 0 || capacity > c->cap_alloc || !std::isfinite(rstar_obs))
        return TEUK_EINVAL;
    R4 x = sub(div(sub(from_double<4>(rstar_obs), c->C.rmin), c->C.dr), from_double<4>((double)c->i_lo));
    int i0 = (int)std::floor(x.x[0]);
    if (x.x[0] < 0 || x.x[0] > c->n_r - 1) return TEUK_EINVAL;
    if (i0 > c->n_r - 2) i0 = c->n_r - 2;
    c->mp_wr = sub(x, from_double<4>((double)i0));
    c->mp_i = i0; c->mp_n = n_ell; c->mp_cap = capacity;
    // weights Q_k(theta_j) = 2 pi w_j _sY_{l_min + k, m}(theta_j), w_j = Fejer-1 weights, in quad-double on the host
    QConst qc = q_constants();
    const int nt = c->n_theta, L = c->L;
    const int lmin = std::max(std::abs(c->s), std::abs(c->m));
    std::vector<double> q((size_t)MP_MAX_ELL * L * nt, 0.0);
    R4 two_pi = scale2(qc.pi, 2.0);
    for (int j = 0; j < nt; ++j) {
        R4 th = mul(c->C.dth, add(from_double<4>((double)j), from_double<4>(0.5)));
        R4 sh, ch;
        q_sincos(scale2(th, 0.5), sh, ch);
        R4 wf = mul(two_pi, q_fejer_weight(j, nt, qc.pi));
        for (int k = 0; k < n_ell; ++k) {
            R4 w = mul(wf, q_swsh(c->s, lmin + k, c->m, sh, ch, qc.pi));
            for (int l = 0; l < L; ++l) q[((size_t)k * L + l) * nt + j] = w.x[l];
        }
    }
    c->drop_graphs();
    CK(cudaMemcpyAsync(c->dptr(c->lay.mp_q), q.data(), q.size() * 8, cudaMemcpyHostToDevice, c->stream));
    // the sample counter is shared with the point observer: BOTH series restart here, as at teuk_set_observer
    CK(cudaMemsetAsync(c->step_base(), 0, 32, c->stream));
    c->series_origin = c->steps_done;
    c->nonfinite = false;
    CK(cudaStreamSynchronize(c->stream));
    return TEUK_OK;
}

extern "C" int teuk_observe_multipoles(teuk_ctx* c, double* host_out, long max_samples, long* count) {
    if (!c || !host_out || !count || max_samples < 0) return TEUK_EINVAL;
    long n = c->steps_done - c->series_origin;
    if (n > c->mp_cap) n = c->mp_cap;
    if (n > max_samples) n = max_samples;
    if (n > 0)
        CK(cudaMemcpyAsync(host_out, c->dptr(c->lay.mp_series), (size_t)n * c->mp_n * 2 * c->L * sizeof(double),
                           cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    *count = n;
    return TEUK_OK;
}

extern "C" int teuk_steps_done(teuk_ctx* c, long* n) {
    if (!c || !n) return TEUK_EINVAL;
    *n = c->steps_done;
    return TEUK_OK;
}
extern "C" int teuk_launch_count(teuk_ctx* c, long* n) {
    if (!c || !n) return TEUK_EINVAL;
    *n = c->launches;
    return TEUK_OK;
}
extern "C" int teuk_step_geometry(teuk_ctx* c, long* o) {
    if (!c || !o) return TEUK_EINVAL;
    if (!c->have_init) return TEUK_ESTATE;
    o[0] = c->ti; o[1] = c->tj; o[2] = c->threads; o[3] = c->grid.x; o[4] = c->grid.y; o[5] = (long)c->smem;
    if (c->use_tb2) { o[3] = c->grid2.x; o[4] = c->grid2.y; o[5] = (long)c->smem2; }
    return TEUK_OK;
}
extern "C" void teuk_destroy(teuk_ctx* c) {
    if (!c) return;
    cudaStreamSynchronize(c->stream);      // the caller may recycle the workspace as soon as this returns
    c->drop_graphs();
    delete c;
}
extern "C" const char* teuk_strerror(int code) {
    switch (code) {
        case TEUK_OK: return "ok";
        case TEUK_EINVAL: return "invalid argument";
        case TEUK_ENOMEM: return "out of memory";
        case TEUK_ECUDA: return "CUDA error";
        case TEUK_ESTATE: return "call not valid in this state";
        case TEUK_ENONFINITE: return "non-finite observer sample";
        case TEUK_ECAPACITY: return "request exceeds the fixed capacity of the static scratch array";
        default: return "unknown error";
    }
}

// ------------------------------------------------------------------------------------ test hooks
extern "C" int teuk_get_tables(teuk_ctx* c, int half, double* host_out) {
    if (!c || !host_out) return TEUK_EINVAL;
    int rows = half ? c->n_r - 1 : c->n_r;
    size_t padded = (size_t)8 * c->L * c->lay.plane * sizeof(double);
    double* tmp = nullptr;
    if (cudaMalloc(&tmp, padded) != cudaSuccess) return TEUK_ENOMEM;
    int rc = launch_coef_any(c, half ? 1 : 0, 0, tmp);
    std::vector<double> h((size_t)8 * c->L * c->lay.plane);
    if (rc == TEUK_OK && (cudaMemcpyAsync(h.data(), tmp, padded, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess ||
                          cudaStreamSynchronize(c->stream) != cudaSuccess))
        rc = TEUK_ECUDA;
    cudaFree(tmp);
    if (rc != TEUK_OK) return rc;
    for (int pl = 0; pl < 8 * c->L; ++pl)
        for (int j = 0; j < c->n_theta; ++j)
            for (int i = 0; i < rows; ++i)
                host_out[((size_t)pl * c->n_theta + j) * rows + i] = h[(size_t)pl * c->lay.plane + (size_t)j * c->lay.pitch + i];
    return TEUK_OK;
}

// test hook: recomputed folded coefficients of one family written as 8 planes [n_theta][pitch]
__global__ void rc_tables_kernel(const double* __restrict__ isig, const double* __restrict__ rt, const double* __restrict__ th,
                                 int cols, int n_theta, int pitch, long plane, double* __restrict__ out, int full) {
    int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= cols) return;
    RcCoef cf;
    // full = variant (c): 1/Sigma from the R^2 and a^2 Delta tables, exactly as step_kernel_f64_rc<.., true> forms it
    double is = full ? rsqrt_refined(fma(-rt[15 * pitch + i], th[j], rt[14 * pitch + i])) : isig[(long)j * pitch + i];
    rc_eval(cf, is, rt + i, pitch, th[j], th[n_theta + j], th[2 * n_theta + j]);
    for (int q = 0; q < 8; ++q) out[q * plane + (long)j * pitch + i] = cf.c[q];
}

extern "C" int teuk_get_folded(teuk_ctx* c, int half, int coef_variant, double* host_out) {
    if (!c || !host_out || c->L != 1 || coef_variant < 0 || coef_variant > 2) return TEUK_EINVAL;
    if (coef_variant == 0 ? !c->has_planes : !c->has_rc) return TEUK_EINVAL;      // supply not resident in this handle
    int rows = half ? c->n_r - 1 : c->n_r;
    size_t n = (size_t)8 * c->lay.plane;
    std::vector<double> h(n);
    const double* src = c->dptr(half ? c->lay.coef_h : c->lay.coef_i);
    double* tmp = nullptr;
    if (coef_variant >= 1) {
        if (cudaMalloc(&tmp, n * 8) != cudaSuccess) return TEUK_ENOMEM;
        rc_tables_kernel<<<dim3((rows + 127) / 128, c->n_theta), 128, 0, c->stream>>>(
            c->dptr(c->lay.rc_isig) + (size_t)(half ? 1 : 0) * c->lay.plane,
            c->dptr(c->lay.rc_rt) + (size_t)(half ? 1 : 0) * RC_NT * c->lay.pitch, c->dptr(c->lay.rc_th), rows, c->n_theta,
            c->lay.pitch, c->lay.plane, tmp, coef_variant == 2);
        src = tmp;
    }
    cudaError_t e = cudaMemcpyAsync(h.data(), src, n * 8, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (tmp) cudaFree(tmp);
    if (e != cudaSuccess) return TEUK_ECUDA;
    for (int pl = 0; pl < 8; ++pl)
        for (int j = 0; j < c->n_theta; ++j)
            for (int i = 0; i < rows; ++i)
                host_out[((size_t)pl * c->n_theta + j) * rows + i] = h[(size_t)pl * c->lay.plane + (size_t)j * c->lay.pitch + i];
    return TEUK_OK;
}

extern "C" int teuk_get_radial(teuk_ctx* c, double* host_r, double* host_delta) {
    if (!c || !host_r || !host_delta) return TEUK_EINVAL;
    size_t bytes = (size_t)4 * (2 * c->n_r - 1) * sizeof(double);
    CK(cudaMemcpyAsync(host_r, c->dptr(c->lay.r_tab), bytes, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaMemcpyAsync(host_delta, c->dptr(c->lay.d_tab), bytes, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return TEUK_OK;
}

template <int L> MPX Real<L> mp_apply(int op, const Real<L>& x, const Real<L>& y) {
    switch (op) {
        case 0: return add(x, y);
        case 1: return sub(x, y);
        case 2: return mul(x, y);
        case 3: return div(x, y);
        case 4: return msqrt(x);
        default: return mul_d(x, y.x[0]);
    }
}
template <int L> __global__ void mp_op_kernel(int op, const double* a, const double* b, double* out, long n) {
    long k = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (k >= n) return;
    Real<L> x, y;
    for (int l = 0; l < L; ++l) { x.x[l] = a[k * L + l]; y.x[l] = b[k * L + l]; }
    Real<L> r = mp_apply<L>(op, x, y);
    for (int l = 0; l < L; ++l) out[k * L + l] = r.x[l];
}
template <int L> static int mp_op_host(int op, const double* a, const double* b, double* out, long n) {
    for (long k = 0; k < n; ++k) {
        Real<L> x, y;
        for (int l = 0; l < L; ++l) { x.x[l] = a[k * L + l]; y.x[l] = b[k * L + l]; }
        Real<L> r = mp_apply<L>(op, x, y);
        for (int l = 0; l < L; ++l) out[k * L + l] = r.x[l];
    }
    return TEUK_OK;
}
template <int L> static int mp_op_dev(int op, const double* a, const double* b, double* out, long n) {
    double *da = nullptr, *db = nullptr, *dout = nullptr;
    size_t bytes = (size_t)n * L * sizeof(double);
    if (cudaMalloc(&da, bytes) != cudaSuccess || cudaMalloc(&db, bytes) != cudaSuccess ||
        cudaMalloc(&dout, bytes) != cudaSuccess) {
        cudaFree(da); cudaFree(db); cudaFree(dout);
        return TEUK_ENOMEM;
    }
    cudaMemcpy(da, a, bytes, cudaMemcpyHostToDevice);
    cudaMemcpy(db, b, bytes, cudaMemcpyHostToDevice);
    mp_op_kernel<L><<<(unsigned)((n + 127) / 128), 128>>>(op, da, db, dout, n);
    cudaError_t e = cudaMemcpy(out, dout, bytes, cudaMemcpyDeviceToHost);
    cudaFree(da); cudaFree(db); cudaFree(dout);
    return e == cudaSuccess ? TEUK_OK : TEUK_ECUDA;
}
extern "C" int teuk_test_mp_op(int op, int L, const double* a, const double* b, double* out, long n, int on_device) {
    if (!a || !b || !out || n < 0 || op < 0 || op > 5 || (L != 2 && L != 4)) return TEUK_EINVAL;
    if (L == 2) return on_device ? mp_op_dev<2>(op, a, b, out, n) : mp_op_host<2>(op, a, b, out, n);
    return on_device ? mp_op_dev<4>(op, a, b, out, n) : mp_op_host<4>(op, a, b, out, n);
}

extern "C" int teuk_test_mp_fn(int fn, const double* a, double* out) {
    if (!a || !out || fn < 0 || fn > 5) return TEUK_EINVAL;
    static QConst qc = q_constants();
    R4 x, r, t;
    for (int l = 0; l < 4; ++l) x.x[l] = a[l];
    switch (fn) {
        case 0: r = q_exp(x, qc.ln2); break;
        case 1: r = q_log(x, qc.ln2); break;
        case 2: q_sincos(x, r, t); break;
        case 3: q_sincos(x, t, r); break;
        case 4: r = qc.pi; break;
        default: r = qc.ln2; break;
    }
    for (int l = 0; l < 4; ++l) out[l] = r.x[l];
    return TEUK_OK;
}

// FP64 issue-rate microbenchmark: 8 independent register chains per thread
template <int KIND> __global__ void fp64_chain_kernel(long iters, double seed, double* sink) {
    double x0 = seed, x1 = seed + 1, x2 = seed + 2, x3 = seed + 3, x4 = seed + 4, x5 = seed + 5, x6 = seed + 6, x7 = seed + 7;
    const double m = 1.0000000001, c = 1e-9;
    for (long i = 0; i < iters; ++i) {
        if (KIND == 0) {
            x0 = __fma_rn(x0, m, c); x1 = __fma_rn(x1, m, c); x2 = __fma_rn(x2, m, c); x3 = __fma_rn(x3, m, c);
            x4 = __fma_rn(x4, m, c); x5 = __fma_rn(x5, m, c); x6 = __fma_rn(x6, m, c); x7 = __fma_rn(x7, m, c);
        } else if (KIND == 1) {
            x0 = __dadd_rn(x0, c); x1 = __dadd_rn(x1, c); x2 = __dadd_rn(x2, c); x3 = __dadd_rn(x3, c);
            x4 = __dadd_rn(x4, c); x5 = __dadd_rn(x5, c); x6 = __dadd_rn(x6, c); x7 = __dadd_rn(x7, c);
        } else {
            x0 = __dmul_rn(x0, m); x1 = __dmul_rn(x1, m); x2 = __dmul_rn(x2, m); x3 = __dmul_rn(x3, m);
            x4 = __dmul_rn(x4, m); x5 = __dmul_rn(x5, m); x6 = __dmul_rn(x6, m); x7 = __dmul_rn(x7, m);
        }
    }
    double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456) *sink = s;
}
extern "C" int teuk_bench_fp64(int kind, long iters, double* inst_per_s, void* cuda_stream) {
    if (!inst_per_s || iters <= 0 || kind < 0 || kind > 2) return TEUK_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double* sink = nullptr;
    CK(cudaMalloc(&sink, 8));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    int blocks = sms * 8, threads = 256;
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0, st);
        if (kind == 0) fp64_chain_kernel<0><<<blocks, threads, 0, st>>>(iters, 1.0, sink);
        else if (kind == 1) fp64_chain_kernel<1><<<blocks, threads, 0, st>>>(iters, 1.0, sink);
        else fp64_chain_kernel<2><<<blocks, threads, 0, st>>>(iters, 1.0, sink);
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    if (cudaGetLastError() != cudaSuccess) return TEUK_ECUDA;
    *inst_per_s = (double)blocks * threads * 8.0 * (double)iters / (best * 1e-3);
    return TEUK_OK;
}

// ------------------------------------------------------------------------------------ allocation-free entry point
// teuk_get_folded_static (include/teuk.h): rc_tables_kernel writing into a file-scope device array instead of a
// cudaMalloc'ed buffer.  In HOST code `g_static_scratch` is only a stand-in for the symbol, not a device address: the
// address a kernel can use comes from cudaGetSymbolAddress, looked up once per device with that device current.
static __device__ __align__(256) double g_static_scratch[TEUK_STATIC_SCRATCH_DOUBLES];

static int static_scratch_ptr(double** out) {
    constexpr int MAX_DEV = 64;
    static double* ptr[MAX_DEV] = {nullptr};
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEV) return TEUK_ECUDA;
    if (!ptr[dev]) {
        double* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_scratch);      // resolves for the CURRENT device
        if (e != cudaSuccess || !p) return cuda_fail(e, "cudaGetSymbolAddress(g_static_scratch)", __LINE__);
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return TEUK_OK;
}

extern "C" int teuk_get_folded_static(teuk_ctx* c, int half, int coef_variant, double* host_out) {
    if (!c || !host_out || c->L != 1 || coef_variant < 1 || coef_variant > 2 || !c->has_rc) return TEUK_EINVAL;
    const size_t n = (size_t)8 * c->lay.plane;                       // 8 planes of n_theta x pitch doubles
    if (n > (size_t)TEUK_STATIC_SCRATCH_DOUBLES) return TEUK_ECAPACITY;
    double* scratch = nullptr;
    int rc = static_scratch_ptr(&scratch);
    if (rc != TEUK_OK) return rc;
    const int rows = half ? c->n_r - 1 : c->n_r;
    // the array keeps the previous call's contents: clear what this call uses (the kernel writes columns < rows only)
    CK(cudaMemsetAsync(scratch, 0, n * sizeof(double), c->stream));
    rc_tables_kernel<<<dim3((rows + 127) / 128, c->n_theta), 128, 0, c->stream>>>(
        c->dptr(c->lay.rc_isig) + (size_t)(half ? 1 : 0) * c->lay.plane,
        c->dptr(c->lay.rc_rt) + (size_t)(half ? 1 : 0) * RC_NT * c->lay.pitch, c->dptr(c->lay.rc_th), rows, c->n_theta,
        c->lay.pitch, c->lay.plane, scratch, coef_variant == 2);
    c->launches++;
    if (cudaGetLastError() != cudaSuccess) return TEUK_ECUDA;
    // unpad on the way out: 8 * n_theta rows of `rows` doubles, source row stride = pitch (planes are contiguous: plane = n_theta * pitch)
    CK(cudaMemcpy2DAsync(host_out, (size_t)rows * sizeof(double), scratch, (size_t)c->lay.pitch * sizeof(double),
                         (size_t)rows * sizeof(double), (size_t)8 * c->n_theta, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return TEUK_OK;
}
