/* teuk.h — C ABI of libteuk.so: the time step of the m-mode-reduced 2+1D Teukolsky equation as a
 * first-order complex (Phi, Pi) system on an (r*, theta) grid in Kerr background, §III.B
 * (PAPER.md:53-112), at three precisions: fp64, double-double, quad-double.
 * The inversion r(r*), all coefficient planes and every step of the time loop (half step, full step, boundary and
 * polar conditions, observer extraction and interpolation) run in CUDA kernels for sm_100a; there is no CPU fallback.
 * Host arithmetic is limited to set-up scalars and 1-D tables that do not depend on r* (theta tables, stencil and
 * quadrature weights), evaluated once per handle in quad-double.
 *
 * Conventions
 *  - All scalar parameters are fp64 and taken as exact.  Grid: r*_i = rstar_min + i dr*,
 *    dr* = (rstar_max - rstar_min)/(n_r - 1), i = 0..n_r-1; theta_j = (j + 1/2) pi/n_theta.
 *  - State planes: double[4][L][n_theta][n_r], i fastest; fields in the order of Eq. (9)
 *    (PAPER.md:88): Phi_R, Phi_I, Pi_R, Pi_I; L = limbs per real (1, 2, 4), limb 0 leading.
 *  - Every function returns a status code (TEUK_OK = 0, negative on error); out-parameters are
 *    untouched on error.  One handle = one CUDA stream; handles are not thread-safe.
 *  - Pointers named host_* are HOST memory owned by the caller; d_workspace is DEVICE memory owned
 *    by the caller (e.g. a torch tensor) that must outlive the handle; cuda_stream is a borrowed
 *    cudaStream_t (NULL = the legacy default stream, on which CUDA graphs are not used).
 */
#ifndef TEUK_H
#define TEUK_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct teuk_ctx teuk_ctx;

enum { TEUK_FP64 = 1, TEUK_DD = 2, TEUK_QD = 4 };      /* value == limbs per real */
enum { TEUK_OK = 0, TEUK_EINVAL = -1, TEUK_ENOMEM = -2, TEUK_ECUDA = -3, TEUK_ESTATE = -4, TEUK_ENONFINITE = -5,
       TEUK_ECAPACITY = -6 /* request exceeds a fixed, documented capacity (teuk_get_folded_static) */ };

/* Bytes of device workspace teuk_create needs for the same (n_r, n_theta, precision, coef_variant, obs_capacity): two
 * state buffers, the coefficient supplies selected by coef_variant, 1-D tables, observer buffers for obs_capacity samples.
 * coef_variant = which coefficient supplies are RESIDENT in the workspace (H1b):
 *   -1  all of them (fp64: 16 stored planes + the two 1/Sigma planes + r-tables), the supply is then chosen per run with
 *       teuk_set_option("coef_variant", ...) and the test hooks can compare them on one handle;
 *    0  the 16 L precomputed folded planes only (the only supply of dd / qd handles);
 *    1, 2  fp64 only: the recompute tables only (two 1/Sigma planes + 1-D tables) -- no stored planes, 128 MiB less on
 *       config 2, 2 GiB less on the 65536 x 256 sweep cell; the handle then steps with that variant and rejects the others.
 * TEUK_EINVAL on bad sizes or variant. */
int teuk_workspace_bytes(int n_r, int n_theta, int precision, int coef_variant, long obs_capacity, size_t *bytes);

/* Build the time-independent tables on the device (r(r*) from Eq. (2); b from Eqs. (6)-(7)
 * PAPER.md:76-80; alpha, gamma, W, kappa of S in Eq. (12) PAPER.md:98 derived from Eq. (1), see
 * DESIGN.md §3), evaluated in quad-double and rounded to L limbs.  M > 0, |a| < M, n_r >= 3,
 * n_theta >= 2, dt > 0, rstar_min < rstar_max, precision in {1, 2, 4}, coef_variant as for teuk_workspace_bytes
 * (only the resident supplies are built); else TEUK_EINVAL.
 * obs_capacity = number of observer samples the workspace was sized for. */
int teuk_create(double M, double a, int s, int m, int n_r, int n_theta, double rstar_min, double rstar_max,
                double dt, int precision, int coef_variant, void *d_workspace, size_t workspace_bytes, long obs_capacity,
                void *cuda_stream, teuk_ctx **out);

/* Radial slab of the same problem (the paper's own domain decomposition):
 * the handle holds columns i_lo .. i_lo + n_win - 1 of the uniform grid of n_r_global nodes on [rstar_min, rstar_max]
 * (r*_i = rstar_min + (i_lo + i) dr*, dr* = (rstar_max - rstar_min)/(n_r_global - 1)): same tables, bit for bit, as the
 * full-grid handle has at those columns.  State planes, teuk_read and the column calls use LOCAL indices 0 .. n_win-1;
 * observer locations stay physical (r*, theta) and must fall inside the slab.  The slab's two edge columns are
 * Dirichlet rows like any handle's: where an edge is a cut and not the physical boundary, the values
 * within k columns of it are invalid k iterations after the caller last refreshed them (r* reach of Eqs. 13-14 is one
 * column per iteration) - the caller keeps a halo and refreshes it with teuk_write_columns_device (see
 * paper_1006_0663_b200/slabs.py).  0 <= i_lo, i_lo + n_win <= n_r_global, n_win >= 3; workspace sized for n_win. */
int teuk_create_slab(double M, double a, int s, int m, int n_r_global, int n_theta, double rstar_min, double rstar_max,
                     double dt, int precision, int coef_variant, int i_lo, int n_win, void *d_workspace,
                     size_t workspace_bytes, long obs_capacity, void *cuda_stream, teuk_ctx **out);

/* Options, only before teuk_set_initial (else TEUK_ESTATE); unknown key or bad value: TEUK_EINVAL.
 *  "graph_steps"   even, >= 2: iterations per captured CUDA graph (default 32); a teuk_step(n) call replays it n / 32
 *                  times and runs the remainder as one more (cached) graph; 0 disables graphs.
 *  "coef_variant"  coefficient supply (H1b).  Default: automatic -- fp64 grids of >= 400 000 points step with variant 1,
 *                  everything else, and every run that sets tile_i / tile_j / use_tma / variant / time_block, with variant 0.
 *                  0 = precomputed folded coefficient planes (192 L B of HBM traffic per update);
 *                  1 = semi-recompute, fp64 only: one 1/Sigma plane per point family + 1-D tables, the eight coefficients
 *                      are rebuilt in registers (80 B per update) -- the fastest fp64 path (column-march kernel);
 *                  2 = full recompute, fp64 only: 1-D tables only, 1/Sigma = rsqrt(R^2 - a^2 Delta sin^2 theta) per point.
 *                  A handle created for one supply (teuk_create's coef_variant >= 0) accepts only that one.
 *  "march"         coef_variant 1: 1 = column-march kernel (default), 0 = the TMA tile kernel for the same supply.
 *  "march_chunk"   column-march kernel: theta rows per work unit; 0 = chosen by the library (default).
 *  "theta_order"   2 = second-order centred theta differences, PAPER.md:110 (default); 10 = the 10th-order 11-point
 *                  operator of PAPER.md:126, needs n_theta >= 5.
 *  "col_run"       fp64, theta_order 10: 1 = a thread owns runs of 4 theta rows of a column (default), 0 = one point per
 *                  thread (the round-1 kernel).
 *  "tile_i", "tile_j"  tile of the tile kernels; 0 = automatic (default).
 *  "use_tma"       fp64: 1 = TMA kernels (default), 0 = the generic tile kernel.
 *  "variant"       dd / qd kernel and launch shape: 0 = default (dd: one thread per point, 32 x 16 tile; qd: the pair
 *                  kernel, two threads per point, 16 x 16 tile); 1, 2 = one thread per point with other launch bounds;
 *                  3 = pair kernel (dd 32 x 16; qd 16 x 16, 32 x 8 or 16 x 8 by tile_i / tile_j); 4 = qd one thread per
 *                  point on its 16 x 8 tile (the default before the pair kernel).  All bitwise identical in result.
 *  "pdl"           programmatic dependent launch of the step kernel (the next step's blocks start their set-up while this
 *                  step drains; results are bitwise the same): 1 = on, 0 = off.  Default: on for the fp64 column-march kernel
 *                  (+2.7 % on config 2), off for the fp64 TMA kernels (measured neutral); other kernels ignore it.
 *  "time_block"    1 = one iteration per launch (default); 2 = EXPERIMENT: two iterations per launch on a shared-memory
 *                  resident tile, fp64 stored-plane TMA path only, else TEUK_EINVAL at teuk_set_initial; an odd last
 *                  iteration and runs with the multipole observer use the one-iteration kernel.  Parity-green but slower
 *                  than coef_variant = 1; kept for the record. */
int teuk_set_option(teuk_ctx *, const char *key, double value);

/* Observer at a fixed location: bilinear interpolation in (r*, theta) from the four
 * surrounding nodes, weights fixed here.  Location must lie inside [r*_0, r*_{n_r-1}] x
 * [theta_0, theta_{n_theta-1}], capacity <= obs_capacity of teuk_create; else TEUK_EINVAL.
 * Resets the recorded series. */
int teuk_set_observer(teuk_ctx *, double rstar_obs, double theta_obs, long capacity);

/* Upload u^0: host_planes is double[4][limbs_in][n_theta][n_r], limbs_in in {1, L} (missing low limbs
 * := 0).  Rows i = 0 and n_r-1 are forced to zero.  Resets step count and series. */
int teuk_set_initial(teuk_ctx *, const double *host_planes, int limbs_in);
/* Same with the planes already in DEVICE memory (no host traffic). */
int teuk_set_initial_device(teuk_ctx *, const double *d_planes, int limbs_in);

/* Advance n >= 0 iterations of Eqs. (13)-(14) with the radial and polar boundary
 * conditions of PAPER.md:112 and one observer sample per iteration; asynchronous on the stream. */
int teuk_step(teuk_ctx *, long n);

/* Download the state, double[4][L][n_theta][n_r]; synchronises the stream. */
int teuk_read(teuk_ctx *, double *host_planes);
/* Copy the state into DEVICE memory of the same layout; asynchronous on the stream. */
int teuk_read_device(teuk_ctx *, double *d_planes);

/* Column strips of the current state (halo exchange between slabs): d_out / d_in are DEVICE buffers
 * double[4][L][n_theta][n_cols], i fastest, holding local columns i_first .. i_first + n_cols - 1; asynchronous on the
 * stream; no boundary condition is applied by the write (never write a physical boundary column).  TEUK_EINVAL if the
 * range leaves the handle's columns, TEUK_ESTATE before teuk_set_initial. */
int teuk_read_columns_device(teuk_ctx *, int i_first, int n_cols, double *d_out);
int teuk_write_columns_device(teuk_ctx *, int i_first, int n_cols, const double *d_in);

/* Observer series: out[count][4][L] = Phi_R, Phi_I, Pi_R, Pi_I at the observer after each completed
 * iteration (sample k <-> t = (k+1) dt), count <= max_samples; synchronises.  Returns
 * TEUK_ENONFINITE (sticky, data still written) if any recorded sample was not finite. */
int teuk_observe(teuk_ctx *, double *host_out, long max_samples, long *count);

/* Multipole-projection observer (the paper's Fig. 1 workload): after every iteration,
 * a_l' = integral of Phi(r*_obs, theta) _sY_l'm(theta) over the sphere, l' = l_min .. l_min + n_ell - 1 with
 * l_min = max(|s|, |m|), 1 <= n_ell <= 9, Fejer's first quadrature rule on the cell-centred theta grid (exact for
 * polynomials of degree < n_theta in cos(theta)), linear interpolation in r*.
 * capacity <= obs_capacity of teuk_create.  Call before teuk_set_initial or between teuk_step calls; the sample index is
 * shared with the point observer: BOTH series restart (count 0, sample 0 = the next completed iteration) at
 * teuk_set_observer, at teuk_set_multipole_observer and at teuk_set_initial. */
int teuk_set_multipole_observer(teuk_ctx *, double rstar_obs, int n_ell, long capacity);
/* host_out[count][n_ell][2][L]: real and imaginary part of a_l' per completed iteration; synchronises. */
int teuk_observe_multipoles(teuk_ctx *, double *host_out, long max_samples, long *count);

int teuk_steps_done(teuk_ctx *, long *n);
/* Number of kernels this handle has launched so far (graph nodes counted per replay). */
int teuk_launch_count(teuk_ctx *, long *n);
/* Launch geometry of the step kernel: out[0..5] = tile_i, tile_j, threads, grid_x, grid_y, smem bytes. */
int teuk_step_geometry(teuk_ctx *, long *out6);
void teuk_destroy(teuk_ctx *);
const char *teuk_strerror(int code);

/* ---- test hooks (used by tests/ only) ------------------------------------------------------- */
/* Coefficient planes as the kernel uses them, double[8][L][n_theta][rows] (rows = n_r, or n_r-1 when
 * half != 0), UNFOLDED: b, alpha_R, alpha_I, gamma_R, gamma_I, W_R, W_I, kappa.  Host output. */
int teuk_get_tables(teuk_ctx *, int half, double *host_out);
/* FOLDED coefficient planes the step kernel multiplies with, double[8][n_theta][rows], fp64 handles only:
 * coef_variant 0 = the stored planes, 1 = rebuilt from the semi-recompute tables by a kernel, 2 = rebuilt with 1/Sigma
 * recomputed as well (full recompute). */
int teuk_get_folded(teuk_ctx *, int half, int coef_variant, double *host_out);
/* ALLOCATION-FREE variant of teuk_get_folded for coef_variant 1 or 2 (the two variants whose planes are rebuilt by a
 * kernel, i.e. the ones teuk_get_folded serves through a cudaMalloc'ed scratch buffer): for callers that must not
 * allocate (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  The kernel's scratch is a
 * file-scope `static __device__` array of TEUK_STATIC_SCRATCH_DOUBLES doubles (4 MiB; every GPU that loads the library
 * holds it until the process exits); its device address is looked up once per device with cudaGetSymbolAddress.  The call
 * allocates nothing on the device or the host (no cudaMalloc / cudaFree / allocating library routine): it clears the part
 * of the scratch it uses, runs the same kernel as teuk_get_folded, and copies the rows straight into host_out
 * (double[8][n_theta][rows], same layout and bit-identical values), then synchronises the handle's stream.
 * Limit: 8 * n_theta * pitch <= TEUK_STATIC_SCRATCH_DOUBLES, pitch = n_r rounded up to 16 (e.g. 1024 x 64, 4096 x 16);
 * larger grids return TEUK_ECAPACITY and touch nothing.  TEUK_EINVAL for non-fp64 handles or coef_variant not in {1, 2}.
 * ALL calls (all handles, all streams of a device) share the one array, which keeps the last call's contents: calls that
 * overlap on the GPU race -- serialise them (one stream, or an event between streams). */
#define TEUK_STATIC_SCRATCH_DOUBLES (512 * 1024)
int teuk_get_folded_static(teuk_ctx *, int half, int coef_variant, double *host_out);
/* r and r - r_+ at the 2 n_r - 1 integer/half points as quad-double limbs, double[2 n_r - 1][4] each. */
int teuk_get_radial(teuk_ctx *, double *host_r, double *host_delta);
/* One arithmetic operation of the multiprecision layer, limbs in/out (L = 2 or 4);
 * op: 0 add, 1 sub, 2 mul, 3 div, 4 sqrt(a), 5 a * b[0];  on_device != 0 runs it in a kernel. */
int teuk_test_mp_op(int op, int L, const double *a, const double *b, double *out, long n, int on_device);
/* Quad-double elementary functions of the setup: fn 0 exp, 1 log, 2 sin, 3 cos, 4 pi, 5 ln2 (host build). */
int teuk_test_mp_fn(int fn, const double *a, double *out);
/* FP64-pipe microbenchmark: register-resident chains of DFMA (kind 0), DADD (1), DMUL (2);
 * returns instructions per second over all SMs (used for the dd/qd roofline denominator). */
int teuk_bench_fp64(int kind, long iters, double *inst_per_s, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
