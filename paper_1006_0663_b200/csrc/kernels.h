// Kernel entry points defined in the per-precision translation units (k_generic*.cu, k_tma.cu, k_tb2.cu) so that the
// library builds as independent objects compiled in parallel.  Each function returns the host-side handle of a
// __global__ function template instantiation (for cudaFuncSetAttribute / cudaLaunchKernel[ExC]); nullptr = no such
// instantiation.
#pragma once

namespace tk {

// step_kernel<L, TI, TJ, THREADS, MINB> (step_kernel.cuh); *threads = block size of the chosen instantiation
const void* generic_step_fn_1(int variant, int ti, int tj, int* threads);
const void* generic_step_fn_2(int variant, int ti, int tj, int* threads);
const void* generic_step_fn_4(int variant, int ti, int tj, int* threads);
// step_kernel_col<L, THREADS, MINB> (10th-order theta operator)
const void* generic_col_fn_1(int* threads);
const void* generic_col_fn_2(int* threads);
const void* generic_col_fn_4(int variant, int* threads);   // variant 4: one thread per point; else step_kernel_col_pair
// fp64 TMA kernels (step_kernel_tma.cuh): stored planes, semi-recompute, 10th-order column kernel
const void* tma_step_fn(int ti, int tj);
const void* rc_step_fn(int ti, int tj, int full);     // full = H1b variant (c)
const void* col_tma_fn(int ti);
const void* col_run_fn(int ti);      // row-run variant (a thread owns 4 consecutive theta rows of a column), ti = 8 | 16
// fp64 column-march kernel (step_kernel_march.cuh): semi-recompute supply, no shared-memory tiles
const void* march_step_fn();
// fp64 two-iterations-per-launch kernel (step_kernel_tb2.cuh, NEXT-3)
const void* tb2_step_fn(int ti, int tj);

}  // namespace tk
