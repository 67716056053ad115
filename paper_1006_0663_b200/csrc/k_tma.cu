// Instantiations of the fp64 TMA step kernels (step_kernel_tma.cuh).
#include "kernels.h"
#include "step_kernel_tma.cuh"

namespace tk {

const void* tma_step_fn(int ti, int tj) {
    if (ti != 32) return nullptr;
    if (tj == 8) return (const void*)step_kernel_f64_tma<32, 8>;
    if (tj == 16) return (const void*)step_kernel_f64_tma<32, 16>;
    return nullptr;
}
const void* rc_step_fn(int ti, int tj, int full) {
    if (ti != 32) return nullptr;
    if (tj == 8) return full ? (const void*)step_kernel_f64_rc<32, 8, true> : (const void*)step_kernel_f64_rc<32, 8, false>;
    if (tj == 16) return full ? (const void*)step_kernel_f64_rc<32, 16, true> : (const void*)step_kernel_f64_rc<32, 16, false>;
    return nullptr;
}
const void* col_tma_fn(int ti) {
    if (ti == 8) return (const void*)step_kernel_f64_col_tma<8>;
    if (ti == 12) return (const void*)step_kernel_f64_col_tma<12>;
    if (ti == 16) return (const void*)step_kernel_f64_col_tma<16>;
    return nullptr;
}

const void* col_run_fn(int ti) {      // 256 threads, registers capped for 2 blocks per SM, runs of 4 rows
    if (ti == 16) return (const void*)step_kernel_f64_col_run<16, 4, 256, 2>;
    if (ti == 8) return (const void*)step_kernel_f64_col_run<8, 4, 256, 2>;
    return nullptr;
}

}  // namespace tk
