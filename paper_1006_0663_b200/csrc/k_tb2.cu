// Instantiations of the fp64 temporally blocked (two iterations per launch) step kernel (step_kernel_tb2.cuh).
#include "kernels.h"
#include "step_kernel_tb2.cuh"

namespace tk {

const void* tb2_step_fn(int ti, int tj) {
    if (ti != 32) return nullptr;
    if (tj == 8) return (const void*)step2_kernel_f64_tma<32, 8>;
    if (tj == 16) return (const void*)step2_kernel_f64_tma<32, 16>;
    return nullptr;
}

}  // namespace tk
