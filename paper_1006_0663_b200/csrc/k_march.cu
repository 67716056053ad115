// Instantiations of the fp64 column-march step kernel (step_kernel_march.cuh).
#include "kernels.h"
#include "step_kernel_march.cuh"

namespace tk {

const void* march_step_fn(int rt_in_registers) {
    return rt_in_registers ? (const void*)step_kernel_f64_march<true> : (const void*)step_kernel_f64_march<false>;
}

}  // namespace tk
