// Instantiation of the fp64 column-march step kernel (step_kernel_march.cuh).
#include "kernels.h"
#include "step_kernel_march.cuh"

namespace tk {

const void* march_step_fn() { return (const void*)step_kernel_f64_march<2>; }

}  // namespace tk
