// Instantiations of the generic fused step kernels for L = 1 limbs (see step_kernel.cuh); one translation unit per
// precision so the library compiles in parallel.
#include "kernels.h"
#include "step_kernel.cuh"

namespace tk {

const void* generic_step_fn_1(int, int, int, int* threads) {
    *threads = 256;
    return (const void*)step_kernel<1, 0, 0, 256, 4>;
}
const void* generic_col_fn_1(int* threads) {
    *threads = 256;
    return (const void*)step_kernel_col<1, 256, 2>;
}

}  // namespace tk
