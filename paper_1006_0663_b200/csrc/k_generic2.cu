// Instantiations of the generic fused step kernels for L = 2 limbs (see step_kernel.cuh); one translation unit per
// precision so the library compiles in parallel.
#include "kernels.h"
#include "step_kernel.cuh"

namespace tk {

const void* generic_step_fn_2(int variant, int ti, int tj, int* threads) {
    *threads = 256;
    if (variant == 1) { *threads = 128; return (const void*)step_kernel<2, 0, 0, 128, 5>; }
    if (variant == 2) { *threads = 128; return (const void*)step_kernel<2, 0, 0, 128, 6>; }
    if (variant == 3 && ti == 32 && tj == 16) return (const void*)step_kernel_pair<2, 32, 16, 256, 2>;
    if (ti == 32 && tj == 16) return (const void*)step_kernel<2, 32, 16, 256, 2>;
    if (ti == 64 && tj == 8) return (const void*)step_kernel<2, 64, 8, 256, 2>;
    return (const void*)step_kernel<2, 0, 0, 256, 2>;
}
const void* generic_col_fn_2(int* threads) {
    *threads = 256;
    return (const void*)step_kernel_col<2, 256, 2>;
}

}  // namespace tk
