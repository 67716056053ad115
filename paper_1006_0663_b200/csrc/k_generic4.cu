// Instantiations of the generic fused step kernels for L = 4 limbs (see step_kernel.cuh); one translation unit per
// precision so the library compiles in parallel.
#include "kernels.h"
#include "step_kernel.cuh"

namespace tk {

// qd: 128 threads x 3 blocks/SM (168 registers, a few spills) measured 1.9x faster than 256 x 1 (254 registers)
const void* generic_step_fn_4(int variant, int ti, int tj, int* threads) {
    *threads = 256;
    if (variant == 1) return (const void*)step_kernel<4, 0, 0, 256, 1>;
    *threads = 128;
    if (variant == 2) return (const void*)step_kernel<4, 0, 0, 128, 4>;
    if (ti == 16 && tj == 8) return (const void*)step_kernel<4, 16, 8, 128, 3>;
    return (const void*)step_kernel<4, 0, 0, 128, 3>;
}
const void* generic_col_fn_4(int* threads) {
    *threads = 128;
    return (const void*)step_kernel_col<4, 128, 3>;
}

}  // namespace tk
