// Instantiations of the generic fused step kernels for L = 4 limbs (see step_kernel.cuh); one translation unit per
// precision so the library compiles in parallel.
#include "kernels.h"
#include "step_kernel.cuh"

namespace tk {

// qd: default = the pair kernel (two threads per point) on 16 x 16 tiles, 256 threads x 2 blocks/SM: half the code per
// thread and eight warps per block walking it together (the instruction fetch was the qd kernel's largest stall) --
// cfg 4: 1.09e9 updates/s against 8.3e8 for the one-thread-per-point kernel (variant 4: 128 threads x 3 blocks, 168
// registers, itself 1.9x faster than 256 x 1 with 254 registers, variant 1).  Other pair shapes stay selectable by tile.
const void* generic_step_fn_4(int variant, int ti, int tj, int* threads) {
    if (variant == 0 || variant == 3) {
        *threads = 256;
        if (ti == 16 && tj == 16) return (const void*)step_kernel_pair<4, 16, 16, 256, 2>;
        if (ti == 32 && tj == 8) return (const void*)step_kernel_pair<4, 32, 8, 256, 2>;
        if (ti == 16 && tj == 8) { *threads = 128; return (const void*)step_kernel_pair<4, 16, 8, 128, 4>; }
    }
    *threads = 256;
    if (variant == 1) return (const void*)step_kernel<4, 0, 0, 256, 1>;
    *threads = 128;
    if (variant == 2) return (const void*)step_kernel<4, 0, 0, 128, 4>;
    if (variant == 4 && ti == 16 && tj == 8) return (const void*)step_kernel<4, 16, 8, 128, 3>;
    return (const void*)step_kernel<4, 0, 0, 128, 3>;
}
const void* generic_col_fn_4(int variant, int* threads) {
    if (variant != 4) { *threads = 256; return (const void*)step_kernel_col_pair<4, 256, 2>; }
    *threads = 128;
    return (const void*)step_kernel_col<4, 128, 3>;
}

}  // namespace tk
