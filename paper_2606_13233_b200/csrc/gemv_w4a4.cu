// gemv_w4a4.cu -- instantiates the KMODE_W4A4_I8 GEMV kernels (all M = 1..8, R = 1, 2).
#include "gemv_dispatch.cuh"

namespace nvfp4 {

cudaError_t launch_gemv_w4a4(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st) {
    return launch_m<KMODE_W4A4_I8>(p, M, R, grid, threads, smem, st);
}

}  // namespace nvfp4
