// gemv_w4a4h.cu -- instantiates the KMODE_W4A4_H GEMV kernels (all M = 1..8, R = 1, 2, 4).
#include "gemv_dispatch.cuh"

namespace nvfp4 {

cudaError_t launch_gemv_w4a4h(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st) {
    return launch_m<KMODE_W4A4_H>(p, M, R, grid, threads, smem, st);
}

}  // namespace nvfp4
