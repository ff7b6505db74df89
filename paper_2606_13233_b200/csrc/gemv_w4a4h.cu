// gemv_w4a4h.cu -- instantiates the KMODE_W4A4_H GEMV kernel (F2FP + HFMA2; used at M = 1 only, R = 1).
#include "gemv_dispatch.cuh"

namespace nvfp4 {

cudaError_t launch_gemv_w4a4h(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st) {
    if (M != 1) return cudaErrorInvalidValue;
    return launch_r<KMODE_W4A4_H, 1>(p, R, grid, threads, smem, st);
}

}  // namespace nvfp4
