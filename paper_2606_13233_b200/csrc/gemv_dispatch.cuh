// gemv_dispatch.cuh -- runtime (M, R) -> template instantiation.  Included by one .cu per mode so
// the families of kernels compile in parallel.  R = 2 (two row tiles per warp step) is instantiated
// for the integer path only (gemv_legalize_config never asks for it elsewhere).
#pragma once
#include "gemv_kernel.cuh"

namespace nvfp4 {

template <int MODE, int M, int R>
static cudaError_t launch_one(const GemvParams& p, dim3 grid, int threads, size_t smem, cudaStream_t st) {
    static size_t configured[MAX_DEVICES] = {};          // per instantiation and device; grows monotonically
    cudaError_t e = ensure_dynamic_smem(gemv_kernel<MODE, M, R>, configured, smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1] = {pdl_attribute()};
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, gemv_kernel<MODE, M, R>, p);
}

template <int MODE, int M>
static cudaError_t launch_r(const GemvParams& p, int R, dim3 grid, int threads, size_t smem, cudaStream_t st) {
    if (R == 1) return launch_one<MODE, M, 1>(p, grid, threads, smem, st);
    if constexpr (MODE == KMODE_W4A4_I8) {
        if (R == 2) return launch_one<MODE, M, 2>(p, grid, threads, smem, st);
    }
    return cudaErrorInvalidValue;
}

template <int MODE>
static cudaError_t launch_m(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st) {
    switch (M) {
        case 1: return launch_r<MODE, 1>(p, R, grid, threads, smem, st);
        case 2: return launch_r<MODE, 2>(p, R, grid, threads, smem, st);
        case 3: return launch_r<MODE, 3>(p, R, grid, threads, smem, st);
        case 4: return launch_r<MODE, 4>(p, R, grid, threads, smem, st);
        case 5: return launch_r<MODE, 5>(p, R, grid, threads, smem, st);
        case 6: return launch_r<MODE, 6>(p, R, grid, threads, smem, st);
        case 7: return launch_r<MODE, 7>(p, R, grid, threads, smem, st);
        case 8: return launch_r<MODE, 8>(p, R, grid, threads, smem, st);
    }
    return cudaErrorInvalidValue;
}

}  // namespace nvfp4
