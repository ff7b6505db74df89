// noalloc.cu -- nvfp4_gemv_noalloc: the GEMV for callers that cannot allocate device memory (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc).  The GEMV's scratch (arrival counters + split
// partials, what nvfp4_gemv takes as `workspace`) lives in ONE file-scope __device__ array of
// NVFP4_NOALLOC_SCRATCH_BYTES bytes; every GPU that loads the library holds it until the process exits.
//
// In host code the array's NAME is a host-side stand-in, not a device address: its device address is looked up once
// per device with cudaGetSymbolAddress (with that device current) and that pointer is what the kernels get.  Device
// code of this file (the clearing kernel) names the array directly.
//
// Every call shares the array, and the array keeps the previous call's contents: the bytes the call is going to use
// are cleared on the caller's stream first (the GEMV needs its arrival counters zero on entry).  Calls that overlap
// on the GPU (two streams, two host threads launching onto different streams) race on the array: serialise them.
// The entry point calls no cudaMalloc / cudaFree / allocating library routine: cudaGetDevice, cudaGetSymbolAddress
// (first call per device), two kernel launches.
#include <stdio.h>

#include <mutex>

#include "nvfp4_common.cuh"
#include "nvfp4_internal.h"

namespace nvfp4 {

static __device__ __align__(256) unsigned char g_noalloc_scratch[NVFP4_NOALLOC_SCRATCH_BYTES];

// zero the first nvec 16-byte vectors of the scratch.  Launched like every kernel of the path (programmatic dependent
// launch): it waits for its stream predecessor -- which may be the previous call's GEMV, still using the scratch --
// before the first store, and the GEMV that follows touches its workspace only after its own griddepcontrol.wait,
// i.e. after this kernel has completed.
__global__ void __launch_bounds__(256) noalloc_clear_kernel(unsigned int nvec) {
    pdl_wait();
    pdl_launch_dependents();
    uint4* p = reinterpret_cast<uint4*>(g_noalloc_scratch);
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += gridDim.x * blockDim.x)
        p[i] = make_uint4(0u, 0u, 0u, 0u);
}

static std::mutex g_noalloc_mutex;
static void* g_noalloc_ptr[MAX_DEVICES] = {};

// device address of the scratch array on the CURRENT device (looked up once per device)
static cudaError_t noalloc_scratch_address(void** out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaGetSymbolAddress(out, g_noalloc_scratch);
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (g_noalloc_ptr[dev] == nullptr) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return cudaSuccess;
}

}  // namespace nvfp4

using namespace nvfp4;

extern "C" int nvfp4_gemv_noalloc(int mode, const void* w_blob, const float* w_gscale, int N, int K, const void* x,
                                  const uint8_t* x_scales, const float* x_gscale, int M, int64_t ldx, void* y, int y_dtype,
                                  int64_t ldy, void* stream) {
    const size_t need = nvfp4_gemv_workspace_bytes(M, N, K);          // 0: unsupported shape (nvfp4_gemv reports it below)
    if (need > (size_t)NVFP4_NOALLOC_SCRATCH_BYTES) {
        char msg[200];
        snprintf(msg, sizeof(msg), "nvfp4_gemv_noalloc: (M=%d, N=%d, K=%d) needs %zu bytes of scratch, the built-in array "
                 "holds %zu: use nvfp4_gemv with a caller-allocated workspace", M, N, K, need, (size_t)NVFP4_NOALLOC_SCRATCH_BYTES);
        set_last_error(msg);
        return NVFP4_ERR_UNSUPPORTED_SHAPE;
    }
    void* scratch = nullptr;
    cudaError_t e = noalloc_scratch_address(&scratch);
    if (e == cudaSuccess && need > 0) {
        const unsigned int nvec = (unsigned int)((need + 15) / 16);
        unsigned int grid = (nvec + 255) / 256;
        if (grid > 148 * 4) grid = 148 * 4;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(grid);
        cfg.blockDim = dim3(256);
        cfg.stream = static_cast<cudaStream_t>(stream);
        cudaLaunchAttribute attr = pdl_attribute();
        cfg.attrs = &attr;
        cfg.numAttrs = 1;
        e = cudaLaunchKernelEx(&cfg, noalloc_clear_kernel, nvec);
    }
    if (e != cudaSuccess) {
        char msg[200];
        snprintf(msg, sizeof(msg), "nvfp4_gemv_noalloc: %s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
        set_last_error(msg);
        (void)cudaGetLastError();
        return NVFP4_ERR_CUDA;
    }
    return nvfp4_gemv(mode, w_blob, w_gscale, N, K, x, x_scales, x_gscale, M, ldx, y, y_dtype, ldy, scratch,
                      (size_t)NVFP4_NOALLOC_SCRATCH_BYTES, stream);
}
