// nvfp4_internal.h -- host-side launch entry points behind the C ABI (api.cu calls these).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace nvfp4 {

// internal `mode` value (beyond NVFP4_MODE_W4A4 / _W4A16): W4A4 with the activation quantizer fused into
// the GEMV's stagers -- x is BF16, x_scales is NULL, x_gscale is an optional OUTPUT
constexpr int MODE_W4A4_FUSED_QUANT = 2;

// launch shape of the GEMV: every field > 0
struct GemvConfig {
    int warps;    // warps per CTA, each owns `rows` row tiles (32 rows each) -> no cross-warp reduce
    int rows;     // R: row tiles (32/KP rows each) per warp (1, 2 or 4)
    int stages;   // depth of each warp's private bulk-copy ring (cells of 4608 B per tile)
    int ksplit;   // number of K ranges (grid.y); > 1 -> partials through the workspace
};

// launch attribute that lets a kernel start before its stream predecessor has finished (PDL)
inline cudaLaunchAttribute pdl_attribute() {
    cudaLaunchAttribute a = {};
    a.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    a.val.programmaticStreamSerializationAllowed = 1;
    return a;
}

cudaError_t launch_quantize_act(const void* x_bf16, int M, int K, int64_t ldx, uint8_t* codes, uint8_t* scales,
                                float* gscale, int gscale_mode, cudaStream_t st);

cudaError_t launch_repack(const uint8_t* codes, const uint8_t* scales, int N, int K, void* blob, cudaStream_t st);
cudaError_t launch_unpack(const void* blob, int N, int K, uint8_t* codes, uint8_t* scales, cudaStream_t st);

GemvConfig gemv_pick_config(int mode, int M, int N, int K);
size_t gemv_workspace_bytes_for(int M, int N, int K, const GemvConfig& c);
size_t gemv_smem_bytes(int mode, int M, int N, int K, const GemvConfig& c);
cudaError_t launch_gemv(int mode, const void* blob, const float* w_gscale, int N, int K, const void* x,
                        const uint8_t* x_scales, const float* x_gscale, int M, int64_t ldx, void* y, int y_dtype,
                        int64_t ldy, void* workspace, size_t ws_bytes, const GemvConfig& cfg, cudaStream_t st);

cudaError_t launch_silu_mul(const void* gu, int M, int I, void* h, cudaStream_t st);

}  // namespace nvfp4
