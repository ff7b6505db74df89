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
    int warps;    // consumer warps per CTA; each streams an equal share of the CTA's cells
    int rows;     // R: row tiles (32/KP rows each) per warp step (1 or 2): x records are loaded once per R tiles
    int stages;   // depth of each warp's private bulk-copy ring (R cells of 4608 B per stage)
    int ksplit;   // number of K slices (grid.y); each slice's activations are staged by its own CTAs
    int whole;    // 1: whole units only (CTAs get base or base + 1 units, no leftover stream); 0: data-parallel + stream-K
    int cps;      // CTAs per SM (1..3): with >= 2 the next kernel's CTAs become resident (and prefetch their first
                  // weight cells) while this kernel's are still running -- programmatic dependent launch
};

// launch attribute that lets a kernel start before its stream predecessor has finished (PDL)
inline cudaLaunchAttribute pdl_attribute() {
    cudaLaunchAttribute a = {};
    a.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    a.val.programmaticStreamSerializationAllowed = 1;
    return a;
}

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per device: remember the largest value set per
// (kernel, device) so that a process driving several GPUs opts every one of them in.
constexpr int MAX_DEVICES = 64;
template <typename Kernel>
inline cudaError_t ensure_dynamic_smem(Kernel kernel, size_t* configured /*[MAX_DEVICES]*/, size_t smem) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (smem > __atomic_load_n(&configured[dev], __ATOMIC_RELAXED)) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        __atomic_store_n(&configured[dev], smem, __ATOMIC_RELAXED);     // racing threads at worst set it twice
    }
    return cudaSuccess;
}

cudaError_t launch_quantize_act(const void* x_bf16, int M, int K, int64_t ldx, uint8_t* codes, uint8_t* scales,
                                float* gscale, int gscale_mode, cudaStream_t st, int pack_mt = 0);
cudaError_t launch_silu_mul_quantize(const void* gu_bf16, int M, int I, uint8_t* codes, uint8_t* scales, float* gscale,
                                     int gscale_mode, void* h_bf16_opt, cudaStream_t st, int pack_mt = 0);

cudaError_t launch_repack(const uint8_t* codes, const uint8_t* scales, int N, int K, int kp, void* blob, cudaStream_t st);
cudaError_t launch_unpack(const void* blob, int N, int K, int kp, uint8_t* codes, uint8_t* scales, cudaStream_t st);

GemvConfig gemv_pick_config(int mode, int M, int N, int K, int kp);
GemvConfig gemv_legalize_config(int mode, int M, int N, int K, int kp, GemvConfig c);
size_t gemv_workspace_bytes_for(int mode, int M, int N, int K, int kp, const GemvConfig& c);
size_t gemv_smem_bytes(int mode, int M, int N, int K, int kp, const GemvConfig& c);
cudaError_t launch_gemv(int mode, const void* blob, const float* w_gscale, int N, int K, int kp, const void* x,
                        const uint8_t* x_scales, const float* x_gscale, int gscale_per_row, int M, int64_t ldx, void* y,
                        int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes, const GemvConfig& cfg, cudaStream_t st,
                        const void* x_records = nullptr);
// activation records of the M = 1 FP16 path (gemv_kernel.cuh XBP_W4A4H): 80 bytes per 32 k = 32 f16 | 2 x FP32 scale | pad
constexpr int GEMV_XRECORD_BYTES = 80;

cudaError_t launch_silu_mul(const void* gu, int M, int I, void* h, cudaStream_t st);

constexpr int RESET_STATE_BYTES = 160;
cudaError_t launch_reset_sampler(const void* logits, int logits_bf16, int B, int V, int64_t ld, void* state, float tau0,
                                 float t_low, float t_high, float top_p, int w, int delimiter, unsigned long long seed,
                                 int* token_out, float* diag_out, cudaStream_t st);

void set_last_error(const char* msg);          // api.cu: text returned by nvfp4_last_cuda_error() (thread-local)

// tensor-core GEMM (gemm_tc.cu)
void gemm_tc_set_config(int stages, int ctas);
bool gemm_tc_supported(int N, int K);
size_t gemm_tc_repacked_bytes(int N, int K);
size_t gemm_tc_workspace_bytes(int M, int N, int K);
int gemm_tc_act_mt(int M);
size_t gemm_tc_packed_act_bytes(int M, int K);
size_t gemm_tc_packed_workspace_bytes(int M, int N, int K);
cudaError_t launch_pack_x(const uint8_t* x_codes, int64_t ldx, const uint8_t* x_scales, int M, int K, void* xpack,
                          cudaStream_t st);
cudaError_t launch_gemm_tc_packed(const void* blob, const float* w_gscale, int N, int K, const void* xpack,
                                  const float* x_gscale, int gscale_per_row, int M, void* y, int y_dtype, int64_t ldy,
                                  void* workspace, size_t ws_bytes, cudaStream_t st, void* qout = nullptr,
                                  const float* qout_gscale = nullptr, int n_quant = 0, int silu = 0);
cudaError_t launch_repack_tc(const uint8_t* codes, const uint8_t* scales, int N, int K, void* blob, cudaStream_t st, int inter = 0);
cudaError_t launch_unpack_tc(const void* blob, int N, int K, uint8_t* codes, uint8_t* scales, cudaStream_t st, int inter = 0);
cudaError_t launch_gemm_tc(const void* blob, const float* w_gscale, int N, int K, const uint8_t* x_codes, int64_t ldx,
                           const uint8_t* x_scales, const float* x_gscale, int gscale_per_row, int M, void* y, int y_dtype,
                           int64_t ldy, void* workspace, size_t ws_bytes, cudaStream_t st);

// tensor-core W4A16 GEMM (gemm_tc16.cu): NVFP4 weights in the tensor-core blob, BF16 activations
size_t gemm_tc16_workspace_bytes(int M, int N, int K);
cudaError_t launch_gemm_tc16(const void* blob, const float* w_gscale, int N, int K, const void* x_bf16, int64_t ldx, int M,
                             void* y, int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes, cudaStream_t st);

}  // namespace nvfp4
