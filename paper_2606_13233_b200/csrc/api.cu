// api.cu -- the C ABI declared in include/nvfp4.h: argument validation, error codes, launch-shape
// override, and nothing else (every step of the path runs in the kernels).  No CPU fallback.
#include <stdio.h>
#include <string.h>

#include <mutex>

#include "nvfp4_common.cuh"
#include "nvfp4_internal.h"

using namespace nvfp4;

namespace nvfp4 { extern unsigned long long* g_trace; }

static thread_local char g_last_err[256] = "";
// process-wide knobs for sweeps (nvfp4_gemv_set_config, nvfp4_set_layout_kparts); 0 = use the tuned table.
// Guarded by a mutex: a call reads one consistent snapshot.
static std::mutex g_knob_mutex;
static GemvConfig g_override = {0, 0, 0, 0, -1, 0};    // whole: -1 = table
static int g_kparts = 0;
static GemvConfig override_snapshot(int* kp_out) {
    std::lock_guard<std::mutex> lock(g_knob_mutex);
    if (kp_out) *kp_out = g_kparts;
    return g_override;
}
static int effective_kparts(int N, int K) {
    int kp = 0;
    (void)override_snapshot(&kp);
    return kp > 0 ? kp : layout_kparts(N, K);
}

namespace nvfp4 {
// lets the other translation units of the library (noalloc.cu) leave a message for nvfp4_last_cuda_error()
void set_last_error(const char* msg) { snprintf(g_last_err, sizeof(g_last_err), "%s", msg); }
}  // namespace nvfp4

static int cuda_fail(cudaError_t e) {
    snprintf(g_last_err, sizeof(g_last_err), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
    (void)cudaGetLastError();                     // clear the sticky-less error state
    return NVFP4_ERR_CUDA;
}
static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
static bool shape_ok(int M, int N, int K) {
    return M >= 1 && M <= 8 && N >= 1 && K >= 16 && (K % 16) == 0 && (int64_t)N * K < ((int64_t)1 << 40);
}
static GemvConfig effective_config(int mode, int M, int N, int K, int kp) {
    GemvConfig c = gemv_pick_config(mode, M, N, K, kp);
    const GemvConfig o = override_snapshot(nullptr);
    if (o.ksplit > 0) c.ksplit = o.ksplit;
    if (o.warps > 0) c.warps = o.warps;
    if (o.rows > 0) c.rows = o.rows;
    if (o.stages > 0) c.stages = o.stages;
    if (o.cps > 0) c.cps = o.cps;
    if (o.whole >= 0) c.whole = o.whole;
    return gemv_legalize_config(mode, M, N, K, kp, c);
}

extern "C" {

int nvfp4_version(void) { return NVFP4_ABI_VERSION; }

const char* nvfp4_last_cuda_error(void) { return g_last_err; }

int nvfp4_quantize_act(const void* x_bf16, int M, int K, int64_t ldx, uint8_t* codes, uint8_t* scales,
                       float* gscale, int gscale_mode, void* workspace, size_t ws_bytes, void* stream) {
    (void)workspace; (void)ws_bytes;
    g_last_err[0] = 0;
    if (!x_bf16 || !codes || !scales || !gscale) return NVFP4_ERR_INVALID_ARG;
    if (gscale_mode != NVFP4_GSCALE_DYNAMIC && gscale_mode != NVFP4_GSCALE_STATIC &&
        gscale_mode != NVFP4_GSCALE_DYNAMIC_PER_ROW) return NVFP4_ERR_INVALID_ARG;
    if (!shape_ok(M, 1, K) || ldx < K || (ldx % 8) != 0) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (gscale_mode == NVFP4_GSCALE_DYNAMIC_PER_ROW && (int64_t)M * K > 524288) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(x_bf16) || !aligned16(codes) || !aligned16(scales) || (reinterpret_cast<uintptr_t>(gscale) & 3u))
        return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_quantize_act(x_bf16, M, K, ldx, codes, scales, gscale, gscale_mode,
                                        static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

size_t nvfp4_repacked_bytes(int N, int K) {
    if (!shape_ok(1, N, K)) return 0;
    const Layout L = make_layout(N, K, effective_kparts(N, K));
    return (size_t)BLOB_HEADER_BYTES + (size_t)L.ntiles * L.ncells * CELL_BYTES;
}

int nvfp4_repack_weight(const uint8_t* codes, const uint8_t* scales, int N, int K, void* blob_out, void* stream) {
    g_last_err[0] = 0;
    if (!codes || !scales || !blob_out) return NVFP4_ERR_INVALID_ARG;
    if (!shape_ok(1, N, K)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(codes) || !aligned16(scales) || !aligned16(blob_out)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_repack(codes, scales, N, K, effective_kparts(N, K), blob_out, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_unpack_weight(const void* blob, int N, int K, uint8_t* codes_out, uint8_t* scales_out, void* stream) {
    g_last_err[0] = 0;
    if (!codes_out || !scales_out || !blob) return NVFP4_ERR_INVALID_ARG;
    if (!shape_ok(1, N, K)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(codes_out) || !aligned16(scales_out) || !aligned16(blob)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_unpack(blob, N, K, effective_kparts(N, K), codes_out, scales_out, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

size_t nvfp4_gemv_workspace_bytes(int M, int N, int K) {
    if (!shape_ok(M, N, K)) return 0;
    const int kp = effective_kparts(N, K);
    size_t need = 0;
    for (int mode : {NVFP4_MODE_W4A4, NVFP4_MODE_W4A16, MODE_W4A4_FUSED_QUANT}) {
        const size_t b = gemv_workspace_bytes_for(mode, M, N, K, kp, effective_config(mode, M, N, K, kp));
        need = b > need ? b : need;
    }
    return need;
}

static int gemv_common(int mode, const void* w_blob, const float* w_gscale, int N, int K, const void* x,
                       const uint8_t* x_scales, const float* x_gscale, int gscale_per_row, int M, int64_t ldx, void* y,
                       int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes, void* stream) {
    g_last_err[0] = 0;
    if (mode != NVFP4_MODE_W4A4 && mode != NVFP4_MODE_W4A16) return NVFP4_ERR_INVALID_ARG;
    if (y_dtype != NVFP4_DTYPE_F32 && y_dtype != NVFP4_DTYPE_BF16) return NVFP4_ERR_INVALID_ARG;
    if (!w_blob || !w_gscale || !x || !y) return NVFP4_ERR_INVALID_ARG;
    if (mode == NVFP4_MODE_W4A4 && (!x_scales || !x_gscale)) return NVFP4_ERR_INVALID_ARG;
    if (!shape_ok(M, N, K) || ldy < N) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (mode == NVFP4_MODE_W4A4) { if (ldx < K / 2 || (ldx % 8) != 0) return NVFP4_ERR_UNSUPPORTED_SHAPE; }
    else                         { if (ldx < K || (ldx % 8) != 0) return NVFP4_ERR_UNSUPPORTED_SHAPE; }
    if (!aligned16(w_blob) || !aligned16(x) || !aligned16(y) || (workspace && !aligned16(workspace)))
        return NVFP4_ERR_ALIGNMENT;
    const int kp = effective_kparts(N, K);
    const GemvConfig cfg = effective_config(mode, M, N, K, kp);
    const size_t need = gemv_workspace_bytes_for(mode, M, N, K, kp, cfg);
    if (!workspace || ws_bytes < need) return NVFP4_ERR_INVALID_ARG;
    cudaError_t e = launch_gemv(mode, w_blob, w_gscale, N, K, kp, x, x_scales, x_gscale, gscale_per_row, M, ldx, y, y_dtype,
                                ldy, workspace, ws_bytes, cfg, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_gemv(int mode, const void* w_blob, const float* w_gscale, int N, int K, const void* x,
               const uint8_t* x_scales, const float* x_gscale, int M, int64_t ldx, void* y, int y_dtype,
               int64_t ldy, void* workspace, size_t ws_bytes, void* stream) {
    return gemv_common(mode, w_blob, w_gscale, N, K, x, x_scales, x_gscale, 0, M, ldx, y, y_dtype, ldy, workspace,
                       ws_bytes, stream);
}

size_t nvfp4_linear_workspace_bytes(int M, int N, int K) {
    if (M < 1 || !shape_ok(1, N, K)) return 0;
    const size_t a = nvfp4_gemv_workspace_bytes(M < 8 ? M : 8, N, K);
    const size_t b = (M > 8 && (M % 8) != 0) ? nvfp4_gemv_workspace_bytes(M % 8, N, K) : 0;
    return a > b ? a : b;
}

int nvfp4_linear(int mode, const void* w_blob, const float* w_gscale, int N, int K, const void* x,
                 const uint8_t* x_scales, const float* x_gscale, int M, int64_t ldx, void* y, int y_dtype,
                 int64_t ldy, void* workspace, size_t ws_bytes, void* stream) {
    if (M < 1 || M > (1 << 20)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (y_dtype != NVFP4_DTYPE_F32 && y_dtype != NVFP4_DTYPE_BF16) return NVFP4_ERR_INVALID_ARG;
    if (mode != NVFP4_MODE_W4A4 && mode != NVFP4_MODE_W4A16) return NVFP4_ERR_INVALID_ARG;
    if (!x || !y) return NVFP4_ERR_INVALID_ARG;
    // dispatch rule (App. C.3 dispatches per (M, shape) between the CUDA-core kernel and a tensor-core GEMM):
    // this library has only the CUDA-core kernel, so any M runs as ceil(M/8) passes of it over 8-row chunks
    const size_t xrow = (mode == NVFP4_MODE_W4A4) ? (size_t)ldx : (size_t)ldx * 2;
    const size_t yrow = (size_t)ldy * (y_dtype == NVFP4_DTYPE_F32 ? 4 : 2);
    for (int r = 0; r < M; r += 8) {
        const int m = (M - r) < 8 ? (M - r) : 8;
        const int rc = gemv_common(mode, w_blob, w_gscale, N, K, static_cast<const uint8_t*>(x) + (size_t)r * xrow,
                                   x_scales ? x_scales + (size_t)r * (K / 16) : nullptr, x_gscale, 0, m, ldx,
                                   static_cast<uint8_t*>(y) + (size_t)r * yrow, y_dtype, ldy, workspace, ws_bytes, stream);
        if (rc != NVFP4_OK) return rc;
    }
    return NVFP4_OK;
}

int nvfp4_gemv_rowscale(const void* w_blob, const float* w_gscale, int N, int K, const void* x_codes,
                        const uint8_t* x_scales, const float* x_gscales, int M, int64_t ldx, void* y, int y_dtype,
                        int64_t ldy, void* workspace, size_t ws_bytes, void* stream) {
    return gemv_common(NVFP4_MODE_W4A4, w_blob, w_gscale, N, K, x_codes, x_scales, x_gscales, 1, M, ldx, y, y_dtype, ldy,
                       workspace, ws_bytes, stream);
}

int nvfp4_gemv_fused_quant(const void* w_blob, const float* w_gscale, int N, int K, const void* x_bf16, int M,
                           int64_t ldx, float* x_gscale_out, void* y, int y_dtype, int64_t ldy,
                           void* workspace, size_t ws_bytes, void* stream) {
    g_last_err[0] = 0;
    if (y_dtype != NVFP4_DTYPE_F32 && y_dtype != NVFP4_DTYPE_BF16) return NVFP4_ERR_INVALID_ARG;
    if (!w_blob || !w_gscale || !x_bf16 || !y) return NVFP4_ERR_INVALID_ARG;
    if (!shape_ok(M, N, K) || ldy < N || ldx < K || (ldx % 8) != 0) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(w_blob) || !aligned16(x_bf16) || !aligned16(y) || (workspace && !aligned16(workspace)))
        return NVFP4_ERR_ALIGNMENT;
    const int kp = effective_kparts(N, K);
    const GemvConfig cfg = effective_config(MODE_W4A4_FUSED_QUANT, M, N, K, kp);
    const size_t need = gemv_workspace_bytes_for(MODE_W4A4_FUSED_QUANT, M, N, K, kp, cfg);
    if (!workspace || ws_bytes < need) return NVFP4_ERR_INVALID_ARG;
    cudaError_t e = launch_gemv(MODE_W4A4_FUSED_QUANT, w_blob, w_gscale, N, K, kp, x_bf16, nullptr, x_gscale_out, 0, M, ldx,
                                y, y_dtype, ldy, workspace, ws_bytes, cfg, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_gemv_set_config(int ksplit, int warps, int rows, int stages, int ctas_per_sm, int balance) {
    if (ksplit < 0 || ksplit > 64 || warps < 0 || warps > 20 || stages < 0 || stages > 16) return NVFP4_ERR_INVALID_ARG;
    if (ctas_per_sm < 0 || ctas_per_sm > 3 || balance < 0 || balance > 2) return NVFP4_ERR_INVALID_ARG;
    if (!(rows == 0 || rows == 1 || rows == 2)) return NVFP4_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_knob_mutex);
    g_override.ksplit = ksplit; g_override.warps = warps; g_override.rows = rows; g_override.stages = stages;
    g_override.cps = ctas_per_sm;
    g_override.whole = balance - 1;                 // 0 = table, 1 = data-parallel + stream-K, 2 = whole units only
    return NVFP4_OK;
}

int nvfp4_set_layout_kparts(int kparts) {
    if (kparts < 0 || kparts > 32 || (kparts & (kparts - 1)) != 0) return NVFP4_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_knob_mutex);
    g_kparts = kparts;
    return NVFP4_OK;
}

int nvfp4_get_layout_kparts(int N, int K) {
    if (!shape_ok(1, N, K)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    return effective_kparts(N, K);
}

int nvfp4_gemv_get_config(int mode, int M, int N, int K, int* ksplit, int* warps, int* rows, int* stages, int* ctas_per_sm, int* balance) {
    if (mode != NVFP4_MODE_W4A4 && mode != NVFP4_MODE_W4A16) return NVFP4_ERR_INVALID_ARG;
    if (!shape_ok(M, N, K)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    const GemvConfig c = effective_config(mode, M, N, K, effective_kparts(N, K));
    if (ksplit) *ksplit = c.ksplit;
    if (warps) *warps = c.warps;
    if (rows) *rows = c.rows;
    if (stages) *stages = c.stages;
    if (ctas_per_sm) *ctas_per_sm = c.cps;
    if (balance) *balance = c.whole + 1;
    return NVFP4_OK;
}

size_t reset_sampler_state_bytes(void) { return RESET_STATE_BYTES; }

int reset_sampler_step(const void* logits, int logits_dtype, int B, int V, int64_t ld, void* state, float tau0, float t_low,
                       float t_high, float top_p, int w, int delimiter_token, unsigned long long seed, int* token_out,
                       float* diag_out, void* stream) {
    g_last_err[0] = 0;
    if (!logits || !state || !token_out) return NVFP4_ERR_INVALID_ARG;
    if (logits_dtype != NVFP4_DTYPE_F32 && logits_dtype != NVFP4_DTYPE_BF16) return NVFP4_ERR_INVALID_ARG;
    if (!(t_low > 0.0f) || !(t_high > 0.0f) || !(top_p > 0.0f) || top_p > 1.0f || w < 1 || w > 32) return NVFP4_ERR_INVALID_ARG;
    if (B < 1 || B > 1024 || V < 1 || V > 163840 || ld < V) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if ((reinterpret_cast<uintptr_t>(state) & 7u) || (reinterpret_cast<uintptr_t>(logits) & 3u)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_reset_sampler(logits, logits_dtype == NVFP4_DTYPE_BF16, B, V, ld, state, tau0, t_low, t_high, top_p,
                                         w, delimiter_token, seed, token_out, diag_out, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

/* debug hook (not declared in include/nvfp4.h): device buffer of 16 x u64 per CTA that the GEMV fills with
 * %globaltimer stamps of its phases; NULL switches tracing off. */
int nvfp4_debug_set_trace(void* device_buffer) {
    g_trace = static_cast<unsigned long long*>(device_buffer);
    return NVFP4_OK;
}

int nvfp4_silu_mul_quantize(const void* gu_bf16, int M, int I, uint8_t* codes, uint8_t* scales, float* gscale,
                            int gscale_mode, void* h_bf16_opt, void* stream) {
    g_last_err[0] = 0;
    if (!gu_bf16 || !codes || !scales || !gscale) return NVFP4_ERR_INVALID_ARG;
    if (gscale_mode != NVFP4_GSCALE_DYNAMIC && gscale_mode != NVFP4_GSCALE_STATIC &&
        gscale_mode != NVFP4_GSCALE_DYNAMIC_PER_ROW) return NVFP4_ERR_INVALID_ARG;
    if (!shape_ok(M, 1, I) || (gscale_mode != NVFP4_GSCALE_STATIC && (int64_t)M * I > 524288)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(gu_bf16) || !aligned16(codes) || !aligned16(scales) || (h_bf16_opt && !aligned16(h_bf16_opt)) ||
        (reinterpret_cast<uintptr_t>(gscale) & 3u)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_silu_mul_quantize(gu_bf16, M, I, codes, scales, gscale, gscale_mode, h_bf16_opt,
                                             static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_silu_mul(const void* gu_bf16, int M, int I, void* h_bf16, void* stream) {
    g_last_err[0] = 0;
    if (!gu_bf16 || !h_bf16) return NVFP4_ERR_INVALID_ARG;
    if (M < 1 || I < 8 || (I % 8) != 0) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(gu_bf16) || !aligned16(h_bf16)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_silu_mul(gu_bf16, M, I, h_bf16, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

// ---- tensor-core GEMM (gemm_tc.cu) ----
size_t nvfp4_gemm_repacked_bytes(int N, int K) {
    if (N < 1 || K < 1 || !gemm_tc_supported(N, K)) return 0;
    return gemm_tc_repacked_bytes(N, K);
}

int nvfp4_gemm_repack_weight(const uint8_t* codes, const uint8_t* scales, int N, int K, void* blob_out, void* stream) {
    g_last_err[0] = 0;
    if (!codes || !scales || !blob_out) return NVFP4_ERR_INVALID_ARG;
    if (N < 1 || K < 1 || !gemm_tc_supported(N, K)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(codes) || !aligned16(scales) || !aligned16(blob_out)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_repack_tc(codes, scales, N, K, blob_out, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_gemm_unpack_weight(const void* blob, int N, int K, uint8_t* codes_out, uint8_t* scales_out, void* stream) {
    g_last_err[0] = 0;
    if (!codes_out || !scales_out || !blob) return NVFP4_ERR_INVALID_ARG;
    if (N < 1 || K < 1 || !gemm_tc_supported(N, K)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(codes_out) || !aligned16(scales_out) || !aligned16(blob)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_unpack_tc(blob, N, K, codes_out, scales_out, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

size_t nvfp4_gemm_workspace_bytes(int M, int N, int K) {
    if (M < 1 || M > (1 << 20) || N < 1 || K < 1 || !gemm_tc_supported(N, K)) return 0;
    return gemm_tc_workspace_bytes(M, N, K);
}

int nvfp4_gemm(const void* w_blob_tc, const float* w_gscale, int N, int K, const void* x_codes, const uint8_t* x_scales,
               const float* x_gscale, int gscale_per_row, int M, int64_t ldx, void* y, int y_dtype, int64_t ldy,
               void* workspace, size_t ws_bytes, void* stream) {
    g_last_err[0] = 0;
    if (y_dtype != NVFP4_DTYPE_F32 && y_dtype != NVFP4_DTYPE_BF16) return NVFP4_ERR_INVALID_ARG;
    if (gscale_per_row != 0 && gscale_per_row != 1) return NVFP4_ERR_INVALID_ARG;
    if (!w_blob_tc || !w_gscale || !x_codes || !x_scales || !x_gscale || !y || !workspace) return NVFP4_ERR_INVALID_ARG;
    if (M < 1 || M > (1 << 20) || N < 1 || K < 1 || !gemm_tc_supported(N, K)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (ldy < N || ldx < K / 2 || (ldx % 16) != 0) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(w_blob_tc) || !aligned16(x_codes) || !aligned16(x_scales) || !aligned16(y) || !aligned16(workspace) ||
        (reinterpret_cast<uintptr_t>(w_gscale) & 3u) || (reinterpret_cast<uintptr_t>(x_gscale) & 3u))
        return NVFP4_ERR_ALIGNMENT;
    if (ws_bytes < gemm_tc_workspace_bytes(M, N, K)) return NVFP4_ERR_INVALID_ARG;
    cudaError_t e = launch_gemm_tc(w_blob_tc, w_gscale, N, K, static_cast<const uint8_t*>(x_codes), ldx, x_scales, x_gscale,
                                   gscale_per_row, M, y, y_dtype, ldy, workspace, ws_bytes, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_gemm_set_config(int stages, int ctas) {
    if (stages < 0 || stages > 16 || ctas < 0 || ctas > 1024) return NVFP4_ERR_INVALID_ARG;
    gemm_tc_set_config(stages, ctas);
    return NVFP4_OK;
}

size_t nvfp4_gemm_packed_act_bytes(int M, int K) {
    if (M < 1 || M > 128 || K < 1 || !gemm_tc_supported(1, K)) return 0;
    return gemm_tc_packed_act_bytes(M, K);
}

int nvfp4_gemm_pack_act(const void* x_codes, const uint8_t* x_scales, int M, int K, int64_t ldx, void* xpack_out, void* stream) {
    g_last_err[0] = 0;
    if (!x_codes || !x_scales || !xpack_out) return NVFP4_ERR_INVALID_ARG;
    if (M < 1 || M > 128 || K < 1 || !gemm_tc_supported(1, K) || ldx < K / 2 || (ldx % 16) != 0) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(x_codes) || !aligned16(x_scales) || !aligned16(xpack_out)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_pack_x(static_cast<const uint8_t*>(x_codes), ldx, x_scales, M, K, xpack_out, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_quantize_act_packed(const void* x_bf16, int M, int K, int64_t ldx, void* xpack_out, float* gscale, int gscale_mode,
                              void* stream) {
    g_last_err[0] = 0;
    if (!x_bf16 || !xpack_out || !gscale) return NVFP4_ERR_INVALID_ARG;
    if (gscale_mode != NVFP4_GSCALE_DYNAMIC && gscale_mode != NVFP4_GSCALE_STATIC &&
        gscale_mode != NVFP4_GSCALE_DYNAMIC_PER_ROW) return NVFP4_ERR_INVALID_ARG;
    if (M < 1 || M > 128 || K < 1 || !gemm_tc_supported(1, K) || ldx < K || (ldx % 8) != 0) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (gscale_mode == NVFP4_GSCALE_DYNAMIC_PER_ROW && (M > 8 || (int64_t)M * K > 524288)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(x_bf16) || !aligned16(xpack_out) || (reinterpret_cast<uintptr_t>(gscale) & 3u)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_quantize_act(x_bf16, M, K, ldx, static_cast<uint8_t*>(xpack_out), nullptr, gscale, gscale_mode,
                                        static_cast<cudaStream_t>(stream), gemm_tc_act_mt(M));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

/* ---- activation records of the CUDA-core GEMV (M = 1): quantizer -> GEMV without the GEMV's load / decode / store stage ---- */
size_t nvfp4_gemv_xrecord_bytes(int N, int K) {
    if (!shape_ok(1, N, K)) return 0;
    const Layout L = make_layout(N, K, effective_kparts(N, K));
    return (size_t)L.ncells * CELL_VECS * L.kp * GEMV_XRECORD_BYTES;          // one record per 32 k of the padded K
}

int nvfp4_quantize_act_records(const void* x_bf16, int M, int K, int64_t ldx, void* xrec_out, float* gscale, int gscale_mode,
                               void* stream) {
    g_last_err[0] = 0;
    if (!x_bf16 || !xrec_out || !gscale) return NVFP4_ERR_INVALID_ARG;
    if (gscale_mode != NVFP4_GSCALE_DYNAMIC && gscale_mode != NVFP4_GSCALE_STATIC) return NVFP4_ERR_INVALID_ARG;
    if (M != 1 || !shape_ok(M, 1, K) || ldx < K || (ldx % 8) != 0) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(x_bf16) || !aligned16(xrec_out) || (reinterpret_cast<uintptr_t>(gscale) & 3u)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_quantize_act(x_bf16, M, K, ldx, static_cast<uint8_t*>(xrec_out), nullptr, gscale, gscale_mode,
                                        static_cast<cudaStream_t>(stream), -1);
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_silu_mul_quantize_records(const void* gu_bf16, int M, int I, void* xrec_out, float* gscale, int gscale_mode,
                                    void* h_bf16_opt, void* stream) {
    g_last_err[0] = 0;
    if (!gu_bf16 || !xrec_out || !gscale) return NVFP4_ERR_INVALID_ARG;
    if (gscale_mode != NVFP4_GSCALE_DYNAMIC && gscale_mode != NVFP4_GSCALE_STATIC) return NVFP4_ERR_INVALID_ARG;
    if (M != 1 || !shape_ok(M, 1, I)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (gscale_mode != NVFP4_GSCALE_STATIC && (int64_t)M * I > 524288) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(gu_bf16) || !aligned16(xrec_out) || (h_bf16_opt && !aligned16(h_bf16_opt)) ||
        (reinterpret_cast<uintptr_t>(gscale) & 3u)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_silu_mul_quantize(gu_bf16, M, I, static_cast<uint8_t*>(xrec_out), nullptr, gscale, gscale_mode,
                                             h_bf16_opt, static_cast<cudaStream_t>(stream), -1);
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_gemv_records(const void* w_blob, const float* w_gscale, int N, int K, const void* xrec, const float* x_gscale, int M,
                       void* y, int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes, void* stream) {
    g_last_err[0] = 0;
    if (y_dtype != NVFP4_DTYPE_F32 && y_dtype != NVFP4_DTYPE_BF16) return NVFP4_ERR_INVALID_ARG;
    if (!w_blob || !w_gscale || !xrec || !x_gscale || !y) return NVFP4_ERR_INVALID_ARG;
    if (M != 1 || !shape_ok(M, N, K) || ldy < N) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(w_blob) || !aligned16(xrec) || !aligned16(y) || (workspace && !aligned16(workspace))) return NVFP4_ERR_ALIGNMENT;
    const int kp = effective_kparts(N, K);
    const GemvConfig cfg = effective_config(NVFP4_MODE_W4A4, M, N, K, kp);
    const size_t need = gemv_workspace_bytes_for(NVFP4_MODE_W4A4, M, N, K, kp, cfg);
    if (!workspace || ws_bytes < need) return NVFP4_ERR_INVALID_ARG;
    cudaError_t e = launch_gemv(NVFP4_MODE_W4A4, w_blob, w_gscale, N, K, kp, xrec, nullptr, x_gscale, 0, M, 0, y, y_dtype, ldy,
                                workspace, ws_bytes, cfg, static_cast<cudaStream_t>(stream), xrec);
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_silu_mul_quantize_packed(const void* gu_bf16, int M, int I, void* xpack_out, float* gscale, int gscale_mode,
                                   void* h_bf16_opt, void* stream) {
    g_last_err[0] = 0;
    if (!gu_bf16 || !xpack_out || !gscale) return NVFP4_ERR_INVALID_ARG;
    if (gscale_mode != NVFP4_GSCALE_DYNAMIC && gscale_mode != NVFP4_GSCALE_STATIC &&
        gscale_mode != NVFP4_GSCALE_DYNAMIC_PER_ROW) return NVFP4_ERR_INVALID_ARG;
    if (M < 1 || M > 128 || I < 1 || !gemm_tc_supported(1, I)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (gscale_mode != NVFP4_GSCALE_STATIC && (int64_t)M * I > 524288) return NVFP4_ERR_UNSUPPORTED_SHAPE;   // one cluster (amax on chip)
    if (gscale_mode == NVFP4_GSCALE_DYNAMIC_PER_ROW && M > 8) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(gu_bf16) || !aligned16(xpack_out) || (h_bf16_opt && !aligned16(h_bf16_opt)) ||
        (reinterpret_cast<uintptr_t>(gscale) & 3u)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_silu_mul_quantize(gu_bf16, M, I, static_cast<uint8_t*>(xpack_out), nullptr, gscale, gscale_mode,
                                             h_bf16_opt, static_cast<cudaStream_t>(stream), gemm_tc_act_mt(M));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

size_t nvfp4_gemm_packed_workspace_bytes(int M, int N, int K) {
    if (M < 1 || M > 128 || N < 1 || K < 1 || !gemm_tc_supported(N, K)) return 0;
    return gemm_tc_packed_workspace_bytes(M, N, K);
}

int nvfp4_gemm_packed(const void* w_blob_tc, const float* w_gscale, int N, int K, const void* xpack, const float* x_gscale,
                      int gscale_per_row, int M, void* y, int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes,
                      void* stream) {
    g_last_err[0] = 0;
    if (y_dtype != NVFP4_DTYPE_F32 && y_dtype != NVFP4_DTYPE_BF16) return NVFP4_ERR_INVALID_ARG;
    if (gscale_per_row != 0 && gscale_per_row != 1) return NVFP4_ERR_INVALID_ARG;
    if (!w_blob_tc || !w_gscale || !xpack || !x_gscale || !y || !workspace) return NVFP4_ERR_INVALID_ARG;
    if (M < 1 || M > 128 || N < 1 || K < 1 || !gemm_tc_supported(N, K) || ldy < N) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(w_blob_tc) || !aligned16(xpack) || !aligned16(y) || !aligned16(workspace) ||
        (reinterpret_cast<uintptr_t>(w_gscale) & 3u) || (reinterpret_cast<uintptr_t>(x_gscale) & 3u))
        return NVFP4_ERR_ALIGNMENT;
    if (ws_bytes < gemm_tc_packed_workspace_bytes(M, N, K)) return NVFP4_ERR_INVALID_ARG;
    cudaError_t e = launch_gemm_tc_packed(w_blob_tc, w_gscale, N, K, xpack, x_gscale, gscale_per_row, M, y, y_dtype, ldy,
                                          workspace, ws_bytes, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_gemm_packed_quant_out(const void* w_blob_tc, const float* w_gscale, int N, int K, const void* xpack,
                                const float* x_gscale, int gscale_per_row, int M, void* y_opt, int y_dtype, int64_t ldy,
                                void* xpack_out, const float* out_gscale, int n_quant, void* workspace, size_t ws_bytes,
                                void* stream) {
    g_last_err[0] = 0;
    if (y_dtype != NVFP4_DTYPE_F32 && y_dtype != NVFP4_DTYPE_BF16) return NVFP4_ERR_INVALID_ARG;
    if (gscale_per_row != 0 && gscale_per_row != 1) return NVFP4_ERR_INVALID_ARG;
    if (!w_blob_tc || !w_gscale || !xpack || !x_gscale || !xpack_out || !out_gscale || !workspace) return NVFP4_ERR_INVALID_ARG;
    if (M < 1 || M > 128 || N < 1 || K < 1 || !gemm_tc_supported(N, K) || (y_opt && ldy < N)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (n_quant < 256 || n_quant > N || (n_quant % 256) != 0) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(w_blob_tc) || !aligned16(xpack) || (y_opt && !aligned16(y_opt)) || !aligned16(xpack_out) || !aligned16(workspace) ||
        (reinterpret_cast<uintptr_t>(w_gscale) & 3u) || (reinterpret_cast<uintptr_t>(x_gscale) & 3u) ||
        (reinterpret_cast<uintptr_t>(out_gscale) & 3u)) return NVFP4_ERR_ALIGNMENT;
    if (ws_bytes < gemm_tc_packed_workspace_bytes(M, N, K)) return NVFP4_ERR_INVALID_ARG;
    cudaError_t e = launch_gemm_tc_packed(w_blob_tc, w_gscale, N, K, xpack, x_gscale, gscale_per_row, M, y_opt, y_dtype, ldy,
                                          workspace, ws_bytes, static_cast<cudaStream_t>(stream), xpack_out, out_gscale, n_quant);
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

size_t nvfp4_gemm_w4a16_workspace_bytes(int M, int N, int K) {
    if (M < 1 || M > (1 << 20) || N < 1 || K < 1 || !gemm_tc_supported(N, K)) return 0;
    return gemm_tc16_workspace_bytes(M, N, K);
}

int nvfp4_gemm_w4a16(const void* w_blob_tc, const float* w_gscale, int N, int K, const void* x_bf16, int M, int64_t ldx,
                     void* y, int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes, void* stream) {
    g_last_err[0] = 0;
    if (y_dtype != NVFP4_DTYPE_F32 && y_dtype != NVFP4_DTYPE_BF16) return NVFP4_ERR_INVALID_ARG;
    if (!w_blob_tc || !w_gscale || !x_bf16 || !y || !workspace) return NVFP4_ERR_INVALID_ARG;
    if (M < 1 || M > (1 << 20) || N < 1 || K < 1 || !gemm_tc_supported(N, K)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (ldy < N || ldx < K || (ldx % 8) != 0) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(w_blob_tc) || !aligned16(x_bf16) || !aligned16(y) || !aligned16(workspace) ||
        (reinterpret_cast<uintptr_t>(w_gscale) & 3u)) return NVFP4_ERR_ALIGNMENT;
    if (ws_bytes < gemm_tc16_workspace_bytes(M, N, K)) return NVFP4_ERR_INVALID_ARG;
    cudaError_t e = launch_gemm_tc16(w_blob_tc, w_gscale, N, K, x_bf16, ldx, M, y, y_dtype, ldy, workspace, ws_bytes,
                                     static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

// ---- fused gate_up: interleaved blob + SiLU * mul + static-scale quantizer in the GEMM epilogue ----
static bool gate_up_shape_ok(int N, int K) { return N >= 128 && (N % 128) == 0 && gemm_tc_supported(N, K); }

int nvfp4_gemm_repack_weight_gate_up(const uint8_t* codes, const uint8_t* scales, int N, int K, void* blob_out, void* stream) {
    g_last_err[0] = 0;
    if (!codes || !scales || !blob_out) return NVFP4_ERR_INVALID_ARG;
    if (N < 1 || K < 1 || !gate_up_shape_ok(N, K)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(codes) || !aligned16(scales) || !aligned16(blob_out)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_repack_tc(codes, scales, N, K, blob_out, static_cast<cudaStream_t>(stream), 1);
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_gemm_unpack_weight_gate_up(const void* blob, int N, int K, uint8_t* codes_out, uint8_t* scales_out, void* stream) {
    g_last_err[0] = 0;
    if (!codes_out || !scales_out || !blob) return NVFP4_ERR_INVALID_ARG;
    if (N < 1 || K < 1 || !gate_up_shape_ok(N, K)) return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(codes_out) || !aligned16(scales_out) || !aligned16(blob)) return NVFP4_ERR_ALIGNMENT;
    cudaError_t e = launch_unpack_tc(blob, N, K, codes_out, scales_out, static_cast<cudaStream_t>(stream), 1);
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

int nvfp4_gemm_packed_silu_quant_out(const void* w_blob_gate_up, const float* w_gscale, int N, int K, const void* xpack,
                                     const float* x_gscale, int gscale_per_row, int M, void* h_opt, int h_dtype, int64_t ldh,
                                     void* xpack_out, const float* out_gscale, void* workspace, size_t ws_bytes, void* stream) {
    g_last_err[0] = 0;
    if (h_dtype != NVFP4_DTYPE_F32 && h_dtype != NVFP4_DTYPE_BF16) return NVFP4_ERR_INVALID_ARG;
    if (gscale_per_row != 0 && gscale_per_row != 1) return NVFP4_ERR_INVALID_ARG;
    if (!w_blob_gate_up || !w_gscale || !xpack || !x_gscale || !xpack_out || !out_gscale || !workspace) return NVFP4_ERR_INVALID_ARG;
    if (M < 1 || M > 128 || N < 1 || K < 1 || !gate_up_shape_ok(N, K) || ((N / 2) % 256) != 0 || (h_opt && ldh < N / 2))
        return NVFP4_ERR_UNSUPPORTED_SHAPE;
    if (!aligned16(w_blob_gate_up) || !aligned16(xpack) || (h_opt && !aligned16(h_opt)) || !aligned16(xpack_out) || !aligned16(workspace) ||
        (reinterpret_cast<uintptr_t>(w_gscale) & 3u) || (reinterpret_cast<uintptr_t>(x_gscale) & 3u) ||
        (reinterpret_cast<uintptr_t>(out_gscale) & 3u)) return NVFP4_ERR_ALIGNMENT;
    if (ws_bytes < gemm_tc_packed_workspace_bytes(M, N, K)) return NVFP4_ERR_INVALID_ARG;
    cudaError_t e = launch_gemm_tc_packed(w_blob_gate_up, w_gscale, N, K, xpack, x_gscale, gscale_per_row, M, h_opt, h_dtype, ldh,
                                          workspace, ws_bytes, static_cast<cudaStream_t>(stream), xpack_out, out_gscale, N / 2, 1);
    return e == cudaSuccess ? NVFP4_OK : cuda_fail(e);
}

}  // extern "C"
