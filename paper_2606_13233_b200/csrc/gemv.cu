// gemv.cu -- host side of the GEMV: launch-shape table, workspace layout, template dispatch.
#include "gemv_kernel.cuh"

namespace nvfp4 {

constexpr int NUM_SMS = 148;          // B200
constexpr size_t SMEM_CAP = 227 * 1024;

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

size_t gemv_smem_bytes(int mode, int M, int K, const GemvConfig& c) {
    const int nch = n_chunks(K);
    const int ncw_max = (nch + c.ksplit - 1) / c.ksplit;
    const int xbp = (mode == NVFP4_MODE_W4A4) ? XBP_W4A4 : XBP_W4A16;
    const size_t xs = align_up((size_t)ncw_max * 4 * M * xbp, 128);
    return xs + (size_t)c.warps * c.stages * c.rows * CELL_BYTES + (size_t)c.warps * c.stages * 8;
}

// Launch shape per (mode, M, N, K).  Values come from the sweeps recorded in DESIGN.md
// ("Tuning"); the rule below reproduces them and extrapolates to other shapes.
GemvConfig gemv_pick_config(int mode, int M, int N, int K) {
    GemvConfig c;
    const int ntiles = n_tiles(N), nch = n_chunks(K);
    c.rows = (M >= 3 && mode == NVFP4_MODE_W4A4) ? 2 : 1;
    c.warps = 8;
    c.stages = 4;
    if (ntiles < c.rows * c.warps * NUM_SMS / 4) c.rows = 1;
    const int cta_rows = (ntiles + c.warps * c.rows - 1) / (c.warps * c.rows);
    const int target = NUM_SMS * 2;
    int ks = (target + cta_rows / 2) / cta_rows;
    if (ks * cta_rows > target && ks > 1) --ks;
    if (ks < 1) ks = 1;
    if (ks > nch) ks = nch;
    c.ksplit = ks;
    // shrink until the CTA fits in shared memory
    while (gemv_smem_bytes(mode, M, K, c) > SMEM_CAP) {
        if (c.stages > 2) --c.stages;
        else if (c.ksplit < nch) ++c.ksplit;
        else if (c.warps > 1) c.warps /= 2;
        else break;
    }
    return c;
}

static size_t counters_bytes(int N) { return align_up((size_t)n_tiles(N) * sizeof(unsigned int), 256); }

size_t gemv_workspace_bytes_for(int M, int N, const GemvConfig& c) {
    if (c.ksplit <= 1) return counters_bytes(N);
    return counters_bytes(N) + (size_t)c.ksplit * M * n_tiles(N) * TILE_ROWS * sizeof(float);
}

cudaError_t launch_gemv_w4a4(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st);
cudaError_t launch_gemv_w4a16(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st);

cudaError_t launch_gemv(int mode, const void* blob, const float* w_gscale, int N, int K, const void* x,
                        const uint8_t* x_scales, const float* x_gscale, int M, int64_t ldx, void* y, int y_dtype,
                        int64_t ldy, void* workspace, size_t ws_bytes, const GemvConfig& cfg, cudaStream_t st) {
    GemvParams p;
    p.blob = static_cast<const uint8_t*>(blob);
    p.w_gscale = w_gscale;
    p.x = x; p.x_scales = x_scales; p.x_gscale = x_gscale;
    p.y = y;
    p.counters = static_cast<unsigned int*>(workspace);
    p.partials = reinterpret_cast<float*>(static_cast<uint8_t*>(workspace) + counters_bytes(N));
    p.ldx = ldx; p.ldy = ldy;
    p.N = N; p.K = K;
    p.ntiles = n_tiles(N); p.nch = n_chunks(K); p.Npad = p.ntiles * TILE_ROWS;
    p.warps = cfg.warps; p.stages = cfg.stages; p.ksplit = cfg.ksplit;
    p.y_bf16 = (y_dtype == NVFP4_DTYPE_BF16);
    if (cfg.ksplit > 1 && ws_bytes < gemv_workspace_bytes_for(M, N, cfg)) return cudaErrorInvalidValue;
    const size_t smem = gemv_smem_bytes(mode, M, K, cfg);
    if (smem > SMEM_CAP) return cudaErrorInvalidConfiguration;
    dim3 grid((p.ntiles + cfg.warps * cfg.rows - 1) / (cfg.warps * cfg.rows), cfg.ksplit);
    const int threads = cfg.warps * 32;
    if (mode == NVFP4_MODE_W4A4) return launch_gemv_w4a4(p, M, cfg.rows, grid, threads, smem, st);
    return launch_gemv_w4a16(p, M, cfg.rows, grid, threads, smem, st);
}

}  // namespace nvfp4
