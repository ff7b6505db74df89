// gemv.cu -- host side of the GEMV: launch-shape table, workspace layout, template dispatch.
#include <stdlib.h>
#include "gemv_kernel.cuh"

namespace nvfp4 {

constexpr int NUM_SMS = 148;          // B200
constexpr size_t SMEM_CAP = 227 * 1024;

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// arithmetic variant: W4A4 runs the FP16 path up to M = NVFP4_MH (default 1), the integer path above
int gemv_kmode(int mode, int M) {
    if (mode == NVFP4_MODE_W4A16) return KMODE_W4A16;
    static int mh = -1;
    if (mh < 0) { const char* e = getenv("NVFP4_MH"); mh = e ? atoi(e) : 1; }
    return M <= mh ? KMODE_W4A4_H : KMODE_W4A4_I8;
}

// CTAs per K range: about one per SM over all K ranges, never more than there are units
static int gemv_ctas(int units, const GemvConfig& c) {
    int ctas = NUM_SMS / c.ksplit;
    if (ctas < 1) ctas = 1;
    return ctas > units ? units : ctas;
}

size_t gemv_smem_bytes(int mode, int M, int N, int K, const GemvConfig& c) {
    const Layout L = make_layout(N, K, layout_kparts(N, K));
    const int ncw_max = (L.ncells + c.ksplit - 1) / c.ksplit;
    const int xbp = xbp_bytes(gemv_kmode(mode, M));
    const size_t xs = align_up((size_t)ncw_max * CELL_VECS * L.kp * xvec_stride(gemv_kmode(mode, M), M), 128);
    const int units = (L.ntiles + c.rows - 1) / c.rows;
    const int ctas = gemv_ctas(units, c);
    const int ucta_max = (units + ctas - 1) / ctas;
    return xs + (size_t)c.warps * c.stages * c.rows * CELL_BYTES             // rings
         + (size_t)c.warps * 2 * c.rows * M * L.rpt * sizeof(float)          // segment slots
         + (size_t)c.warps * c.stages * 8                                    // ring mbarriers
         + ((size_t)ncw_max * L.kp * M * 4 * CELL_VECS / (mode == MODE_W4A4_FUSED_QUANT ? 160 : STAGE_ITEMS) + 2) * 8   // staging-batch mbarriers
         + (size_t)(ucta_max + c.warps + 40) * sizeof(int);                  // unit counters + share starts + fused-quant scratch
}

// Launch shape per (mode, M, N, K).  Values come from the sweeps recorded in DESIGN.md
// ("Tuning"); the rule below reproduces them and extrapolates to other shapes.
GemvConfig gemv_pick_config(int mode, int M, int N, int K) {
    GemvConfig c;
    const Layout L = make_layout(N, K, layout_kparts(N, K));
    // from the round-1 sweeps on B200 (profiles/r01_sweep.md): with 4608-byte cells two stages per warp
    // keep enough bytes in flight; one tile per warp (R = 1) and 12-16 consumer warps are best everywhere
    const bool half_path = (gemv_kmode(mode, M) == KMODE_W4A4_H);
    c.rows = 1;
    // small weights (qkv, o: <= 64 M weights) at M = 2..4: 12 warps measured 3-6 % faster than 16 (fewer, longer shares)
    const bool small_w = (M >= 2 && M <= 4 && (long long)N * K <= (64ll << 20));
    c.warps = (M >= 8 || (half_path && K < 16384) || small_w) ? 12 : 16;
    c.stages = 2;
    c.ksplit = 1;
    // one persistent CTA per SM: shrink only if it does not fit in the 227 KB of shared memory
    while (gemv_smem_bytes(mode, M, N, K, c) > SMEM_CAP) {
        const int ncw_max = (L.ncells + c.ksplit - 1) / c.ksplit;
        const size_t xs = (size_t)ncw_max * CELL_VECS * L.kp * xvec_stride(gemv_kmode(mode, M), M);
        if (xs > SMEM_CAP / 2 && c.ksplit < L.ncells) ++c.ksplit;       // activations dominate: split K
        else if (c.warps > 8) c.warps -= 2;
        else if (c.ksplit < L.ncells) ++c.ksplit;
        else if (c.warps > 1) --c.warps;
        else break;
    }
    return c;
}

static size_t counters_bytes(int N, int K) {
    return align_up((size_t)make_layout(N, K, layout_kparts(N, K)).ntiles * sizeof(unsigned int), 256);
}

size_t gemv_workspace_bytes_for(int M, int N, int K, const GemvConfig& c) {
    if (c.ksplit <= 1) return counters_bytes(N, K);
    const Layout L = make_layout(N, K, layout_kparts(N, K));
    return counters_bytes(N, K) + (size_t)c.ksplit * M * L.ntiles * L.rpt * sizeof(float);
}

cudaError_t launch_gemv_w4a4(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st);
cudaError_t launch_gemv_w4a16(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st);
cudaError_t launch_gemv_w4a4h(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st);

cudaError_t launch_gemv(int mode, const void* blob, const float* w_gscale, int N, int K, const void* x,
                        const uint8_t* x_scales, const float* x_gscale, int M, int64_t ldx, void* y, int y_dtype,
                        int64_t ldy, void* workspace, size_t ws_bytes, const GemvConfig& cfg, cudaStream_t st) {
    const bool fuse_quant = (mode == MODE_W4A4_FUSED_QUANT);
    GemvParams p;
    p.blob = static_cast<const uint8_t*>(blob);
    p.w_gscale = w_gscale;
    p.x = x; p.x_scales = x_scales; p.x_gscale = x_gscale;
    p.y = y;
    p.counters = static_cast<unsigned int*>(workspace);
    p.partials = reinterpret_cast<float*>(static_cast<uint8_t*>(workspace) + counters_bytes(N, K));
    p.ldx = ldx; p.ldy = ldy;
    p.N = N; p.K = K;
    const Layout L = make_layout(N, K, layout_kparts(N, K));
    p.ntiles = L.ntiles; p.nch = L.ncells; p.Npad = L.ntiles * L.rpt;
    p.kp = L.kp; p.kp_shift = 0;
    while ((1 << p.kp_shift) < L.kp) ++p.kp_shift;
    p.warps = cfg.warps; p.stages = cfg.stages; p.ksplit = cfg.ksplit;
    p.y_bf16 = (y_dtype == NVFP4_DTYPE_BF16);
    p.zero = 0;
    p.fuse_quant = fuse_quant ? 1 : 0;
    p.x_gscale_out = fuse_quant ? const_cast<float*>(x_gscale) : nullptr;
    if (cfg.ksplit > 1 && ws_bytes < gemv_workspace_bytes_for(M, N, K, cfg)) return cudaErrorInvalidValue;
    const size_t smem = gemv_smem_bytes(mode, M, N, K, cfg);
    if (smem > SMEM_CAP) return cudaErrorInvalidConfiguration;
    p.units = (p.ntiles + cfg.rows - 1) / cfg.rows;
    const int ctas = gemv_ctas(p.units, cfg);
    // every consumer warp needs at least one cell of the smallest CTA's flat stream
    const int min_cells = (p.units / ctas) * (p.nch / cfg.ksplit);
    if (p.warps > min_cells) p.warps = min_cells;
    const int max_warps = (gemv_max_threads(gemv_kmode(mode, M), M, cfg.rows) - STAGER_THREADS) / 32;   // launch bounds of the instantiation
    if (p.warps > max_warps) p.warps = max_warps;
    p.units_q = p.units / ctas; p.units_r = p.units % ctas;
    p.cells_q = p.nch / cfg.ksplit; p.cells_r = p.nch % cfg.ksplit;
    dim3 grid(ctas, cfg.ksplit);
    const int threads = p.warps * 32 + STAGER_THREADS;
    const int kmode = gemv_kmode(mode, M);
    if (kmode == KMODE_W4A4_I8) return launch_gemv_w4a4(p, M, cfg.rows, grid, threads, smem, st);
    if (kmode == KMODE_W4A4_H) return launch_gemv_w4a4h(p, M, cfg.rows, grid, threads, smem, st);
    return launch_gemv_w4a16(p, M, cfg.rows, grid, threads, smem, st);
}

}  // namespace nvfp4
