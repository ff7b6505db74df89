// gemv.cu -- host side of the GEMV: launch-shape table, stream-K plan, workspace layout, template dispatch.
#include "gemv_kernel.cuh"

namespace nvfp4 {

constexpr int NUM_SMS = 148;          // B200
constexpr size_t SMEM_CAP = 227 * 1024;

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// arithmetic variant: W4A4 runs the FP16 path (F2FP + HFMA2) at M = 1, the integer path (PRMT + dp4a) above
int gemv_kmode(int mode, int M) {
    if (mode == NVFP4_MODE_W4A16) return KMODE_W4A16;
    return M <= 1 ? KMODE_W4A4_H : KMODE_W4A4_I8;
}

// everything the launch derives from (mode, M, N, K, kp, config): one place for smem, workspace and kernel params
struct GemvPlan {
    int kmode, M, R, W, S, ksplit, nb;
    Layout L;
    int units, cells_q, cells_r, ncw_max;
    int share_q[2], share_r[2];
    float inv_share[2];
    int jmax, ucta_max, nxb, threads, Npad;
    SmemMap map;
};

static GemvPlan gemv_plan(int mode, int M, int N, int K, int kp, const GemvConfig& c) {
    GemvPlan P;
    P.kmode = gemv_kmode(mode, M);
    P.M = M; P.R = c.rows; P.S = c.stages;
    P.L = make_layout(N, K, kp);
    P.ksplit = c.ksplit < 1 ? 1 : (c.ksplit > P.L.ncells ? P.L.ncells : c.ksplit);
    P.units = (P.L.ntiles + P.R - 1) / P.R;
    P.Npad = P.units * P.R * P.L.rpt;
    P.cells_q = P.L.ncells / P.ksplit; P.cells_r = P.L.ncells % P.ksplit;
    P.ncw_max = P.cells_q + (P.cells_r > 0 ? 1 : 0);
    // CTAs per K slice: about one per SM over all slices, never more than the smallest slice has cells
    const long long t_min = (long long)P.units * P.cells_q;
    int nb = NUM_SMS / P.ksplit;
    if (nb < 1) nb = 1;
    if (nb > t_min) nb = (int)t_min;
    P.nb = nb;
    // every consumer warp needs at least one cell of the smallest CTA share
    const int max_warps = (gemv_max_threads(P.kmode, M, P.R) - STAGER_THREADS) / 32;   // launch bounds of the instantiation
    int W = c.warps < 1 ? 1 : c.warps;
    if (W > t_min / nb) W = (int)(t_min / nb);
    if (W > max_warps) W = max_warps;
    P.W = W;
    P.threads = W * 32 + STAGER_THREADS;
    P.jmax = 1; P.ucta_max = 1;
    for (int v = 0; v < 2; ++v) {
        const long long ncw = P.cells_q + v;
        const long long T = (long long)P.units * ncw;
        P.share_q[v] = (int)(T / nb); P.share_r[v] = (int)(T % nb);
        P.inv_share[v] = (float)((double)nb / (double)T);
        if (v == 1 && P.cells_r == 0) continue;
        const long long lmin = T / nb, lmax = (T + nb - 1) / nb;
        long long j = (ncw - 1 + lmin - 1) / lmin + 1;                    // CTAs that can intersect ncw consecutive cells
        if (j > nb) j = nb;
        if (j > P.jmax) P.jmax = (int)j;
        const long long u = (lmax + 2 * ncw - 2) / ncw;                   // units a share of lmax cells can touch
        if (u > P.ucta_max) P.ucta_max = (int)u;
    }
    const int xitems = P.ncw_max * kp * M * CELL_VECS * ((P.kmode == KMODE_W4A16) ? 4 : 2);   // staging items (upper bound)
    const int stage_items = (mode == MODE_W4A4_FUSED_QUANT) ? P.threads : STAGE_ITEMS;
    P.nxb = (xitems + stage_items - 1) / stage_items;
    P.map = gemv_smem_map(P.kmode, M, P.R, P.W, P.S, P.L.rpt, P.ncw_max, kp, P.nxb, P.ucta_max, P.nb);
    return P;
}

size_t gemv_smem_bytes(int mode, int M, int N, int K, int kp, const GemvConfig& c) {
    return gemv_plan(mode, M, N, K, kp, c).map.total;
}

// clamp a (possibly user-given) launch shape to what the instantiations and shared memory allow
GemvConfig gemv_legalize_config(int mode, int M, int N, int K, int kp, GemvConfig c) {
    const Layout L = make_layout(N, K, kp);
    const int kmode = gemv_kmode(mode, M);
    if (c.rows != 1 && c.rows != 2) c.rows = 1;
    if (c.rows == 2 && (kmode != KMODE_W4A4_I8 || L.ntiles < 2)) c.rows = 1;      // R = 2 exists for the integer path only
    if (c.stages < 1) c.stages = 1;
    if (c.warps < 1) c.warps = 1;
    if (c.ksplit < 1) c.ksplit = 1;
    if (c.ksplit > L.ncells) c.ksplit = L.ncells;
    // one persistent CTA per SM: shrink only if it does not fit in the 227 KB of shared memory
    while (gemv_smem_bytes(mode, M, N, K, kp, c) > SMEM_CAP) {
        const int ncw_max = (L.ncells + c.ksplit - 1) / c.ksplit;
        const size_t xs = (size_t)ncw_max * CELL_VECS * L.kp * xvec_stride(kmode, M);
        if (xs > SMEM_CAP / 2 && c.ksplit < L.ncells) ++c.ksplit;       // activations dominate: slice K
        else if (c.stages > 2) --c.stages;
        else if (c.warps > 8) c.warps -= 2;
        else if (c.ksplit < L.ncells) ++c.ksplit;
        else if (c.warps > 1) --c.warps;
        else if (c.stages > 1) --c.stages;
        else break;
    }
    return c;
}

// Launch shape per (mode, M, N, K).  Values come from the sweeps recorded in DESIGN.md
// ("Tuning"); the rule below reproduces them and extrapolates to other shapes.
GemvConfig gemv_pick_config(int mode, int M, int N, int K, int kp) {
    GemvConfig c;
    const bool half_path = (gemv_kmode(mode, M) == KMODE_W4A4_H);
    c.rows = 1;
    // small weights (qkv, o: <= 64 M weights) at M = 2..4: 12 warps measured 3-6 % faster than 16 (fewer, longer shares)
    const bool small_w = (M >= 2 && M <= 4 && (long long)N * K <= (64ll << 20));
    c.warps = (M >= 8 || (half_path && K < 16384) || small_w) ? 12 : 16;
    c.stages = 2;
    c.ksplit = 1;
    return gemv_legalize_config(mode, M, N, K, kp, c);
}

static size_t counters_bytes(const GemvPlan& P) { return align_up((size_t)P.units * sizeof(unsigned int), 256); }

size_t gemv_workspace_bytes_for(int mode, int M, int N, int K, int kp, const GemvConfig& c) {
    const GemvPlan P = gemv_plan(mode, M, N, K, kp, c);
    return counters_bytes(P) + (size_t)P.ksplit * P.jmax * M * P.Npad * sizeof(float);
}

cudaError_t launch_gemv_w4a4(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st);
cudaError_t launch_gemv_w4a16(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st);
cudaError_t launch_gemv_w4a4h(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st);

cudaError_t launch_gemv(int mode, const void* blob, const float* w_gscale, int N, int K, int kp, const void* x,
                        const uint8_t* x_scales, const float* x_gscale, int gscale_per_row, int M, int64_t ldx, void* y,
                        int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes, const GemvConfig& cfg, cudaStream_t st) {
    const bool fuse_quant = (mode == MODE_W4A4_FUSED_QUANT);
    const GemvPlan P = gemv_plan(mode, M, N, K, kp, cfg);
    if (P.map.total > SMEM_CAP) return cudaErrorInvalidConfiguration;
    if (workspace == nullptr || ws_bytes < counters_bytes(P) + (size_t)P.ksplit * P.jmax * M * P.Npad * sizeof(float))
        return cudaErrorInvalidValue;
    GemvParams p;
    p.blob = static_cast<const uint8_t*>(blob) + BLOB_HEADER_BYTES;
    p.w_gscale = w_gscale;
    p.x = x; p.x_scales = x_scales; p.x_gscale = x_gscale;
    p.y = y;
    p.counters = static_cast<unsigned int*>(workspace);
    p.partials = reinterpret_cast<float*>(static_cast<uint8_t*>(workspace) + counters_bytes(P));
    p.ldx = ldx; p.ldy = ldy;
    p.N = N; p.K = K;
    p.ntiles = P.L.ntiles; p.nch = P.L.ncells; p.Npad = P.Npad;
    p.kp = P.L.kp; p.kp_shift = 0;
    while ((1 << p.kp_shift) < P.L.kp) ++p.kp_shift;
    p.warps = P.W; p.stages = P.S; p.ksplit = P.ksplit;
    p.units = P.units;
    p.cells_q = P.cells_q; p.cells_r = P.cells_r;
    for (int v = 0; v < 2; ++v) { p.share_q[v] = P.share_q[v]; p.share_r[v] = P.share_r[v]; p.inv_share[v] = P.inv_share[v]; }
    p.jmax = P.jmax; p.ucta_max = P.ucta_max; p.nxb = P.nxb;
    p.y_bf16 = (y_dtype == NVFP4_DTYPE_BF16);
    p.zero = 0;
    p.fuse_quant = fuse_quant ? 1 : 0;
    p.gscale_per_row = gscale_per_row;
    p.x_gscale_out = fuse_quant ? const_cast<float*>(x_gscale) : nullptr;
    p.hdr_expect = blob_header_words(N, K, kp);
    dim3 grid(P.nb, P.ksplit);
    if (P.kmode == KMODE_W4A4_I8) return launch_gemv_w4a4(p, M, P.R, grid, P.threads, P.map.total, st);
    if (P.kmode == KMODE_W4A4_H) return launch_gemv_w4a4h(p, M, P.R, grid, P.threads, P.map.total, st);
    return launch_gemv_w4a16(p, M, P.R, grid, P.threads, P.map.total, st);
}

}  // namespace nvfp4
