// gemv.cu -- host side of the GEMV: launch-shape table, stream-K plan, workspace layout, template dispatch.
#include "gemv_kernel.cuh"

namespace nvfp4 {

constexpr int NUM_SMS = 148;          // B200
constexpr size_t SMEM_CAP = 227 * 1024;

unsigned long long* g_trace = nullptr;     // debug only (nvfp4_debug_set_trace)

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// arithmetic variant: W4A4 runs the FP16 path (F2FP + HFMA2) at M = 1, the integer path (PRMT + dp4a) above
int gemv_kmode(int mode, int M) {
    if (mode == NVFP4_MODE_W4A16) return KMODE_W4A16;
    return M <= 1 ? KMODE_W4A4_H : KMODE_W4A4_I8;
}

// everything the launch derives from (mode, M, N, K, kp, config): one place for smem, workspace and kernel params
struct GemvPlan {
    int kmode, M, R, W, S, ksplit, nb, cps, stager_warps, whole;
    Layout L;
    int units, cells_q, cells_r, ncw_max;
    int base, ur;
    int nba[2], a_q[2], a_r[2];
    float inv_a[2];
    int amax, jmax, nxb, nhand, threads, npad_a, npad_b;
    SmemMap map;
};

static GemvPlan gemv_plan(int mode, int M, int N, int K, int kp, const GemvConfig& c) {
    GemvPlan P;
    P.kmode = gemv_kmode(mode, M);
    P.M = M; P.R = c.rows; P.S = c.stages;
    P.L = make_layout(N, K, kp);
    P.ksplit = c.ksplit < 1 ? 1 : (c.ksplit > P.L.ncells ? P.L.ncells : c.ksplit);
    P.units = (P.L.ntiles + P.R - 1) / P.R;
    P.cells_q = P.L.ncells / P.ksplit; P.cells_r = P.L.ncells % P.ksplit;
    P.ncw_max = P.cells_q + (P.cells_r > 0 ? 1 : 0);
    // CTAs per K slice: about one per SM over all slices, never more than the smallest slice has cells
    const long long t_min = (long long)P.units * P.cells_q;
    P.cps = c.cps < 1 ? 1 : (c.cps > 3 ? 3 : c.cps);
    P.stager_warps = P.cps > 1 ? 2 : STAGER_WARPS;
    int nb = NUM_SMS * P.cps / P.ksplit;
    if (nb < 1) nb = 1;
    if (nb > t_min) nb = (int)t_min;
    P.nb = nb;
    // data-parallel part: `base` whole units per CTA; stream-K part: the leftover units' cells in equal shares
    P.base = P.units / nb;
    P.ur = P.units - P.base * nb;
    P.whole = c.whole ? 1 : 0;
    P.npad_a = P.whole ? 0 : P.ur * P.R * P.L.rpt;
    P.npad_b = P.units * P.R * P.L.rpt;
    P.amax = 0; P.jmax = 1;
    long long min_cells = 1ll << 40;                                      // smallest per-CTA cell count
    for (int v = 0; v < 2; ++v) {
        const long long ncw = P.cells_q + v;
        const long long Tr = P.whole ? 0 : (long long)P.ur * ncw;
        const long long nba = Tr < nb ? Tr : nb;
        P.nba[v] = (int)nba;
        P.a_q[v] = nba ? (int)(Tr / nba) : 0; P.a_r[v] = nba ? (int)(Tr % nba) : 0;
        P.inv_a[v] = Tr ? (float)((double)nba / (double)Tr) : 0.0f;
        if (v == 1 && P.cells_r == 0) continue;
        const long long cta_min = P.base * ncw + (nba == nb ? Tr / nb : 0);
        if (cta_min < min_cells) min_cells = cta_min;
        if (nba == 0) continue;
        const long long amin = Tr / nba, amax = (Tr + nba - 1) / nba;
        if (amax > P.amax) P.amax = (int)amax;
        long long j = (ncw - 1 + amin - 1) / amin + 1;                    // CTAs that can intersect ncw consecutive cells
        if (j > nba) j = nba;
        if (j > P.jmax) P.jmax = (int)j;
    }
    // every consumer warp gets at least one cell of phase B (if there is one); launch bounds of the instantiation
    const int max_warps = (gemv_max_threads(P.kmode, M, P.R) - STAGER_THREADS) / 32 / P.cps;   // registers: cps CTAs share the SM
    int W = c.warps < 1 ? 1 : c.warps;
    if (P.base > 0 && W > (long long)P.base * P.cells_q) W = (int)((long long)P.base * P.cells_q);
    if (P.base == 0 && W > min_cells) W = (int)(min_cells > 1 ? min_cells : 1);
    if (W > max_warps) W = max_warps;
    P.W = W;
    P.threads = (W + P.stager_warps) * 32;
    const int xitems = P.ncw_max * kp * M * CELL_VECS * ((P.kmode == KMODE_W4A16) ? 4 : 2);   // staging items (upper bound)
    const int stage_items = (mode == MODE_W4A4_FUSED_QUANT) ? P.threads : P.threads * STAGE_BATCH;
    P.nxb = (xitems + stage_items - 1) / stage_items;
    P.nhand = 2 + (P.ksplit > 1 ? P.base + 1 : 0);
    P.map = gemv_smem_map(P.kmode, M, P.R, P.W, P.S, P.L.rpt, P.ncw_max, kp, P.nxb, P.base, P.nb, P.amax, P.nhand);
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
    if (c.cps < 1) c.cps = 1;
    if (c.cps > 3) c.cps = 3;
    if (c.ksplit < 1) c.ksplit = 1;
    if (c.ksplit > L.ncells) c.ksplit = L.ncells;
    // one persistent CTA per SM: shrink only if it does not fit in the 227 KB of shared memory
    while (gemv_smem_bytes(mode, M, N, K, kp, c) > SMEM_CAP / c.cps - (c.cps > 1 ? 1024 : 0)) {
        const int ncw_max = (L.ncells + c.ksplit - 1) / c.ksplit;
        const size_t xs = (size_t)ncw_max * CELL_VECS * L.kp * xvec_stride(kmode, M);
        if (c.cps > 1 && xs > SMEM_CAP / c.cps / 2) --c.cps;                // activations too large for several CTAs per SM
        else if (xs > SMEM_CAP / 2 && c.ksplit < L.ncells) ++c.ksplit;  // activations dominate: slice K
        else if (c.stages > 2) --c.stages;
        else if (c.warps > 8) c.warps -= 2;
        else if (c.ksplit < L.ncells) ++c.ksplit;
        else if (c.warps > 1) --c.warps;
        else if (c.stages > 1) --c.stages;
        else break;
    }
    return c;
}

// Launch shape per (mode, M, N, K).  Values come from the round-2 sweeps on B200 (profiles/r02_sweep.md, DESIGN.md
// "Tuning"); the rule below reproduces them and extrapolates to other shapes.
GemvConfig gemv_pick_config(int mode, int M, int N, int K, int kp) {
    GemvConfig c;
    const int kmode = gemv_kmode(mode, M);
    const bool big = (long long)N * K >= (128ll << 20);                   // gate_up-sized weights: 16 warps pay (M <= 2)
    const bool mid = (long long)N * K >= (120ll << 20);                   // down-sized: 16 warps pay at M = 1 (profiles/r02_sweep.md)
    c.rows = 1;
    c.warps = (kmode == KMODE_W4A16 || M >= 3) ? 12 : ((big || (mid && M == 1)) ? 16 : 12);
    c.stages = 2;        // three stages measured 3-5 % slower everywhere: more bytes in flight than the memory system wants
    c.ksplit = 1;
    c.cps = 1;           // two half-size CTAs per SM measured no faster
    // balance: whole units per CTA unless the rows are long (K >= 16384) and M >= 2: there the equal-bytes split wins
    c.whole = (M >= 2 && K >= 16384) ? 0 : 1;
    return gemv_legalize_config(mode, M, N, K, kp, c);
}

// workspace: [units] arrival counters | partials of the leftover units | partials of the whole units (K slices only)
static size_t counters_bytes(const GemvPlan& P) { return align_up((size_t)P.units * sizeof(unsigned int), 256); }
static size_t partials_a_bytes(const GemvPlan& P) { return align_up((size_t)P.ksplit * P.jmax * P.M * P.npad_a * sizeof(float), 256); }
static size_t partials_b_bytes(const GemvPlan& P) { return P.ksplit > 1 ? (size_t)P.ksplit * P.M * P.npad_b * sizeof(float) : 0; }

size_t gemv_workspace_bytes_for(int mode, int M, int N, int K, int kp, const GemvConfig& c) {
    const GemvPlan P = gemv_plan(mode, M, N, K, kp, c);
    return counters_bytes(P) + partials_a_bytes(P) + partials_b_bytes(P);
}

cudaError_t launch_gemv_w4a4(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st);
cudaError_t launch_gemv_w4a16(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st);
cudaError_t launch_gemv_w4a4h(const GemvParams& p, int M, int R, dim3 grid, int threads, size_t smem, cudaStream_t st);

cudaError_t launch_gemv(int mode, const void* blob, const float* w_gscale, int N, int K, int kp, const void* x,
                        const uint8_t* x_scales, const float* x_gscale, int gscale_per_row, int M, int64_t ldx, void* y,
                        int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes, const GemvConfig& cfg, cudaStream_t st,
                        const void* x_records) {
    const bool fuse_quant = (mode == MODE_W4A4_FUSED_QUANT);
    const GemvPlan P = gemv_plan(mode, M, N, K, kp, cfg);
    if (x_records != nullptr && (mode != NVFP4_MODE_W4A4 || P.kmode != KMODE_W4A4_H)) return cudaErrorInvalidValue;
    if (P.map.total > SMEM_CAP) return cudaErrorInvalidConfiguration;
    if (workspace == nullptr || ws_bytes < counters_bytes(P) + partials_a_bytes(P) + partials_b_bytes(P))
        return cudaErrorInvalidValue;
    GemvParams p;
    p.blob = static_cast<const uint8_t*>(blob) + BLOB_HEADER_BYTES;
    p.w_gscale = w_gscale;
    p.x = x; p.x_scales = x_scales; p.x_gscale = x_gscale;
    p.y = y;
    p.counters = static_cast<unsigned int*>(workspace);
    p.partials_a = reinterpret_cast<float*>(static_cast<uint8_t*>(workspace) + counters_bytes(P));
    p.partials_b = reinterpret_cast<float*>(static_cast<uint8_t*>(workspace) + counters_bytes(P) + partials_a_bytes(P));
    p.ldx = ldx; p.ldy = ldy;
    p.N = N; p.K = K;
    p.ntiles = P.L.ntiles; p.nch = P.L.ncells; p.npad_a = P.npad_a; p.npad_b = P.npad_b;
    p.kp = P.L.kp; p.kp_shift = 0;
    while ((1 << p.kp_shift) < P.L.kp) ++p.kp_shift;
    p.warps = P.W; p.stages = P.S; p.ksplit = P.ksplit;
    p.units = P.units;
    p.cells_q = P.cells_q; p.cells_r = P.cells_r;
    p.base = P.base; p.ur = P.ur; p.whole_units = P.whole;
    for (int v = 0; v < 2; ++v) { p.nba[v] = P.nba[v]; p.a_q[v] = P.a_q[v]; p.a_r[v] = P.a_r[v]; p.inv_a[v] = P.inv_a[v]; }
    p.amax = P.amax; p.jmax = P.jmax; p.nxb = P.nxb; p.nhand = P.nhand;
    p.fd_w = fastdiv_make((uint32_t)P.W);
    for (int v = 0; v < 2; ++v) { p.fd_ncw[v] = fastdiv_make((uint32_t)(P.cells_q + v)); p.fd_nba[v] = fastdiv_make((uint32_t)P.nba[v]); }
    {
        const uint32_t mm[13] = {P.map.xs, P.map.ring, P.map.slots, P.map.aslots, P.map.hand, P.map.bars, P.map.xbars, P.map.hbars,
                                 P.map.cnt, P.map.bstart, P.map.astart, P.map.misc, P.map.total};
        for (int i = 0; i < 13; ++i) p.smem_map[i] = mm[i];
    }
    p.y_bf16 = (y_dtype == NVFP4_DTYPE_BF16);
    p.zero = 0;
    p.fuse_quant = fuse_quant ? 1 : 0;
    p.gscale_per_row = gscale_per_row;
    p.x_gscale_out = fuse_quant ? const_cast<float*>(x_gscale) : nullptr;
    p.x_records = static_cast<const uint8_t*>(x_records);
    p.hdr_expect = blob_header_words(N, K, kp);
    p.trace = g_trace;
    dim3 grid(P.nb, P.ksplit);
    if (P.kmode == KMODE_W4A4_I8) return launch_gemv_w4a4(p, M, P.R, grid, P.threads, P.map.total, st);
    if (P.kmode == KMODE_W4A4_H) return launch_gemv_w4a4h(p, M, P.R, grid, P.threads, P.map.total, st);
    return launch_gemv_w4a16(p, M, P.R, grid, P.threads, P.map.total, st);
}

}  // namespace nvfp4
