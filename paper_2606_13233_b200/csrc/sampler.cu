// sampler.cu -- the ReSET sampler step (Sec. 4 :107-139): ONE launch per decoded
// token and sequence does
//   token entropy H_t of softmax(z_t)  ->  running global mean and the hybrid step-entropy estimate
//   HSE (Eq. 3 :130-137)  ->  step-aware threshold SAT (Eq. 2 :113)  ->  temperature (Eq. 1 :90)  ->  top-p (0.95,
//   :412) sample from softmax(z_t / T_t)  ->  step-boundary update (delimiter token, :367).
//
// Design: one thread-block CLUSTER of 8 CTAs x 512 threads per sequence holds the whole vocabulary in registers
// (<= 40 logits per thread, V <= 163840; Qwen3: 151936): the logits are read from HBM exactly once, every
// vocabulary-wide reduction (max, sums, the top-p threshold search, the arg-max of the exponential race) is
// warp shuffle -> shared memory -> distributed shared memory -> cluster.sync, in a FIXED order (deterministic).
// top-p needs no sort: the kept set is {v : key(z_v) >= k*}, k* = the smallest order-preserving 32-bit key whose
// strictly-above probability mass is < p, found by bisection on the key bits (<= 32 cluster reductions).
// The draw is the exponential race argmax_v z_v/T - log(-log u_v) over the kept tokens with u_v from
// Philox4x32-10 (counter = (v, t, 0, 0), key = seed): the oracle implements the same generator (R19).
// The scalar state (ring of the last 32 entropies, sums, t, t0) lives in device memory owned by the caller.
#include <cooperative_groups.h>

#include "nvfp4_common.cuh"
#include "nvfp4_internal.h"

namespace cg = cooperative_groups;

namespace nvfp4 {

constexpr int SAMP_CTAS = 8, SAMP_THREADS = 512, SAMP_E = 40;      // 128 registers per thread: logits and their exponentials stay in registers
constexpr int SAMP_VMAX = SAMP_CTAS * SAMP_THREADS * SAMP_E;      // 163840
constexpr int SAMP_RING = 32;                                     // w <= 32 (the paper's w)

struct ResetStateDev {            // RESET_STATE_BYTES = 160
    float ring[SAMP_RING];        // H_i of the last 32 positions, slot = i % 32
    double gsum;                  // sum of all H_i
    double ssum;                  // sum of H_i with i >= t0 (current step)
    int t;                        // positions processed so far
    int t0;                       // first position of the current step
    int pad[2];
};
static_assert(sizeof(ResetStateDev) == 160, "state layout is part of the ABI");

struct SamplerParams {
    const void* logits; int logits_bf16; int64_t ld; int V;
    ResetStateDev* state;         // [B]
    float tau0, t_low, t_high, top_p; int w; int delimiter;
    unsigned int seed_lo, seed_hi;
    int* token_out;               // [B]
    float* diag_out;              // [B][8] or NULL: H, H_step, H_bar, tau, T, nucleus size, t, t0 (after the step)
};

__device__ __forceinline__ uint32_t order_key(float z) {          // monotone float -> uint32
    const uint32_t b = __float_as_uint(z);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ uint32_t philox_x0(uint32_t c0, uint32_t c1, uint32_t k0, uint32_t k1) {
    uint32_t c2 = 0u, c3 = 0u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return c0;
}

// ---- cluster-wide reductions in a fixed order --------------------------------------------------------------------
struct RedScratch {
    float warp[3][32];            // per-warp partials (up to 3 components; 16 warps, the rest stays at the identity)
    float cta[2][3][SAMP_CTAS];   // [phase][component][source CTA], written through DSMEM
};
// sums (or maxima) of NC floats over the whole cluster; every thread gets the result
template <int NC, bool IS_MAX>
__device__ __forceinline__ void cluster_reduce(float (&v)[NC], RedScratch* sc, int& phase, cg::cluster_group& cluster) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int c = 0; c < NC; ++c) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            const float o = __shfl_xor_sync(0xFFFFFFFFu, v[c], off);
            v[c] = IS_MAX ? fmaxf(v[c], o) : v[c] + o;
        }
        if (lane == 0) sc->warp[c][warp] = v[c];
    }
    __syncthreads();
    if (warp == 0) {
        const unsigned rank = cluster.block_rank();
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            float x = lane < SAMP_THREADS / 32 ? sc->warp[c][lane] : (IS_MAX ? -INFINITY : 0.0f);
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                const float o = __shfl_xor_sync(0xFFFFFFFFu, x, off);
                x = IS_MAX ? fmaxf(x, o) : x + o;
            }
            if (lane < SAMP_CTAS) cluster.map_shared_rank(&sc->cta[phase][c][0], lane)[rank] = x;   // to every CTA's slot[rank]
        }
    }
    cluster.sync();
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        float x = sc->cta[phase][c][0];
#pragma unroll
        for (int r = 1; r < SAMP_CTAS; ++r) x = IS_MAX ? fmaxf(x, sc->cta[phase][c][r]) : x + sc->cta[phase][c][r];
        v[c] = x;
    }
    phase ^= 1;
}

__global__ void __launch_bounds__(SAMP_THREADS) reset_sampler_kernel(const SamplerParams p) {
    __shared__ RedScratch sc;
    __shared__ float bcast[8];
    cg::cluster_group cluster = cg::this_cluster();
    const unsigned rank = cluster.block_rank();
    const int seq = blockIdx.x / SAMP_CTAS;
    int phase = 0;
    pdl_wait();                                                   // the logits come from the previous kernel
    pdl_launch_dependents();
    ResetStateDev* st = p.state + seq;

    // ---- the vocabulary in registers ----
    float z[SAMP_E];
    const int v0 = (int)rank * SAMP_THREADS + (int)threadIdx.x;
#pragma unroll
    for (int i = 0; i < SAMP_E; ++i) {
        const int v = v0 + i * (SAMP_CTAS * SAMP_THREADS);
        float x = -INFINITY;
        if (v < p.V) {
            if (p.logits_bf16) x = bf16_bits_to_float(__ldg(static_cast<const uint16_t*>(p.logits) + (int64_t)seq * p.ld + v));
            else               x = __ldg(static_cast<const float*>(p.logits) + (int64_t)seq * p.ld + v);
        }
        z[i] = x;
    }
    cluster.sync();          // every CTA of the cluster runs (required before the first distributed-shared-memory store)
    // ---- H_t = -sum p log p of softmax(z_t)  (entropy at temperature 1, R14) ----
    float mx[1] = {-INFINITY};
#pragma unroll
    for (int i = 0; i < SAMP_E; ++i) mx[0] = fmaxf(mx[0], z[i]);
    cluster_reduce<1, true>(mx, &sc, phase, cluster);
    const float m = mx[0];
    // numerically careful for near-deterministic positions (H << 1): the maximal logits contribute exactly 1 each, the
    // rest A' = sum_{z<m} e^(z-m) is summed on its own, log A = log(n_max) + log1p(A'/n_max), and
    // H = sum_v p_v (log A - (z_v - m)) is a sum of NON-NEGATIVE terms (no cancellation)
    float na[2] = {0.0f, 0.0f};                                   // {n_max, A'}
#pragma unroll
    for (int i = 0; i < SAMP_E; ++i) {
        const float d = z[i] - m;                                 // -inf for padding: e = 0, contributes nothing
        if (d == 0.0f) na[0] += 1.0f; else na[1] += expf(d);
    }
    cluster_reduce<2, false>(na, &sc, phase, cluster);
    const float logA = logf(na[0]) + log1pf(na[1] / na[0]);
    float hs[1] = {0.0f};
#pragma unroll
    for (int i = 0; i < SAMP_E; ++i) {
        const float d = z[i] - m;
        const float e = expf(d);
        hs[0] += (d < 0.0f && e > 0.0f) ? e * (logA - d) : 0.0f;
    }
    cluster_reduce<1, false>(hs, &sc, phase, cluster);
    const float H = (na[0] * logA + hs[0]) / (na[0] + na[1]);

    // ---- Eqs. 3, 2, 1: scalar bookkeeping (one thread per CTA, identical in every CTA; double for the sums) ----
    if (threadIdx.x == 0) {
        const int t = st->t, t0 = st->t0;
        const double gsum = st->gsum + (double)H;
        const double ssum = st->ssum + (double)H;
        const double h_bar = gsum / (double)(t + 1);
        double h_step;
        if (t - t0 < p.w) {                                       // window of the min(w, t+1) most recent positions (R15)
            const int n = (t + 1 < p.w) ? t + 1 : p.w;
            double s = (double)H;
            for (int j = 1; j < n; ++j) s += (double)st->ring[(t - j) & (SAMP_RING - 1)];
            h_step = s / (double)n;
        } else {
            h_step = ssum / (double)(t - t0 + 1);
        }
        const double tau = (h_step <= h_bar) ? (double)p.tau0 : h_step;       // Eq. 2 (tie -> confident, R17)
        const float T = ((double)H < tau) ? p.t_low : p.t_high;              // Eq. 1
        bcast[0] = T; bcast[1] = (float)h_step; bcast[2] = (float)h_bar; bcast[3] = (float)tau;
    }
    __syncthreads();
    const float T = bcast[0];
    const float inv_T = 1.0f / T;

    // ---- top-p on softmax(z / T): kept = {v : mass of strictly more probable tokens < p}  (R18) ----
    float e[SAMP_E];
    float at[1] = {0.0f};
#pragma unroll
    for (int i = 0; i < SAMP_E; ++i) { e[i] = expf((z[i] - m) * inv_T); at[0] += e[i]; }
    cluster_reduce<1, false>(at, &sc, phase, cluster);
    const float limit = p.top_p * at[0];
    uint32_t lo = 0u, hi = 0xFFFFFFFFu;                           // smallest key k with mass{key > k} < p * A_T
    while (lo < hi) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        float s[1] = {0.0f};
#pragma unroll
        for (int i = 0; i < SAMP_E; ++i) s[0] += (order_key(z[i]) > mid) ? e[i] : 0.0f;
        cluster_reduce<1, false>(s, &sc, phase, cluster);
        if (s[0] < limit) hi = mid; else lo = mid + 1u;
    }
    const uint32_t kstar = lo;

    // ---- exponential race over the kept tokens: argmax z/T - log(-log u), ties to the lowest index (R19) ----
    const uint32_t t_now = (uint32_t)st->t;
    float best = -INFINITY; int best_v = 0x7FFFFFFF; float kept = 0.0f;
#pragma unroll
    for (int i = 0; i < SAMP_E; ++i) {
        const int v = v0 + i * (SAMP_CTAS * SAMP_THREADS);
        if (v < p.V && order_key(z[i]) >= kstar) {
            kept += 1.0f;
            const uint32_t x0 = philox_x0((uint32_t)v, t_now, p.seed_lo, p.seed_hi);
            const float u = ((float)(x0 >> 9) + 0.5f) * 1.1920928955078125e-07f;     // (k + 0.5) * 2^-23: exact
            const float score = (z[i] - m) * inv_T - logf(-logf(u));
            if (score > best || (score == best && v < best_v)) { best = score; best_v = v; }
        }
    }
    // arg-max across the cluster: first the maximum, then the lowest index that attains it
    float bm[2] = {best, kept};
    {
        float b1[1] = {best};
        cluster_reduce<1, true>(b1, &sc, phase, cluster);
        bm[0] = b1[0];
        float k1[1] = {kept};
        cluster_reduce<1, false>(k1, &sc, phase, cluster);
        bm[1] = k1[0];
    }
    float cand[1] = {(best == bm[0]) ? -(float)best_v : -INFINITY};          // V < 2^24: indices are exact in FP32
    cluster_reduce<1, true>(cand, &sc, phase, cluster);
    const int token = (int)(-cand[0]);

    // ---- write back (rank 0, thread 0; every CTA finished reading the state before the last cluster.sync) ----
    if (rank == 0 && threadIdx.x == 0) {
        const int t = st->t;
        int t0 = st->t0;
        st->ring[t & (SAMP_RING - 1)] = H;
        st->gsum += (double)H;
        st->ssum = (token == p.delimiter) ? 0.0 : st->ssum + (double)H;     // the delimiter ends its step (R16)
        if (token == p.delimiter) t0 = t + 1;
        st->t0 = t0;
        st->t = t + 1;
        p.token_out[seq] = token;
        if (p.diag_out != nullptr) {
            float* d = p.diag_out + (int64_t)seq * 8;
            d[0] = H; d[1] = bcast[1]; d[2] = bcast[2]; d[3] = bcast[3]; d[4] = T; d[5] = bm[1];
            d[6] = (float)(t + 1); d[7] = (float)t0;
        }
    }
}

cudaError_t launch_reset_sampler(const void* logits, int logits_bf16, int B, int V, int64_t ld, void* state, float tau0,
                                 float t_low, float t_high, float top_p, int w, int delimiter, unsigned long long seed,
                                 int* token_out, float* diag_out, cudaStream_t st) {
    if (V > SAMP_VMAX) return cudaErrorInvalidConfiguration;
    SamplerParams p;
    p.logits = logits; p.logits_bf16 = logits_bf16; p.ld = ld; p.V = V;
    p.state = static_cast<ResetStateDev*>(state);
    p.tau0 = tau0; p.t_low = t_low; p.t_high = t_high; p.top_p = top_p; p.w = w; p.delimiter = delimiter;
    p.seed_lo = (unsigned int)(seed & 0xFFFFFFFFull); p.seed_hi = (unsigned int)(seed >> 32);
    p.token_out = token_out; p.diag_out = diag_out;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(SAMP_CTAS * B);
    cfg.blockDim = dim3(SAMP_THREADS);
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = SAMP_CTAS; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    attr[1] = pdl_attribute();
    cfg.attrs = attr; cfg.numAttrs = 2;
    return cudaLaunchKernelEx(&cfg, reset_sampler_kernel, p);
}

}  // namespace nvfp4
