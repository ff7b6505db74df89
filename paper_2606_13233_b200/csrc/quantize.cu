// quantize.cu -- fused BF16 -> NVFP4 activation quantizer (steps a1+a2; the paper's kernel "Q",
// PAPER.md:242, Table 3 :209-217).  One launch: every thread keeps its 16-element blocks in
// registers, the tensor-wide amax is reduced warp -> CTA -> thread-block cluster (DSMEM), then the
// same registers are quantised.  X is read from HBM/L2 exactly once.
//
// Bit-exact contract (R1/R2): every op below is ONE binary32 RNE operation
// (__fdiv_rn / __fmul_rn; this file must never be compiled with -use_fast_math).
#include <cooperative_groups.h>

#include "nvfp4_common.cuh"
#include "nvfp4_internal.h"
#include "quant_block.cuh"

namespace cg = cooperative_groups;

namespace nvfp4 {

constexpr int QTHREADS_MAX = 1024;
constexpr int QCLUSTER_MAX = 8;

// quantise one 16-element block held as 8 packed BF16 pairs; returns 8 code bytes + scale byte
__device__ __forceinline__ void quantize_block(const uint4& a, const uint4& b, uint32_t ab_bits, float g,
                                               uint2& out_codes, uint8_t& out_scale) {
    out_codes = make_uint2(0u, 0u);
    out_scale = 0;
    if (!(g > 0.0f)) return;                                   // amax == 0 (or bad static g): all zero
    uint8_t sc; float d;
    block_scale(ab_bits, g, sc, d);
    out_scale = sc;
    if (d == 0.0f) return;                                     // flushed block (R5): codes 0x0
    const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
    uint32_t lo = 0, hi = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float x0 = __uint_as_float(w[i] << 16);          // element 2i   (low half)
        const float x1 = __uint_as_float(w[i] & 0xFFFF0000u);  // element 2i+1 (high half)
        const uint32_t byte = float2_to_e2m1x2(__fdiv_rn(x0, d), __fdiv_rn(x1, d));
        if (i < 4) lo |= byte << (8 * i); else hi |= byte << (8 * (i - 4));
    }
    out_codes = make_uint2(lo, hi);
}

// ---- block loaders: where a thread's 16-element block comes from -------------------------------------
// plain: BF16 X[M,K] (row stride ldx)
struct LoadX {
    const uint16_t* x; int64_t ldx;
    __device__ __forceinline__ void operator()(int m, int kb, uint4& a, uint4& b) const {
        const uint4* p = reinterpret_cast<const uint4*>(x + (int64_t)m * ldx + (int64_t)kb * 16);
        a = __ldg(p); b = __ldg(p + 1);
    }
    // L2 prefetch of the block's line, issued BEFORE griddepcontrol.wait: harmless whoever writes X (L2 is the point of
    // coherence), and when X is not the predecessor's output (a fresh token's hidden state, DRAM-cold) the loads after the
    // wait find it in L2
    __device__ __forceinline__ void prefetch(int m, int kb) const {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(x + (int64_t)m * ldx + (int64_t)kb * 16));
    }
};
// fused SiLU*mul (step a8 + a1 + a2 in one launch): the block is
// h[m, 16kb..] = RN_bf16(silu(gu[m, j]) * gu[m, I + j]) -- the same FP32 expression and BF16 rounding as
// silu_mul_kernel (misc.cu), so codes / scales / g equal nvfp4_silu_mul followed by nvfp4_quantize_act bit for bit.
struct LoadSiluMul {
    const uint16_t* gu; int I; uint16_t* h_out;     // h_out: optional BF16 [M, I] copy of the intermediate
    __device__ __forceinline__ void operator()(int m, int kb, uint4& a, uint4& b) const {
        const uint4* pg = reinterpret_cast<const uint4*>(gu + (int64_t)m * 2 * I + (int64_t)kb * 16);
        const uint4* pu = reinterpret_cast<const uint4*>(gu + (int64_t)m * 2 * I + I + (int64_t)kb * 16);
        const uint4 g0 = __ldg(pg), g1 = __ldg(pg + 1), u0 = __ldg(pu), u1 = __ldg(pu + 1);
        const uint32_t gw[8] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
        const uint32_t uw[8] = {u0.x, u0.y, u0.z, u0.w, u1.x, u1.y, u1.z, u1.w};
        uint32_t o[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const float ga = __uint_as_float(gw[i] << 16), gb = __uint_as_float(gw[i] & 0xFFFF0000u);
            const float ua = __uint_as_float(uw[i] << 16), ub = __uint_as_float(uw[i] & 0xFFFF0000u);
            const float ha = __fdiv_rn(ga, 1.0f + expf(-ga)) * ua;
            const float hb = __fdiv_rn(gb, 1.0f + expf(-gb)) * ub;
            o[i] = (uint32_t)float_to_bf16_rn(ha) | ((uint32_t)float_to_bf16_rn(hb) << 16);
        }
        a = make_uint4(o[0], o[1], o[2], o[3]); b = make_uint4(o[4], o[5], o[6], o[7]);
        if (h_out != nullptr) {
            uint4* ph = reinterpret_cast<uint4*>(h_out + (int64_t)m * I + (int64_t)kb * 16);
            ph[0] = a; ph[1] = b;
        }
    }
    __device__ __forceinline__ void prefetch(int, int) const {}      // (gate_up was just written: L2-hot)
};

constexpr int QMODE_STATIC = 0, QMODE_DYNAMIC = 1, QMODE_DYNAMIC_PER_ROW = 2;

// where block b = (m, kb) of the result goes.  pack_mt == 0: canonical codes [M,K/2] / scales [M,K/16];
// pack_mt = MT > 0: the tensor-core GEMM's activation records (gemm_tc.cu: per 256 k a record of MT*128 code bytes in
// 8-token x 16-byte core matrices + four 512-byte scale chunks in tcgen05.cp order), `codes` = first record.
// pack_mt < 0: the CUDA-core GEMV's own activation records at M = 1 (GEMV_XRECORD_BYTES per 32 k: the 2 x 16 E2M1 values
// as f16 -- exact --, then the two block scales as FP32), so that the GEMV stages them with one bulk copy.
__device__ __forceinline__ void store_block(uint8_t* codes, uint8_t* scales, int pack_mt, int b, int m, int kb, uint2 c, uint8_t s) {
    if (pack_mt < 0) {
        uint8_t* rec = codes + (size_t)(kb >> 1) * GEMV_XRECORD_BYTES;
        uint32_t lo[4], hi[4];
        cvt_word_e2m1(c.x, lo);
        cvt_word_e2m1(c.y, hi);
        uint4* dst = reinterpret_cast<uint4*>(rec + (kb & 1) * 32);
        dst[0] = make_uint4(lo[0], lo[1], lo[2], lo[3]);
        dst[1] = make_uint4(hi[0], hi[1], hi[2], hi[3]);
        *reinterpret_cast<float*>(rec + 64 + (kb & 1) * 4) = e4m3_to_float(s);
    } else if (pack_mt == 0) {
        *reinterpret_cast<uint2*>(codes + (int64_t)b * 8) = c;      // [M,K/2] contiguous: block b -> 8 bytes
        scales[b] = s;
    } else {
        uint8_t* rec = codes + (size_t)(kb >> 4) * (size_t)(pack_mt * 128 + 2048);
        const int kc = (kb & 15) >> 1;
        *reinterpret_cast<uint2*>(rec + (size_t)(kc * (pack_mt >> 3) + (m >> 3)) * 128 + (m & 7) * 16 + (kb & 1) * 8) = c;
        rec[pack_mt * 128 + ((kb & 15) >> 2) * 512 + (m & 31) * 16 + (m >> 5) * 4 + (kb & 3)] = s;
    }
}

// One cluster (gridDim.x CTAs == cluster size) covers the whole tensor; BPT blocks per thread.
template <int BPT, int QMODE, typename Loader>
__global__ void __launch_bounds__(QTHREADS_MAX)
quantize_act_kernel(Loader load, int M, int K, uint8_t* __restrict__ codes, uint8_t* __restrict__ scales,
                    float* __restrict__ gscale, int pack_mt) {
    __shared__ uint32_t warp_max[32];
    __shared__ uint32_t row_max[8];                     // per-row mode: CTA-wide row maxima
    __shared__ uint32_t cta_max[QCLUSTER_MAX][8];       // [source CTA][row] (row 0 only in per-tensor mode)
    const int kb_per_row = K >> 4;
    const int NB = M * kb_per_row;
    const int nthreads = gridDim.x * blockDim.x;
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x;
    cg::cluster_group cluster = cg::this_cluster();
    // every CTA of the cluster must be running before its shared memory is written remotely: arrive now, wait
    // right before the DSMEM stores (the latency hides under the loads)
    if (QMODE != QMODE_STATIC && gridDim.x > 1) asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");
    if (QMODE == QMODE_DYNAMIC_PER_ROW && threadIdx.x < 8) row_max[threadIdx.x] = 0u;
#pragma unroll
    for (int i = 0; i < BPT; ++i) {
        const int b = gtid + i * nthreads;
        if (b < NB) load.prefetch(b / kb_per_row, b % kb_per_row);
    }
    pdl_wait();                                       // X is the previous kernel's output
    pdl_launch_dependents();                          // the GEMV may start streaming its weights now

    uint4 va[BPT], vb[BPT];
    uint32_t ab[BPT];
    int rowm[BPT];
    uint32_t tmax = 0;
#pragma unroll
    for (int i = 0; i < BPT; ++i) {
        const int b = gtid + i * nthreads;
        va[i] = vb[i] = make_uint4(0, 0, 0, 0);
        ab[i] = 0; rowm[i] = 0;
        if (b < NB) {
            const int m = b / kb_per_row, kb = b - m * kb_per_row;
            rowm[i] = m;
            load(m, kb, va[i], vb[i]);
            ab[i] = absmax_bits16(va[i], vb[i]);
            tmax = max(tmax, ab[i]);
        }
    }

    float g[BPT];
    if (QMODE == QMODE_DYNAMIC) {
        tmax = __reduce_max_sync(0xFFFFFFFFu, tmax);
        if ((threadIdx.x & 31) == 0) warp_max[threadIdx.x >> 5] = tmax;
        __syncthreads();
        if (threadIdx.x < 32) {
            const int nw = (blockDim.x + 31) >> 5;
            uint32_t v = (threadIdx.x < nw) ? warp_max[threadIdx.x] : 0u;
            v = __reduce_max_sync(0xFFFFFFFFu, v);
            if (threadIdx.x == 0) warp_max[0] = v;
        }
        __syncthreads();
        uint32_t amax_bits = warp_max[0];
        if (gridDim.x > 1) {
            const unsigned rank = cluster.block_rank();
            asm volatile("barrier.cluster.wait.aligned;" ::: "memory");
            if (threadIdx.x < gridDim.x)                         // push my max into every CTA's slot[rank]
                cluster.map_shared_rank(&cta_max[0][0], threadIdx.x)[rank * 8] = amax_bits;
            cluster.sync();
            amax_bits = 0;
            for (unsigned r = 0; r < gridDim.x; ++r) amax_bits = max(amax_bits, cta_max[r][0]);
        }
        const float gg = __fdiv_rn(__uint_as_float(amax_bits << 16), 2688.0f);
        if (gtid == 0) *gscale = gg;
#pragma unroll
        for (int i = 0; i < BPT; ++i) g[i] = gg;
    } else if (QMODE == QMODE_DYNAMIC_PER_ROW) {
        // per-token global scales (R3 variant): row maxima through shared-memory atomics, one per group of lanes
        // that hold blocks of the same row
        __syncthreads();                                         // row_max zeroed
#pragma unroll
        for (int i = 0; i < BPT; ++i) {
            const unsigned grp = __match_any_sync(0xFFFFFFFFu, rowm[i]);
            const uint32_t v = __reduce_max_sync(grp, ab[i]);
            if ((threadIdx.x & 31) == __ffs(grp) - 1 && v != 0u) atomicMax(&row_max[rowm[i]], v);
        }
        __syncthreads();
        if (gridDim.x > 1) {
            const unsigned rank = cluster.block_rank();
            asm volatile("barrier.cluster.wait.aligned;" ::: "memory");
            if (threadIdx.x < gridDim.x * 8) {                   // push my row maxima into every CTA's slot[rank][row]
                const unsigned dst = threadIdx.x >> 3, row = threadIdx.x & 7;
                cluster.map_shared_rank(&cta_max[0][0], dst)[rank * 8 + row] = row_max[row];
            }
            cluster.sync();
            if (threadIdx.x < 8) {
                uint32_t v = 0;
                for (unsigned r = 0; r < gridDim.x; ++r) v = max(v, cta_max[r][threadIdx.x]);
                row_max[threadIdx.x] = v;
            }
            __syncthreads();
        }
        if (gtid < M) gscale[gtid] = __fdiv_rn(__uint_as_float(row_max[gtid] << 16), 2688.0f);
#pragma unroll
        for (int i = 0; i < BPT; ++i) g[i] = __fdiv_rn(__uint_as_float(row_max[rowm[i]] << 16), 2688.0f);
    } else {
        const float gg = __ldg(gscale);
#pragma unroll
        for (int i = 0; i < BPT; ++i) g[i] = gg;
    }

#pragma unroll
    for (int i = 0; i < BPT; ++i) {
        const int b = gtid + i * nthreads;
        if (b < NB) {
            uint2 c; uint8_t s;
            quantize_block(va[i], vb[i], ab[i], g[i], c, s);
            const int kb = b - rowm[i] * kb_per_row;
            store_block(codes, scales, pack_mt, b, rowm[i], kb, c, s);
        }
    }
}

// ---- generic two-kernel path for tensors larger than one cluster can hold in registers ----
__global__ void __launch_bounds__(1024) amax_kernel(const uint16_t* __restrict__ x, int M, int K, int64_t ldx,
                                                    float* __restrict__ gscale) {
    __shared__ uint32_t warp_max[32];
    const int kb_per_row = K >> 4;
    const int NB = M * kb_per_row;
    uint32_t tmax = 0;
    for (int b = threadIdx.x; b < NB; b += blockDim.x) {
        const int m = b / kb_per_row, kb = b - m * kb_per_row;
        const uint4* p = reinterpret_cast<const uint4*>(x + (int64_t)m * ldx + (int64_t)kb * 16);
        tmax = max(tmax, absmax_bits16(__ldg(p), __ldg(p + 1)));
    }
    tmax = __reduce_max_sync(0xFFFFFFFFu, tmax);
    if ((threadIdx.x & 31) == 0) warp_max[threadIdx.x >> 5] = tmax;
    __syncthreads();
    if (threadIdx.x < 32) {
        uint32_t v = warp_max[threadIdx.x];
        v = __reduce_max_sync(0xFFFFFFFFu, v);
        if (threadIdx.x == 0) *gscale = __fdiv_rn(__uint_as_float(v << 16), 2688.0f);
    }
}

__global__ void __launch_bounds__(256) quantize_blocks_kernel(const uint16_t* __restrict__ x, int M, int K, int64_t ldx,
                                                              uint8_t* __restrict__ codes, uint8_t* __restrict__ scales,
                                                              const float* __restrict__ gscale, int pack_mt) {
    const int kb_per_row = K >> 4;
    const int NB = M * kb_per_row;
    const float g = *gscale;
    for (int b = blockIdx.x * blockDim.x + threadIdx.x; b < NB; b += gridDim.x * blockDim.x) {
        const int m = b / kb_per_row, kb = b - m * kb_per_row;
        const uint4* p = reinterpret_cast<const uint4*>(x + (int64_t)m * ldx + (int64_t)kb * 16);
        const uint4 a = __ldg(p), bb = __ldg(p + 1);
        uint2 c; uint8_t s;
        quantize_block(a, bb, absmax_bits16(a, bb), g, c, s);
        store_block(codes, scales, pack_mt, b, m, kb, c, s);
    }
}

template <int BPT, int QMODE, typename Loader>
static cudaError_t launch_cluster(int nctas, int threads, cudaStream_t st, Loader load, int M, int K,
                                  uint8_t* codes, uint8_t* scales, float* gscale, int pack_mt) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(nctas);
    cfg.blockDim = dim3(threads);
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    attr[1] = pdl_attribute();
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = nctas;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    if (nctas > 1) { cfg.attrs = attr; cfg.numAttrs = 2; }
    else           { cfg.attrs = attr + 1; cfg.numAttrs = 1; }      // single CTA: no cluster launch needed
    return cudaLaunchKernelEx(&cfg, quantize_act_kernel<BPT, QMODE, Loader>, load, M, K, codes, scales, gscale, pack_mt);
}

// STATIC global scale: no tensor-wide reduction, so no cluster -- a plain grid wide enough to spread the blocks over all SMs
// (a cluster of <= 8 CTAs keeps a [8, 25600] producer on 8 SMs: 8.6 us against 3.5 us on a wide grid), any size
constexpr int QWIDE_THREADS = 128;
template <typename Loader>
static cudaError_t launch_static_wide(cudaStream_t st, Loader load, int M, int K, uint8_t* codes, uint8_t* scales, float* gscale,
                                      int pack_mt) {
    const int64_t NB = (int64_t)M * (K / 16);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)((NB + QWIDE_THREADS - 1) / QWIDE_THREADS));
    cfg.blockDim = dim3(QWIDE_THREADS);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0] = pdl_attribute();
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, quantize_act_kernel<1, QMODE_STATIC, Loader>, load, M, K, codes, scales, gscale, pack_mt);
}

// smallest cluster that covers NB blocks with <= 4 blocks per thread; prefer 1 block per thread
static bool cluster_shape(int NB, int& bpt, int& nctas, int& threads) {
    bpt = 1; nctas = 1;
    while (nctas * QTHREADS_MAX * bpt < NB) {
        if (nctas < QCLUSTER_MAX) nctas *= 2; else if (bpt < 4) bpt *= 2; else break;
    }
    if (nctas * QTHREADS_MAX * bpt < NB) return false;
    threads = (NB + nctas * bpt - 1) / (nctas * bpt);
    threads = ((threads + 31) / 32) * 32;
    if (threads > QTHREADS_MAX) threads = QTHREADS_MAX;
    return true;
}

template <typename Loader>
static cudaError_t launch_cluster_any(int bpt, int qmode, int nctas, int threads, cudaStream_t st, Loader load, int M, int K,
                                      uint8_t* codes, uint8_t* scales, float* gscale, int pack_mt) {
#define NVFP4_Q_CASE(B, Q) if (bpt == B && qmode == Q) return launch_cluster<B, Q, Loader>(nctas, threads, st, load, M, K, codes, scales, gscale, pack_mt);
    NVFP4_Q_CASE(1, QMODE_STATIC) NVFP4_Q_CASE(1, QMODE_DYNAMIC) NVFP4_Q_CASE(1, QMODE_DYNAMIC_PER_ROW)
    NVFP4_Q_CASE(2, QMODE_STATIC) NVFP4_Q_CASE(2, QMODE_DYNAMIC) NVFP4_Q_CASE(2, QMODE_DYNAMIC_PER_ROW)
    NVFP4_Q_CASE(4, QMODE_STATIC) NVFP4_Q_CASE(4, QMODE_DYNAMIC) NVFP4_Q_CASE(4, QMODE_DYNAMIC_PER_ROW)
#undef NVFP4_Q_CASE
    return cudaErrorInvalidValue;
}

static int qmode_of(int gscale_mode) {
    return gscale_mode == NVFP4_GSCALE_DYNAMIC ? QMODE_DYNAMIC
         : gscale_mode == NVFP4_GSCALE_DYNAMIC_PER_ROW ? QMODE_DYNAMIC_PER_ROW : QMODE_STATIC;
}

cudaError_t launch_quantize_act(const void* x_bf16, int M, int K, int64_t ldx, uint8_t* codes, uint8_t* scales,
                                float* gscale, int gscale_mode, cudaStream_t st, int pack_mt) {
    const uint16_t* x = static_cast<const uint16_t*>(x_bf16);
    const int NB = M * (K / 16);
    const bool dyn = (gscale_mode == NVFP4_GSCALE_DYNAMIC);
    int bpt, nctas, threads;
    if (gscale_mode == NVFP4_GSCALE_STATIC && NB > QTHREADS_MAX)
        return launch_static_wide(st, LoadX{x, ldx}, M, K, codes, scales, gscale, pack_mt);
    if (!cluster_shape(NB, bpt, nctas, threads)) {              // too large for one cluster: two kernels
        if (gscale_mode == NVFP4_GSCALE_DYNAMIC_PER_ROW) return cudaErrorInvalidConfiguration;
        if (dyn) amax_kernel<<<1, 1024, 0, st>>>(x, M, K, ldx, gscale);
        int grid = (NB + 255) / 256; if (grid > 148 * 8) grid = 148 * 8;
        quantize_blocks_kernel<<<grid, 256, 0, st>>>(x, M, K, ldx, codes, scales, gscale, pack_mt);
        return cudaGetLastError();
    }
    return launch_cluster_any(bpt, qmode_of(gscale_mode), nctas, threads, st, LoadX{x, ldx}, M, K, codes, scales, gscale, pack_mt);
}

// nvfp4_silu_mul_quantize: h = RN_bf16(silu(gate) * up), then the quantizer on h[M, I] -- one launch
cudaError_t launch_silu_mul_quantize(const void* gu_bf16, int M, int I, uint8_t* codes, uint8_t* scales, float* gscale,
                                     int gscale_mode, void* h_bf16_opt, cudaStream_t st, int pack_mt) {
    const int NB = M * (I / 16);
    int bpt, nctas, threads;
    if (gscale_mode == NVFP4_GSCALE_STATIC && NB > QTHREADS_MAX)
        return launch_static_wide(st, LoadSiluMul{static_cast<const uint16_t*>(gu_bf16), I, static_cast<uint16_t*>(h_bf16_opt)}, M, I,
                                  codes, scales, gscale, pack_mt);
    if (!cluster_shape(NB, bpt, nctas, threads)) return cudaErrorInvalidConfiguration;
    const LoadSiluMul load{static_cast<const uint16_t*>(gu_bf16), I, static_cast<uint16_t*>(h_bf16_opt)};
    return launch_cluster_any(bpt, qmode_of(gscale_mode), nctas, threads, st, load, M, I, codes, scales, gscale, pack_mt);
}

}  // namespace nvfp4
