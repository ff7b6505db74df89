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

// One cluster (gridDim.x CTAs == cluster size) covers the whole tensor; BPT blocks per thread.
template <int BPT, bool DYNAMIC>
__global__ void __launch_bounds__(QTHREADS_MAX)
quantize_act_kernel(const uint16_t* __restrict__ x, int M, int K, int64_t ldx,
                    uint8_t* __restrict__ codes, uint8_t* __restrict__ scales, float* __restrict__ gscale) {
    __shared__ uint32_t warp_max[32];
    __shared__ uint32_t cta_max[QCLUSTER_MAX];
    const int kb_per_row = K >> 4;
    const int NB = M * kb_per_row;
    const int nthreads = gridDim.x * blockDim.x;
    const int gtid = blockIdx.x * blockDim.x + threadIdx.x;
    pdl_wait();                                       // X is the previous kernel's output
    pdl_launch_dependents();                          // the GEMV may start streaming its weights now

    uint4 va[BPT], vb[BPT];
    uint32_t ab[BPT];
    uint32_t tmax = 0;
#pragma unroll
    for (int i = 0; i < BPT; ++i) {
        const int b = gtid + i * nthreads;
        va[i] = vb[i] = make_uint4(0, 0, 0, 0);
        ab[i] = 0;
        if (b < NB) {
            const int m = b / kb_per_row, kb = b - m * kb_per_row;
            const uint4* p = reinterpret_cast<const uint4*>(x + (int64_t)m * ldx + (int64_t)kb * 16);
            va[i] = __ldg(p);
            vb[i] = __ldg(p + 1);
            ab[i] = absmax_bits16(va[i], vb[i]);
            tmax = max(tmax, ab[i]);
        }
    }

    float g;
    if (DYNAMIC) {
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
            cg::cluster_group cluster = cg::this_cluster();
            const unsigned rank = cluster.block_rank();
            if (threadIdx.x < gridDim.x)                         // push my max into every CTA's slot[rank]
                cluster.map_shared_rank(cta_max, threadIdx.x)[rank] = amax_bits;
            cluster.sync();
            amax_bits = 0;
            for (unsigned r = 0; r < gridDim.x; ++r) amax_bits = max(amax_bits, cta_max[r]);
        }
        g = __fdiv_rn(__uint_as_float(amax_bits << 16), 2688.0f);
        if (gtid == 0) *gscale = g;
    } else {
        g = __ldg(gscale);
    }

#pragma unroll
    for (int i = 0; i < BPT; ++i) {
        const int b = gtid + i * nthreads;
        if (b < NB) {
            uint2 c; uint8_t s;
            quantize_block(va[i], vb[i], ab[i], g, c, s);
            *reinterpret_cast<uint2*>(codes + (int64_t)b * 8) = c;   // [M,K/2] contiguous: block b -> 8 bytes
            scales[b] = s;
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
                                                              const float* __restrict__ gscale) {
    const int kb_per_row = K >> 4;
    const int NB = M * kb_per_row;
    const float g = *gscale;
    for (int b = blockIdx.x * blockDim.x + threadIdx.x; b < NB; b += gridDim.x * blockDim.x) {
        const int m = b / kb_per_row, kb = b - m * kb_per_row;
        const uint4* p = reinterpret_cast<const uint4*>(x + (int64_t)m * ldx + (int64_t)kb * 16);
        const uint4 a = __ldg(p), bb = __ldg(p + 1);
        uint2 c; uint8_t s;
        quantize_block(a, bb, absmax_bits16(a, bb), g, c, s);
        *reinterpret_cast<uint2*>(codes + (int64_t)b * 8) = c;
        scales[b] = s;
    }
}

template <int BPT, bool DYN>
static cudaError_t launch_cluster(int nctas, int threads, cudaStream_t st, const uint16_t* x, int M, int K,
                                  int64_t ldx, uint8_t* codes, uint8_t* scales, float* gscale) {
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
    return cudaLaunchKernelEx(&cfg, quantize_act_kernel<BPT, DYN>, x, M, K, ldx, codes, scales, gscale);
}

cudaError_t launch_quantize_act(const void* x_bf16, int M, int K, int64_t ldx, uint8_t* codes, uint8_t* scales,
                                float* gscale, int gscale_mode, cudaStream_t st) {
    const uint16_t* x = static_cast<const uint16_t*>(x_bf16);
    const int NB = M * (K / 16);
    const bool dyn = (gscale_mode == NVFP4_GSCALE_DYNAMIC);
    // smallest cluster that covers NB with <= 4 blocks per thread; prefer 1 block per thread
    int bpt = 1, nctas = 1;
    while (nctas * QTHREADS_MAX * bpt < NB) {
        if (nctas < QCLUSTER_MAX) nctas *= 2; else if (bpt < 4) bpt *= 2; else break;
    }
    if (nctas * QTHREADS_MAX * bpt < NB) {                      // too large for one cluster: two kernels
        if (dyn) amax_kernel<<<1, 1024, 0, st>>>(x, M, K, ldx, gscale);
        int grid = (NB + 255) / 256; if (grid > 148 * 8) grid = 148 * 8;
        quantize_blocks_kernel<<<grid, 256, 0, st>>>(x, M, K, ldx, codes, scales, gscale);
        return cudaGetLastError();
    }
    int threads = (NB + nctas * bpt - 1) / (nctas * bpt);
    threads = ((threads + 31) / 32) * 32;
    if (threads > QTHREADS_MAX) threads = QTHREADS_MAX;
#define NVFP4_Q_CASE(B)                                                                                   \
    case B: return dyn ? launch_cluster<B, true>(nctas, threads, st, x, M, K, ldx, codes, scales, gscale) \
                       : launch_cluster<B, false>(nctas, threads, st, x, M, K, ldx, codes, scales, gscale);
    switch (bpt) {
        NVFP4_Q_CASE(1)
        NVFP4_Q_CASE(2)
        NVFP4_Q_CASE(4)
    }
#undef NVFP4_Q_CASE
    return cudaErrorInvalidValue;
}

}  // namespace nvfp4
