// gemm_tc16.cu -- W4A16 on the tensor cores (BASELINE.json configs[3]): NVFP4 weights, BF16 activations
// consumed directly, FP32 accumulation:  Y[M,N] = X_bf16[M,K] . dequant(W)[N,K]^T.
//
// The CUDA-core W4A16 GEMV (gemv_kernel<KMODE_W4A16>) pays per (row m, weight): it is HBM-competitive at M <= 2 and
// 2-3x slower than cuBLAS BF16 at M = 8.  Here the per-weight work is done ONCE whatever M is:
//   * the weights stream from HBM in the tensor-core blob of gemm_tc.cu (0.5625 B per weight, one bulk copy per
//     128-row x 256-k stage),
//   * twelve "dequant" warps expand a stage to FP16: cvt.rn.f16x2.e2m1x2 (exact) times the block scale as FP16 (exact: a
//     2-bit times a 4-bit significand, |value| <= 6 * 448), and write it with tcgen05.st straight into TENSOR MEMORY as the
//     MMA's A operand (lane = weight row, two FP16 per 32-bit column along k).  A first version kept the FP16 image in
//     shared memory: every K = 16 MMA then re-read 4 KB of A from shared memory (~90 cycles per MMA, 16 per stage) and
//     the kernel ran at 0.3 of the copy ceiling.  The global weight scale stays out (epilogue),
//   * tcgen05.mma kind::f16 with A = those FP16 weights (128 rows = TMEM lanes), B = the activations (tokens = MMA N), FP32
//     accumulator in tensor memory.  The hardware rejects mixed FP16 x BF16 operands (illegal instruction, measured), and a
//     BF16 image of the weights costs twice the instructions per weight (there is no e2m1 -> bf16 conversion), so the
//     ACTIVATIONS are brought to FP16: the re-layout kernel scales each token row by a power of two, 2^-p with
//     amax_row * 2^-p in [2^14, 2^15), before the conversion.  Every BF16 value (8 significant bits) within 2^-29 of its
//     row's maximum is then an FP16 normal, i.e. converted EXACTLY; smaller elements round at 2^-24 * 2^-15 of the row
//     maximum, below the FP32 accumulator's own resolution (R23).  2^p is multiplied back in the epilogue,
//   * epilogue: y = acc * gW * 2^p[m], BF16 or FP32.
// Measured limit: with a handful of token columns the tensor core cannot reuse the A operand, and it takes A in at ~64 B per
// clock: a K = 16 FP16 MMA (4 KB of A) costs ~62 cycles whatever N is (independent accumulators do not help, A from
// shared memory costs ~88), i.e. ~1000 cycles per 128 x 256 stage against the ~830 cycles the stage's 18 KB take to arrive
// from HBM: the kernel is A-feed bound at 0.32-0.55 of the copy ceiling (gate_up 42 us), flat in M up to 32.  (The W4A4 kernel's FP4 A
// operand is four times smaller: 4 MMAs x 64 cycles per stage, which is why it stays on the HBM roofline.)
// Work split: items = (tile, K slice), one after the other per persistent CTA; with K slices the partial sums meet in the
// workspace and the last slice to arrive (per-tile counter) adds them in slice order (deterministic).
#include "nvfp4_common.cuh"
#include "nvfp4_internal.h"
#include "tc_common.cuh"

namespace nvfp4 {

constexpr int T16_DQ_WARPS  = 12;                      // dequant warps: three groups of four, group i expands the stages g = i (mod 3) into A buffer i
constexpr int T16_THREADS   = (6 + T16_DQ_WARPS) * 32; // producer, MMA issuer, 4 epilogue warps, dequant warps
constexpr int T16_ACOLS     = TC_STAGE_K / 2;          // 128 TMEM columns hold one stage of FP16 weights (2 per column)
constexpr int T16_A0        = 64;                      // first A column (after the two accumulators of <= 32 columns)
constexpr int T16_NBUF      = 3;                       // A buffers in tensor memory: 64 + 3 * 128 = 448 of the 512 columns
constexpr int T16_TMEM_COLS = 512;
constexpr int T16_MAX_MT    = 32;
constexpr int T16_MAX_CTAS  = 148;

__host__ __device__ constexpr int t16_xrec_bytes(int MT) { return MT * TC_STAGE_K * 2; }            // BF16 activations of a stage
__host__ __device__ constexpr int t16_slot_bytes(int MT) { return TC_STAGE_BYTES + t16_xrec_bytes(MT); }
__host__ __device__ constexpr int t16_dstride(int MT) { return MT < 32 ? 32 : MT; }

// instruction descriptor of kind::f16: D = F32, A = B = F16 (format 0), both K-major, D = 128 x MT, K = 16
__host__ __device__ constexpr uint32_t t16_idesc(int MT) {
    return (1u << 4) | (0u << 7) | (0u << 10) | ((uint32_t)(MT >> 3) << 17) | ((uint32_t)(TC_TILE_N >> 4) << 24);
}
// A from tensor memory, B from shared memory
__device__ __forceinline__ void tc_mma_f16_ts(uint32_t d, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n"
        "}\n" ::"r"(d), "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// this thread's TMEM lane, 16 consecutive 32-bit columns
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
                 ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]),
                   "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// ---- activations: BF16 X[M,K] (row stride ldx elements) -> FP16, per 256-k stage the MMA's B image: 8-token x 16-byte
// core matrices, chunk kc8 (8 k) of token t at (kc8*(MT/8) + t/8)*128 + (t%8)*16; tokens >= M are zero.
// One CTA per token row: pass 1 finds the row's largest magnitude, pass 2 scales by 2^-p (exact) and converts.
// rowscale[t] = 2^p (the epilogue multiplies it back).
__global__ void __launch_bounds__(256) pack_x16_kernel(const uint16_t* __restrict__ x, int64_t ldx, int M, int K, int MT,
                                                       uint8_t* __restrict__ xpack, float* __restrict__ rowscale) {
    __shared__ uint32_t wmax[8];
    pdl_wait();
    pdl_launch_dependents();
    const int t = blockIdx.x, nchunk = K / 8;
    const uint16_t* row = x + (int64_t)t * ldx;
    uint32_t mx = 0;
    if (t < M) {
        for (int c = threadIdx.x; c < nchunk; c += blockDim.x) {
            const uint4 v = *reinterpret_cast<const uint4*>(row + (size_t)c * 8);
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const uint32_t a = w[i] & 0x7FFF7FFFu;
                mx = max(mx, max(a & 0xFFFFu, a >> 16));
            }
        }
    }
    mx = __reduce_max_sync(0xFFFFFFFFu, mx);
    if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = mx;
    __syncthreads();
    mx = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) mx = max(mx, wmax[i]);
    // amax = 1.m * 2^(e-127) with e = mx >> 7: scale by 2^-(e-127-14) so that the maximum lands in [2^14, 2^15)
    int e = (int)(mx >> 7);
    if (e < 1) e = 127 + 14;                            // all-zero (or subnormal-only) row: scale 1
    if (e > 254) e = 254;                               // inf / nan rows: behaviour undefined (documented), keep the scale finite
    int up = 127 + 14 + 127 - e;                        // biased exponent of 2^-p
    float down = 1.0f;                                  // 2^-p may exceed the float range for tiny rows: apply it in two steps
    if (up > 254) { down = __uint_as_float((uint32_t)(up - 254 + 127) << 23); up = 254; }
    if (up < 1) { down = __uint_as_float((uint32_t)(up - 1 + 127) << 23); up = 1; }
    const float f1 = __uint_as_float((uint32_t)up << 23);
    if (threadIdx.x == 0 && t < MT) rowscale[t] = (t < M) ? exp2f((float)(e - 127 - 14)) : 0.0f;
    for (int c = threadIdx.x; c < nchunk; c += blockDim.x) {
        uint4 o = make_uint4(0u, 0u, 0u, 0u);
        if (t < M) {
            const uint4 v = *reinterpret_cast<const uint4*>(row + (size_t)c * 8);
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
            uint32_t r[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float lo = __uint_as_float(w[i] << 16) * f1 * down, hi = __uint_as_float(w[i] & 0xFFFF0000u) * f1 * down;
                asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r[i]) : "f"(hi), "f"(lo));
            }
            o = make_uint4(r[0], r[1], r[2], r[3]);
        }
        const int ks = c >> 5, kc8 = c & 31;            // 32 chunks of 8 k per 256-k stage
        *reinterpret_cast<uint4*>(xpack + (size_t)ks * t16_xrec_bytes(MT) + (size_t)((kc8 * (MT / 8) + (t >> 3)) * 128 + (t & 7) * 16)) = o;
    }
}

struct Gemm16Params {
    const uint8_t* blob;          // first stage record of the tensor-core blob
    const uint8_t* xpack;         // [KS] records of t16_xrec_bytes(MT)
    const float* w_gscale;
    const float* rowscale;        // [MT] 2^p per token row (pack_x16_kernel)
    void* y;
    float* partials;              // [T][ksplit][MT][128] (K slices only)
    unsigned int* counters;       // [T], zero on entry, zero on exit
    int64_t ldy;
    int N, K, M, T, KS;
    int ksplit;                   // K slices per tile; items = T * ksplit
    int stages;                   // ring depth
    int y_bf16;
    uint4 hdr_expect;
};

__device__ __forceinline__ void t16_store_y(const Gemm16Params& p, int m, int n, float v) {
    if (p.y_bf16) static_cast<uint16_t*>(p.y)[(int64_t)m * p.ldy + n] = float_to_bf16_rn(v);
    else static_cast<float*>(p.y)[(int64_t)m * p.ldy + n] = v;
}

__device__ __forceinline__ uint32_t t16_hmul2(uint32_t a, uint32_t b) {
    uint32_t d;
    asm("mul.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}
__device__ __forceinline__ uint32_t t16_prmt(uint32_t a, uint32_t b, uint32_t sel) {
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}
// eight E2M1 codes (one 32-bit word, low nibble first) times an FP16 scale pair {s, s} -> eight FP16 (exact)
__device__ __forceinline__ void t16_expand8(uint32_t w, uint32_t s2, uint32_t* out) {
    uint32_t h[4];
    cvt_word_e2m1(w, h);
#pragma unroll
    for (int i = 0; i < 4; ++i) out[i] = t16_hmul2(h[i], s2);
}
__device__ __forceinline__ void t16_epi_sync() { asm volatile("bar.sync 1, 128;" ::: "memory"); }   // the 4 epilogue warps

template <int MT>
__global__ void __launch_bounds__(T16_THREADS, 1) gemm_tc16_kernel(const Gemm16Params p) {
    extern __shared__ __align__(128) uint8_t smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int S = p.stages;
    constexpr int SLOT = t16_slot_bytes(MT), XREC = t16_xrec_bytes(MT);
    constexpr int DSTRIDE = t16_dstride(MT), NCOLS = T16_TMEM_COLS;
    uint8_t* ring = smem;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)S * SLOT);
    uint64_t *full = bars, *empty = bars + S, *afull = bars + 2 * S, *aempty = afull + T16_NBUF, *tfull = afull + 2 * T16_NBUF, *tempty = tfull + 2;
    volatile uint32_t* misc = reinterpret_cast<volatile uint32_t*>(tempty + 2);       // [0] TMEM base [1] last [2] blob ok

    const int KS = p.KS, ksplit = p.ksplit, items = p.T * ksplit;
    auto item_range = [&](int item, int& tile, int& slice, int& k0, int& k1) {
        tile = item / ksplit; slice = item - tile * ksplit;
        k0 = (int)((int64_t)slice * KS / ksplit); k1 = (int)((int64_t)(slice + 1) * KS / ksplit);
    };

    uint4 hdr = make_uint4(0u, 0u, 0u, 0u);
    if (threadIdx.x == 64) hdr = __ldg(reinterpret_cast<const uint4*>(p.blob - BLOB_HEADER_BYTES));

    // the first stages of this CTA's first item: their weights do not depend on the previous kernel
    int npre = 0;
    if ((int)blockIdx.x < items) {
        int tile, slice, k0, k1;
        item_range(blockIdx.x, tile, slice, k0, k1);
        npre = k1 - k0 < S ? k1 - k0 : S;
        if (threadIdx.x == 0) {
            for (int i = 0; i < S; ++i) { mbar_init(smem_u32(full + i), 1); mbar_init(smem_u32(empty + i), 1); }
            for (int i = 0; i < T16_NBUF; ++i) { mbar_init(smem_u32(afull + i), 4); mbar_init(smem_u32(aempty + i), 1); }
            for (int i = 0; i < 2; ++i) { mbar_init(smem_u32(tfull + i), 1); mbar_init(smem_u32(tempty + i), 4); }
            mbar_fence_init();
            for (int i = 0; i < npre; ++i) {
                mbar_arrive_expect_tx(smem_u32(full + i), (uint32_t)SLOT);
                bulk_g2s(smem_u32(ring + (size_t)i * SLOT), p.blob + ((int64_t)tile * KS + k0 + i) * TC_STAGE_BYTES, TC_STAGE_BYTES,
                         smem_u32(full + i));
            }
        }
    }
    if (warp == 1) tmem_alloc(smem_u32(const_cast<uint32_t*>(misc)), NCOLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tbase = misc[0];

    if (warp == 0) {                                          // ---- producer ----
        const bool elected = elect_one();
        pdl_wait();                                           // the activation records come from the previous kernel
        pdl_launch_dependents();
        const uint32_t ring0 = smem_u32(ring), full0 = smem_u32(full), empty0 = smem_u32(empty);
        int g = 0;                                            // stage counter of this CTA over all its items
        for (int item = blockIdx.x; item < items; item += gridDim.x) {
            int tile, slice, k0, k1;
            item_range(item, tile, slice, k0, k1);
            for (int k = k0; k < k1; ++k, ++g) {
                const int slot = g % S, use = g / S;
                const uint32_t bar = full0 + 8u * slot, dst = ring0 + (uint32_t)slot * SLOT;
                if (g < npre) {                               // weights already requested before the wait
                    if (elected) bulk_g2s(dst + TC_STAGE_BYTES, p.xpack + (size_t)k * XREC, XREC, bar);
                    continue;
                }
                mbar_wait(empty0 + 8u * slot, (uint32_t)((use - 1) & 1));
                if (elected) {
                    mbar_arrive_expect_tx(bar, (uint32_t)SLOT);
                    bulk_g2s(dst, p.blob + ((int64_t)tile * KS + k) * TC_STAGE_BYTES, TC_STAGE_BYTES, bar);
                    bulk_g2s(dst + TC_STAGE_BYTES, p.xpack + (size_t)k * XREC, XREC, bar);
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {                                   // ---- MMA issuer ----
        const bool elected = elect_one();
        constexpr uint32_t IDESC = t16_idesc(MT);
        constexpr uint32_t B_LBO = (MT / 8) * 128;
        constexpr uint32_t HI = (128u >> 4) | (1u << 14);                                 // SBO = 128 | descriptor version 1
        constexpr uint32_t B_LO = (B_LBO >> 4) << 16;                                     // LBO
        const uint32_t ring0 = smem_u32(ring);
        const uint32_t full0 = smem_u32(full), empty0 = smem_u32(empty), afull0 = smem_u32(afull), aempty0 = smem_u32(aempty);
        const uint32_t tfull0 = smem_u32(tfull), tempty0 = smem_u32(tempty);
        int g = 0, il = 0;
        for (int item = blockIdx.x; item < items; item += gridDim.x, ++il) {
            int tile, slice, k0, k1;
            item_range(item, tile, slice, k0, k1);
            const int ab = il & 1, abuse = il >> 1;
            if (abuse >= 1) mbar_wait(tempty0 + 8u * ab, (uint32_t)((abuse - 1) & 1));
            tc_fence_after();
            const uint32_t d = tbase + (uint32_t)ab * DSTRIDE;
            uint32_t acc = 0;
            for (int k = k0; k < k1; ++k, ++g) {
                const int slot = g % S, use = g / S, buf = g % T16_NBUF, bround = g / T16_NBUF;
                mbar_wait(full0 + 8u * slot, (uint32_t)(use & 1));                      // the stage's activations have landed
                mbar_wait(afull0 + 8u * buf, (uint32_t)(bround & 1));                 // its FP16 weights are in tensor memory
                tc_fence_after();
                const uint32_t xb = (ring0 + (uint32_t)slot * SLOT + TC_STAGE_BYTES) >> 4;
                const uint32_t at = tbase + T16_A0 + (uint32_t)buf * T16_ACOLS;
                if (elected) {
#pragma unroll
                    for (int j = 0; j < TC_STAGE_K / 16; ++j) {
                        tc_mma_f16_ts(d, at + 8u * j, tc_desc((xb + (uint32_t)((j * 2 * B_LBO) >> 4)) | B_LO, HI), IDESC, acc);
                        acc = 1;
                    }
                    tc_commit(aempty0 + 8u * buf);            // the dequant warps may refill this A buffer
                    tc_commit(empty0 + 8u * slot);            // and the producer the ring slot
                }
                acc = 1;
            }
            if (elected) tc_commit(tfull0 + 8u * ab);
        }
        __syncwarp();
    } else if (warp >= 6) {                                   // ---- dequant warps ----
        // a warp can only reach the 32 TMEM lanes of its quarter (warp % 4): it expands those 32 weight rows, all 256 k of a
        // stage.  Three groups of four warps take the stages round-robin, group i always into A buffer i: a warp works
        // through its stages one after the other (wait, load, convert, tcgen05.st, wait::st, arrive), so several stages must
        // be in expansion at any time; three A buffers are what fits into tensor memory.  (One group per buffer also keeps
        // every mbarrier wait within one phase of the barrier: a group that could run two buffer generations ahead of the
        // MMAs would see the parity of an older phase and pass -- measured as an intermittent deadlock.)
        const int dw = warp - 6, grp = dw >> 2, rg = warp & 3, r = rg * 32 + lane;
        constexpr int NGRP = T16_DQ_WARPS / 4;
        static_assert(NGRP == T16_NBUF, "one dequant group per A buffer");
        const uint32_t full0 = smem_u32(full), afull0 = smem_u32(afull), aempty0 = smem_u32(aempty);
        const uint32_t tlane = tbase + ((uint32_t)(rg * 32) << 16) + T16_A0;
        int g = 0;
        for (int item = blockIdx.x; item < items; item += gridDim.x) {
            int tile, slice, k0, k1;
            item_range(item, tile, slice, k0, k1);
            for (int k = k0; k < k1; ++k, ++g) {
                if (g % NGRP != grp) continue;
                const int slot = g % S, use = g / S, buf = g % T16_NBUF, bround = g / T16_NBUF;
                mbar_wait(full0 + 8u * slot, (uint32_t)(use & 1));
                const uint8_t* st = ring + (size_t)slot * SLOT;
#pragma unroll
                for (int b4 = 0; b4 < 2; ++b4) {              // the quarter's eight 32-k chunks in two batches of four
                    uint4 cw[4];
                    uint16_t sc2[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) {             // all loads first: the expansion is latency bound
                        const int kc = b4 * 4 + i;
                        cw[i] = *reinterpret_cast<const uint4*>(st + (size_t)((kc * 16 + (r >> 3)) * 128 + (r & 7) * 16));
                        sc2[i] = *reinterpret_cast<const uint16_t*>(st + TC_CODE_BYTES + (kc >> 1) * 512 + (r & 31) * 16 + (r >> 5) * 4 + (kc & 1) * 2);
                    }
                    if (b4 == 0) {
                        if (bround >= 1) mbar_wait(aempty0 + 8u * buf, (uint32_t)((bround - 1) & 1));   // the MMAs that read this buffer are done
                        tc_fence_after();
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        uint32_t s2;
                        asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(s2) : "h"(sc2[i]));
                        const uint32_t sA = t16_prmt(s2, s2, 0x1010u), sB = t16_prmt(s2, s2, 0x3232u);
                        uint32_t v[16];
                        t16_expand8(cw[i].x, sA, v); t16_expand8(cw[i].y, sA, v + 4);
                        t16_expand8(cw[i].z, sB, v + 8); t16_expand8(cw[i].w, sB, v + 12);
                        tmem_st16(tlane + (uint32_t)buf * T16_ACOLS + (uint32_t)(b4 * 4 + i) * 16, v);
                    }
                }
                tmem_st_wait();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive_plain(afull0 + 8u * buf);
            }
        }
    } else {                                                  // ---- epilogue (warps 2..5) ----
        const int q = warp & 3, r = q * 32 + lane;
        pdl_wait();
        if (threadIdx.x == 64)
            misc[2] = (hdr.x == p.hdr_expect.x) && (hdr.y == p.hdr_expect.y) && (hdr.z == p.hdr_expect.z) && (hdr.w == p.hdr_expect.w);
        t16_epi_sync();
        const bool blob_ok = misc[2] != 0;
        const float gw = __ldg(p.w_gscale);
        const float nanv = __uint_as_float(0x7FC00000u);
        int il = 0;
        for (int item = blockIdx.x; item < items; item += gridDim.x, ++il) {
            int tile, slice, k0, k1;
            item_range(item, tile, slice, k0, k1);
            const int ab = il & 1, abuse = il >> 1;
            mbar_wait(smem_u32(tfull + ab), (uint32_t)(abuse & 1));
            tc_fence_after();
            const uint32_t taddr = tbase + ((uint32_t)(q * 32) << 16) + (uint32_t)ab * DSTRIDE;
            const int n = tile * TC_TILE_N + r;
            float* part = p.partials + ((size_t)(tile * ksplit + slice) * MT) * TC_TILE_N;
#pragma unroll 1
            for (int c8 = 0; c8 < MT; c8 += 8) {
                if (c8 >= p.M) break;
                uint32_t v[8];
                tmem_ld8(taddr + c8, v);
                tmem_ld_wait();
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int m = c8 + j;
                    if (m >= p.M) continue;
                    if (ksplit == 1) { if (n < p.N) t16_store_y(p, m, n, blob_ok ? __uint_as_float(v[j]) * (gw * __ldg(p.rowscale + m)) : nanv); }
                    else part[(size_t)m * TC_TILE_N + r] = __uint_as_float(v[j]);
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_plain(smem_u32(tempty + ab));
            if (ksplit > 1) {                                 // the last slice to arrive adds the partials in slice order
                t16_epi_sync();
                if (threadIdx.x == 64) {
                    unsigned int old;
                    asm volatile("atom.add.acq_rel.gpu.global.u32 %0, [%1], 1;" : "=r"(old) : "l"(p.counters + tile) : "memory");
                    const bool last = old == (unsigned int)(ksplit - 1);
                    if (last) p.counters[tile] = 0u;
                    misc[1] = last ? 1u : 0u;
                }
                t16_epi_sync();
                if (misc[1]) {
                    const float* base = p.partials + ((size_t)tile * ksplit * MT) * TC_TILE_N + r;
                    for (int m0 = 0; m0 < p.M; m0 += 8) {
                        float a[8];
#pragma unroll
                        for (int j = 0; j < 8; ++j) a[j] = 0.0f;
                        for (int c = 0; c < ksplit; ++c)
#pragma unroll
                            for (int j = 0; j < 8; ++j)
                                if (m0 + j < p.M) a[j] += __ldcg(base + ((size_t)c * MT + m0 + j) * TC_TILE_N);
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            if (m0 + j < p.M && n < p.N) t16_store_y(p, m0 + j, n, blob_ok ? a[j] * (gw * __ldg(p.rowscale + m0 + j)) : nanv);
                    }
                }
                t16_epi_sync();                               // misc[1] is reused by the next item
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc(tbase, NCOLS);
}

// ---- host side ----------------------------------------------------------------------------------------------------
// kind::f16 with 128 accumulator rows needs N % 16 == 0 (N = 8 traps as an illegal instruction): 16 token columns at least
static int t16_pick_mt(int m) { return m <= 16 ? 16 : 32; }
static int t16_pick_stages(int MT) {
    const int s = (227 * 1024 - 512) / t16_slot_bytes(MT);
    return s > 8 ? 8 : s;
}
// K slices per tile and persistent CTAs: as for the W4A4 tensor-core kernel (tc_pick_ctas), items are whole K slices of
// one tile; T <= 148: floor(148/T) slices per tile, T > 148: whole tiles on the largest divisor of T in [74, 148]
static void t16_pick_split(int T, int KS, int& ksplit, int& grid) {
    if (T <= T16_MAX_CTAS) {
        ksplit = T16_MAX_CTAS / T;
        if (ksplit > KS) ksplit = KS;
        if (ksplit > 8) ksplit = 8;
        grid = T * ksplit;
        return;
    }
    ksplit = 1;
    grid = T16_MAX_CTAS;
    for (int g = T16_MAX_CTAS; g >= T16_MAX_CTAS / 2; --g)
        if (T % g == 0) { grid = g; break; }
}
static size_t t16_align(size_t v) { return (v + 255) & ~(size_t)255; }
static size_t t16_counters_bytes(int N) { return t16_align((size_t)tc_tiles(N) * sizeof(unsigned int)); }
static size_t t16_xpack_bytes(int K, int MT) { return t16_align((size_t)(K / TC_STAGE_K) * t16_xrec_bytes(MT)) + 256; }   // + [MT] row scales
static size_t t16_partials_bytes(int N, int K, int MT) {
    int ksplit, grid;
    t16_pick_split(tc_tiles(N), K / TC_STAGE_K, ksplit, grid);
    return ksplit > 1 ? (size_t)tc_tiles(N) * ksplit * MT * TC_TILE_N * sizeof(float) : 0;
}

size_t gemm_tc16_workspace_bytes(int M, int N, int K) {
    const int MT = t16_pick_mt(M > T16_MAX_MT ? T16_MAX_MT : M);
    return t16_counters_bytes(N) + t16_xpack_bytes(K, MT) + t16_partials_bytes(N, K, MT);
}

template <int MT>
static cudaError_t launch_gemm_tc16_mt(const Gemm16Params& p, int grid, cudaStream_t st) {
    static size_t configured[MAX_DEVICES] = {};
    const size_t smem = (size_t)p.stages * t16_slot_bytes(MT) + (size_t)(2 * p.stages + 2 * T16_NBUF + 4) * 8 + 32;
    cudaError_t e = ensure_dynamic_smem(gemm_tc16_kernel<MT>, configured, smem);
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(T16_THREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr = pdl_attribute();
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, gemm_tc16_kernel<MT>, p);
}

cudaError_t launch_gemm_tc16(const void* blob, const float* w_gscale, int N, int K, const void* x_bf16, int64_t ldx, int M,
                             void* y, int y_dtype, int64_t ldy, void* workspace, size_t ws_bytes, cudaStream_t st) {
    if (ws_bytes < gemm_tc16_workspace_bytes(M, N, K)) return cudaErrorInvalidValue;
    const int T = tc_tiles(N), KS = K / TC_STAGE_K;
    uint8_t* ws = static_cast<uint8_t*>(workspace);
    const int MTmax = t16_pick_mt(M > T16_MAX_MT ? T16_MAX_MT : M);
    uint8_t* xpack = ws + t16_counters_bytes(N);
    float* partials = reinterpret_cast<float*>(xpack + t16_xpack_bytes(K, MTmax));
    const size_t esz = (y_dtype == NVFP4_DTYPE_BF16) ? 2 : 4;
    for (int m0 = 0; m0 < M; m0 += T16_MAX_MT) {
        const int mc = M - m0 < T16_MAX_MT ? M - m0 : T16_MAX_MT;
        const int MT = t16_pick_mt(mc);
        float* rowscale = reinterpret_cast<float*>(xpack + t16_xpack_bytes(K, MTmax) - 256);
        {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3((unsigned)MT);           // one CTA per token row (rows >= mc are zero-filled)
            cfg.blockDim = dim3(256);
            cfg.stream = st;
            cudaLaunchAttribute attr = pdl_attribute();
            cfg.attrs = &attr;
            cfg.numAttrs = 1;
            cudaError_t e = cudaLaunchKernelEx(&cfg, pack_x16_kernel, static_cast<const uint16_t*>(x_bf16) + (size_t)m0 * ldx, ldx, mc, K,
                                               MT, xpack, rowscale);
            if (e != cudaSuccess) return e;
        }
        Gemm16Params p = {};
        p.blob = static_cast<const uint8_t*>(blob) + BLOB_HEADER_BYTES;
        p.xpack = xpack;
        p.w_gscale = w_gscale;
        p.rowscale = rowscale;
        p.y = static_cast<uint8_t*>(y) + (size_t)m0 * ldy * esz;
        p.partials = partials;
        p.counters = reinterpret_cast<unsigned int*>(ws);
        p.ldy = ldy;
        p.N = N; p.K = K; p.M = mc; p.T = T; p.KS = KS;
        int grid;
        t16_pick_split(T, KS, p.ksplit, grid);
        p.stages = t16_pick_stages(MT);
        p.y_bf16 = (y_dtype == NVFP4_DTYPE_BF16);
        p.hdr_expect = tc_header_words(N, K);
        cudaError_t e;
        if (MT == 16) e = launch_gemm_tc16_mt<16>(p, grid, st);
        else e = launch_gemm_tc16_mt<32>(p, grid, st);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace nvfp4
