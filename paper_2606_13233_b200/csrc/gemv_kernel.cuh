// gemv_kernel.cuh -- the weight-streaming NVFP4 GEMV / skinny GEMM (steps a3..a7),
//   Y[m,n] = sum_k vX[m,k] * vW[n,k]     (CUDA cores only)
//
// Design (differs from the paper's FP16 cvt+hfma2 kernel):
//  * lane <-> (weight row, K part): lane = p*(32/KP) + r.  The KP lanes of a row take interleaved 32-k
//    vectors and are summed by log2(KP) warp shuffles once per segment.  KP is a property of the
//    repacked layout (nvfp4_common.cuh).
//  * BALANCE (data-parallel + stream-K): unit = R row tiles x all cells of the K slice (cell = 256*KP k,
//    4608 B).  Every CTA (about one per SM) owns `base` = units / CTAs whole units (phase B) plus an EQUAL
//    share of the flat cell stream of the leftover units (phase A), so every SM streams the same number of
//    bytes whatever N and K are.  Phase A comes FIRST and its cells are dealt round-robin to the consumer
//    warps (one cell each, typically), so the leftover units are finished within the first microseconds:
//    their FP32 partials go through the workspace and the last CTA to arrive sums them in a fixed order
//    (deterministic) -- on the otherwise idle stager warps, in the shadow of phase B.  Phase B is a
//    contiguous run per warp; a unit cut between warps is recombined through shared-memory slots by the
//    last warp to arrive, in fixed warp order.  With one K slice no CTA waits on another one at the end.
//  * the activations of the CTA's K slice are decoded ONCE per CTA into shared memory by dedicated
//    stager warps; lanes read them with LDS.128 (KP distinct addresses per instruction, conflict free).
//  * each warp has a PRIVATE ring of S stages filled by 1-D bulk copies (cp.async.bulk ->
//    UBLKCP, completion on an mbarrier); lane 0 refills a stage as soon as the warp has read
//    it.  HBM bytes in flight do not depend on registers or on how fast the math runs.
//  * W4A4 math is integer and exact inside a 16-block: PRMT byte-LUTs turn 4 nibbles into
//    4 bytes u = 12 + 2*e (two PRMT, one per sign, OR-ed), dp4a against int8 x = 2*e_x with the
//    accumulator pre-loaded with a magic bias - 12*sum(x); packed FP32 ops apply sW*sX per block pair.
//    Cross-block accumulation is FP32 (R8).  M = 1 uses cvt.rn.f16x2.e2m1x2 + HFMA2 instead.
//  * W4A16: cvt.rn.f16x2.e2m1x2 -> FP32, packed FP32 FMA against FP32 copies of the BF16 activations.
//  * K slices (grid.y > 1) are used only when the M*K activation records do not fit in shared memory.
#pragma once
#include "nvfp4_common.cuh"
#include "nvfp4_internal.h"
#include "quant_block.cuh"

namespace nvfp4 {

struct GemvParams {
    const uint8_t* blob;      // first cell (the 128-byte header precedes it)
    const float* w_gscale;
    const void* x;            // W4A4: codes (uint8, row stride ldx bytes); W4A16 / fused: BF16 bits (row stride ldx elements)
    const uint8_t* x_scales;  // W4A4: [M, K/16]
    const float* x_gscale;    // W4A4: one float, or M floats (gscale_per_row)
    void* y;
    float* partials_a;        // [ksplit][jmax][M][npad_a]: leftover units (phase A), one slot per contributing CTA
    float* partials_b;        // [ksplit][M][npad_b]: whole units (phase B), used with K slices only
    unsigned int* counters;   // [units], zero on entry, zero on exit
    int64_t ldx, ldy;
    int N, K, ntiles, nch;         // tiles of 32/kp rows, cells of 256*kp k
    int npad_a, npad_b;            // padded row counts of the leftover / whole units
    int kp, kp_shift;              // K parts per row inside a warp (power of two) and its log2
    int warps, stages, ksplit;
    int units;                     // ceil(ntiles / R): a unit = R adjacent row tiles
    int cells_q, cells_r;          // nch / ksplit and nch % ksplit   (K slice `by` has q + (by < r) cells per unit)
    // work split: every CTA of a slice owns `base` whole units (phase B) and an equal
    // share of the flat cell stream of the `ur` = units - base*gridDim.x leftover units (phase A).  Slice
    // variant v (0: cells_q cells per unit, 1: cells_q + 1): nba[v] = min(gridDim.x, ur*ncw_v) CTAs take part
    // in phase A; CTA b < nba owns leftover cells [b*a_q[v] + (b*a_r[v])/nba[v], same for b + 1).
    int base, ur;
    int whole_units;               // 1: no leftover stream; the first `ur` CTAs own base + 1 whole units instead
    int nba[2], a_q[2], a_r[2];
    FastDiv fd_w, fd_ncw[2], fd_nba[2];   // divisors: consumer warps, cells per unit (per variant), phase-A CTAs (per variant)
    float inv_a[2];                // nba / (ur*ncw_v): estimate for the inverse of the share start
    int amax;                      // max leftover cells per CTA
    int jmax;                      // max number of CTAs of one slice that share a leftover unit
    int nxb;                       // staging-batch mbarriers
    int nhand;                     // hand-off slots: 2 leftover units (+ base whole units with K slices)
    int y_bf16;
    int zero;                      // always 0 (see make_wlut)
    int fuse_quant;                // x is BF16 [M,K] (ldx elements): quantise it inside the kernel (W4A4 modes)
    int gscale_per_row;            // x_gscale holds M per-row (per-token) global scales
    float* x_gscale_out;           // fuse_quant: optional device float that receives the activation global scale
    const uint8_t* x_records;      // W4A4, M = 1 (FP16 path): activations already in this kernel's shared-memory record layout
                                   // for the whole padded K (nvfp4_quantize_act_records); each CTA takes its K range with ONE
                                   // bulk copy instead of loading, decoding and storing it (NULL: x / x_scales are used)
    uint4 hdr_expect;              // blob_header_words(N, K, kp)
    uint32_t smem_map[13];         // gemv_smem_map(...) computed by the host (same order as struct SmemMap)
    unsigned long long* trace;     // debug only (nvfp4_debug_set_trace): 16 timestamps per CTA, else NULL
};

// shared-memory bytes of activations per 32-k block pair and per m
constexpr int XBP_W4A4  = 48;    // 32 int8 + {init0, init1, sX0, sX1}
constexpr int XBP_W4A16 = 128;   // 32 floats
constexpr int XBP_W4A4H = 80;    // 32 f16 (e2m1 values, exact) + {sX0, sX1} + pad

// kernel arithmetic variants (template parameter MODE of gemv_kernel)
constexpr int KMODE_W4A4_I8 = 0;   // integer: PRMT LUT decode + dp4a          (best for M >= 2)
constexpr int KMODE_W4A16   = 1;   // FP32 FMA against BF16 activations
constexpr int KMODE_W4A4_H  = 2;   // cvt.rn.f16x2.e2m1x2 + HFMA2, exact per 8 k (best for M = 1)
// Bytes between the records of consecutive 32-k vectors (all M rows of a vector are adjacent).  The
// lanes of a quarter warp read the records of 8 consecutive vectors (their K parts) with one
// LDS.128, so the stride must be an ODD multiple of 16 B to spread them over all 32 banks: pad by
// 16 B when M*XBP/16 is even (otherwise e.g. M = 8 gives an 8-way bank conflict on every load).
__host__ __device__ constexpr int xvec_stride(int kmode, int M);
__host__ __device__ constexpr int xbp_bytes(int kmode) {
    return kmode == KMODE_W4A4_I8 ? XBP_W4A4 : (kmode == KMODE_W4A16 ? XBP_W4A16 : XBP_W4A4H);
}
__host__ __device__ constexpr int xvec_stride(int kmode, int M) {
    return M * xbp_bytes(kmode) + (((M * xbp_bytes(kmode) / 16) % 2 == 0) ? 16 : 0);
}
static_assert(xvec_stride(KMODE_W4A4_H, 1) == GEMV_XRECORD_BYTES, "nvfp4_quantize_act_records writes this layout");

__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
    uint32_t d;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
    return d;
}
__device__ __forceinline__ int dp4a_us(uint32_t a_unsigned, uint32_t b_signed, int c) {
    int d;
    asm("dp4a.u32.s32 %0, %1, %2, %3;" : "=r"(d) : "r"(a_unsigned), "r"(b_signed), "r"(c));
    return d;
}

// byte LUTs of u = 12 + 2*e2m1: positive codes (index = low 3 bits) and negative codes.  PRMT
// with selector bit 3 set replicates the MSB (0) of the selected byte, i.e. yields 0x00, so the
// "wrong sign" half of each lookup vanishes and the two lookups can be OR-ed.
struct WLut { uint32_t p_lo, p_hi, n_lo, n_hi; };
__device__ __forceinline__ WLut make_wlut(uint32_t zero) {
    // The constants are OR-ed with a per-thread value the compiler cannot prove to be 0, so it treats
    // them as ordinary per-thread registers: otherwise it keeps them in UNIFORM registers and
    // copies them back with one IMAD.U32 per PRMT (54 extra instructions per 128 weights).
    WLut l;
    const uint32_t z = threadIdx.x * zero;     // zero is a kernel parameter that is always 0
    asm volatile("or.b32 %0, %4, 0x0F0E0D0C; or.b32 %1, %4, 0x18141210; or.b32 %2, %4, 0x090A0B0C; or.b32 %3, %4, 0x00040608;"
                 : "=r"(l.p_lo), "=r"(l.p_hi), "=r"(l.n_lo), "=r"(l.n_hi) : "r"(z));
    return l;
}
// 8 nibbles (one word, low nibble = lowest k) -> two words of bytes u = 12 + 2*e2m1(code)
__device__ __forceinline__ void decode_w_u8(const WLut& l, uint32_t w, uint32_t& u_lo, uint32_t& u_hi) {
    const uint32_t t = w ^ 0x88888888u;
    u_lo = prmt(l.p_lo, l.p_hi, w) | prmt(l.n_lo, l.n_hi, t);
    u_hi = prmt(l.p_lo, l.p_hi, w >> 16) | prmt(l.n_lo, l.n_hi, t >> 16);
}

// ---- activation staging: decode the CTA's K range once into shared memory ----------------
// Done by ALL threads of the CTA right after the consumer warps have requested their first weight cells (the
// L2 round trip of the activation loads hides under the HBM latency of those cells); readiness is signalled
// per batch through mbarriers.  Loads are issued STAGE_BATCH at a time per thread, so the L2 latency is paid
// once per batch.  STAGER_WARPS extra warps take part in the staging and afterwards complete the row tiles
// the CTA shares with other CTAs (closer role).
constexpr int STAGE_BATCH = 4;
constexpr int STAGER_WARPS = 4;
constexpr int STAGER_THREADS = STAGER_WARPS * 32;

// one mbarrier per staging batch (blockDim.x * STAGE_BATCH work items): every thread arrives on it
// after its stores (release), a consumer waits (acquire) on the batch that contains the last item it
// needs -- no polling loop, no CTA-wide barrier.
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

constexpr uint32_t I8_MAGIC_BITS = 0x4B400000u;   // 1.5 * 2^23 = 12582912.0f: ulp 1, integers n with |n| < 2^22 add exactly
constexpr float    I8_MAGIC      = 12582912.0f;
__device__ __forceinline__ void decode_x_block(uint2 cw, float sx, uint8_t* base, int half) {
    // nibble -> signed int8 x = 2*e2m1: magnitude LUT through PRMT once per sign, per-byte subtract
    uint32_t out[4];
    int sum = 0;
#pragma unroll
    for (int wi = 0; wi < 2; ++wi) {
        const uint32_t w = wi ? cw.y : cw.x;
        const uint32_t t = w ^ 0x88888888u;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const uint32_t pos = prmt(0x03020100u, 0x0C080604u, w >> (16 * h));   // negative codes -> 0
            const uint32_t neg = prmt(0x03020100u, 0x0C080604u, t >> (16 * h));   // positive codes -> 0
            out[wi * 2 + h] = __vsub4(pos, neg);
            sum += (int)__dp4a(pos, 0x01010101u, 0u) - (int)__dp4a(neg, 0x01010101u, 0u);
        }
    }
    *reinterpret_cast<uint4*>(base + half * 16) = make_uint4(out[0], out[1], out[2], out[3]);
    // the dp4a accumulator starts at MAGIC - 12*sum(x): the finished integer dot, read as FP32 bits, IS the float
    // 12582912 + dot (exact, |dot| <= 2304), so one packed FADD replaces two I2F (block_pair_w4a4)
    *reinterpret_cast<int*>(base + 32 + half * 4) = (int)I8_MAGIC_BITS - 12 * sum;
    *reinterpret_cast<float*>(base + 40 + half * 4) = sx;
}

// tid = index among the stager threads.  Work item i -> (block = i / M, m = i % M): progress is
// monotone in the block index, which is what consumers wait on.
// FP16 variant of the record: 16 e2m1 values as f16 (8 x F2FP), the block scale as FP32
__device__ __forceinline__ void decode_x_block_h(uint2 cw, float sx, uint8_t* base, int half) {
    uint32_t h[8];
    {
        uint32_t a[4], b[4];
        cvt_word_e2m1(cw.x, a);
        cvt_word_e2m1(cw.y, b);
#pragma unroll
        for (int i = 0; i < 4; ++i) { h[i] = a[i]; h[4 + i] = b[i]; }
    }
    uint4* dst = reinterpret_cast<uint4*>(base + half * 32);
    dst[0] = make_uint4(h[0], h[1], h[2], h[3]);
    dst[1] = make_uint4(h[4], h[5], h[6], h[7]);
    *reinterpret_cast<float*>(base + 64 + half * 4) = sx;
}

// `between` runs once, right after the first batch's loads have been issued (their L2 latency hides it)
template <int M, bool HALF, typename Between>
__device__ __forceinline__ void stage_x_w4a4(const GemvParams& p, uint8_t* xs, int c0, int ncw, int tid, int nthr,
                                             uint64_t* xbars, Between&& between) {
    const int nblk = ncw * 2 * CELL_VECS * p.kp;                 // 16-blocks in the range
    const int kb_total = p.K >> 4;
    const int kb0 = c0 * 2 * CELL_VECS * p.kp;
    const uint8_t* xc = static_cast<const uint8_t*>(p.x);
    const int total = nblk * M;
    for (int base = 0, batch = 0; base < total; base += nthr * STAGE_BATCH, ++batch) {
        uint2 cw[STAGE_BATCH];
        uint32_t sb[STAGE_BATCH];
#pragma unroll
        for (int t = 0; t < STAGE_BATCH; ++t) {
            const int i = base + t * nthr + tid;
            const int blk = i / M, m = i - blk * M;
            cw[t] = make_uint2(0u, 0u);
            sb[t] = 0;
            if (i < total && kb0 + blk < kb_total) {
                cw[t] = __ldg(reinterpret_cast<const uint2*>(xc + (int64_t)m * p.ldx + (int64_t)(kb0 + blk) * 8));
                sb[t] = __ldg(p.x_scales + (int64_t)m * kb_total + kb0 + blk);
            }
        }
        if (batch == 0) between();
#pragma unroll
        for (int t = 0; t < STAGE_BATCH; ++t) {
            const int i = base + t * nthr + tid;
            if (i < total) {
                const int blk = i / M, m = i - blk * M;
                if (HALF) decode_x_block_h(cw[t], e4m3_to_float((uint8_t)sb[t]), xs + (size_t)(blk >> 1) * xvec_stride(KMODE_W4A4_H, M) + m * XBP_W4A4H, blk & 1);
                else      decode_x_block(cw[t], e4m3_to_float((uint8_t)sb[t]), xs + (size_t)(blk >> 1) * xvec_stride(KMODE_W4A4_I8, M) + m * XBP_W4A4, blk & 1);
            }
        }
        mbar_arrive(smem_u32(xbars + batch));
    }
}

// Fused quantization (nvfp4_gemv_fused_quant): ALL threads of the CTA run the activation quantizer themselves --
// pass 1: tensor-wide amax of the BF16 activations (whole [M,K], every CTA redundantly: <= 410 KB from L2),
// pass 2: per 16-block the R2 sequence of quant_block.cuh, then straight to the f16 record (the E2M1 code is
// produced by cvt.rn.satfinite.e2m1x2.f32 and expanded by cvt.rn.f16x2.e2m1x2, so the values are exactly
// those of quantize_act followed by the normal staging).  `red` = one word per warp of the CTA (32 reserved in the shared-memory map).
template <int M, bool HALF>
__device__ __forceinline__ void stage_x_fused(const GemvParams& p, uint8_t* xs, int c0, int ncw, int tid, int nthr,
                                                uint64_t* xbars, uint32_t* red, float* gx_slot) {
    // called by EVERY thread of the CTA (consumer warps right after they have started their weight stream)
    const uint16_t* xb = static_cast<const uint16_t*>(p.x);
    const int kb_total = p.K >> 4;
    uint32_t tmax = 0;
    for (int i = tid; i < kb_total * M; i += nthr) {
        const int m = i / kb_total, kb = i - m * kb_total;
        const uint4* src = reinterpret_cast<const uint4*>(xb + (int64_t)m * p.ldx + (int64_t)kb * 16);
        tmax = max(tmax, absmax_bits16(__ldg(src), __ldg(src + 1)));
    }
    tmax = __reduce_max_sync(0xFFFFFFFFu, tmax);
    if ((tid & 31) == 0) red[tid >> 5] = tmax;
    asm volatile("bar.sync 1, %0;" ::"r"(nthr) : "memory");
    uint32_t amax_bits = 0;
    for (int w = 0; w < (nthr >> 5); ++w) amax_bits = max(amax_bits, red[w]);
    const float g = __fdiv_rn(__uint_as_float(amax_bits << 16), 2688.0f);
    if (tid == 0) {
        *gx_slot = g;
        if (p.x_gscale_out != nullptr && blockIdx.x == 0 && blockIdx.y == 0) *p.x_gscale_out = g;
    }
    const int nblk = ncw * 2 * CELL_VECS * p.kp;
    const int kb0 = c0 * 2 * CELL_VECS * p.kp;
    const int total = nblk * M;
    for (int base = 0, batch = 0; base < total; base += nthr, ++batch) {     // one block per thread and batch
        const int i = base + tid;
        if (i < total) {
            const int blk = i / M, m = i - blk * M;
            constexpr int KM = HALF ? KMODE_W4A4_H : KMODE_W4A4_I8;
            uint8_t* rec = xs + (size_t)(blk >> 1) * xvec_stride(KM, M) + m * xbp_bytes(KM);
            uint32_t h[8] = {0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};        // HALF: f16 pairs; else: one code byte each
            float sx = 0.0f;
            if (kb0 + blk < kb_total && g > 0.0f) {
                const uint4* src = reinterpret_cast<const uint4*>(xb + (int64_t)m * p.ldx + (int64_t)(kb0 + blk) * 16);
                const uint4 a = __ldg(src), b = __ldg(src + 1);
                uint8_t sc; float d;
                block_scale(absmax_bits16(a, b), g, sc, d);
                sx = e4m3_to_float(sc);
                if (d != 0.0f) {
                    const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const float x0 = __uint_as_float(w[e] << 16), x1 = __uint_as_float(w[e] & 0xFFFF0000u);
                        const uint32_t byte = float2_to_e2m1x2(__fdiv_rn(x0, d), __fdiv_rn(x1, d));
                        h[e] = HALF ? e2m1x2_to_f16x2(byte) : byte;
                    }
                }
            }
            if (HALF) {
                uint4* dst = reinterpret_cast<uint4*>(rec + (blk & 1) * 32);
                dst[0] = make_uint4(h[0], h[1], h[2], h[3]);
                dst[1] = make_uint4(h[4], h[5], h[6], h[7]);
                *reinterpret_cast<float*>(rec + 64 + (blk & 1) * 4) = sx;
            } else {        // canonical code bytes -> the integer record (same routine as the normal staging)
                const uint2 cw = make_uint2(h[0] | (h[1] << 8) | (h[2] << 16) | (h[3] << 24),
                                            h[4] | (h[5] << 8) | (h[6] << 16) | (h[7] << 24));
                decode_x_block(cw, sx, rec, blk & 1);
            }
        }
        mbar_arrive(smem_u32(xbars + batch));
    }
}

// W4A16: work item i -> (8-element vector = i / M, m = i % M); progress published in 16-blocks
template <int M, typename Between>
__device__ __forceinline__ void stage_x_w4a16(const GemvParams& p, uint8_t* xs, int c0, int ncw, int tid, int nthr,
                                              uint64_t* xbars, Between&& between) {
    const int nvec = ncw * 4 * CELL_VECS * p.kp;                 // 8-element vectors per row in the range
    const uint16_t* xb = static_cast<const uint16_t*>(p.x);
    const int total = nvec * M;
    const int k_base = c0 * 32 * CELL_VECS * p.kp;
    for (int base = 0, batch = 0; base < total; base += nthr * STAGE_BATCH, ++batch) {
        uint4 raw[STAGE_BATCH];
#pragma unroll
        for (int t = 0; t < STAGE_BATCH; ++t) {
            const int i = base + t * nthr + tid;
            const int v = i / M, m = i - v * M;
            raw[t] = make_uint4(0, 0, 0, 0);
            if (i < total && k_base + v * 8 < p.K)
                raw[t] = __ldg(reinterpret_cast<const uint4*>(xb + (int64_t)m * p.ldx + k_base + v * 8));
        }
        if (batch == 0) between();
#pragma unroll
        for (int t = 0; t < STAGE_BATCH; ++t) {
            const int i = base + t * nthr + tid;
            if (i < total) {
                const int v = i / M, m = i - v * M;
                float* dst = reinterpret_cast<float*>(xs + (size_t)(v >> 2) * xvec_stride(KMODE_W4A16, M) + m * XBP_W4A16) + (v & 3) * 8;
                const uint32_t w[4] = {raw[t].x, raw[t].y, raw[t].z, raw[t].w};
                float4 lo, hi;
                lo.x = __uint_as_float(w[0] << 16); lo.y = __uint_as_float(w[0] & 0xFFFF0000u);
                lo.z = __uint_as_float(w[1] << 16); lo.w = __uint_as_float(w[1] & 0xFFFF0000u);
                hi.x = __uint_as_float(w[2] << 16); hi.y = __uint_as_float(w[2] & 0xFFFF0000u);
                hi.z = __uint_as_float(w[3] << 16); hi.w = __uint_as_float(w[3] & 0xFFFF0000u);
                reinterpret_cast<float4*>(dst)[0] = lo;
                reinterpret_cast<float4*>(dst)[1] = hi;
            }
        }
        mbar_arrive(smem_u32(xbars + batch));
    }
}

// ---- one 32-k vector (two 16-blocks) of R rows against all M activation rows ------------------
// packed FP32 helpers (two lanes per instruction; FFMA2 issues at the FFMA rate, _work microbenchmarks)
__device__ __forceinline__ uint64_t pack2u(uint32_t lo, uint32_t hi) {
    uint64_t v;
    asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "r"(lo), "r"(hi));
    return v;
}
__device__ __forceinline__ uint64_t fadd2(uint64_t a, uint64_t b) {
    uint64_t d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ uint64_t fmul2(uint64_t a, uint64_t b) {
    uint64_t d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ uint64_t ffma2_i8(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
// The two 16-blocks of the vector ride in the two halves of packed FP32 registers: per (row, m)
// 8 dp4a + FADD2 (remove the magic bias = int->float) + FMUL2 (sW*sX) + FFMA2, instead of
// 2 I2F + 2 FMUL + 2 FFMA.  accp[r][m] = {sum over even blocks, sum over odd blocks}.
template <int M, int R>
__device__ __forceinline__ void block_pair_w4a4(const WLut& lut, const uint4 (&wv)[R], const uint8_t* xbp,
                                                const uint64_t (&swp)[R][4], int j, uint64_t (&accp)[R][M]) {
    uint32_t u[R][8];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        decode_w_u8(lut, wv[r].x, u[r][0], u[r][1]);
        decode_w_u8(lut, wv[r].y, u[r][2], u[r][3]);
        decode_w_u8(lut, wv[r].z, u[r][4], u[r][5]);
        decode_w_u8(lut, wv[r].w, u[r][6], u[r][7]);
    }
    const uint64_t unbias = pack2u(__float_as_uint(-I8_MAGIC), __float_as_uint(-I8_MAGIC));
#pragma unroll
    for (int m = 0; m < M; ++m) {
        const uint4 xa = *reinterpret_cast<const uint4*>(xbp + m * XBP_W4A4);
        const uint4 xb = *reinterpret_cast<const uint4*>(xbp + m * XBP_W4A4 + 16);
        const uint4 ax = *reinterpret_cast<const uint4*>(xbp + m * XBP_W4A4 + 32);
        const uint64_t sx2 = pack2u(ax.z, ax.w);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            int d0 = (int)ax.x, d1 = (int)ax.y;
            d0 = dp4a_us(u[r][0], xa.x, d0); d0 = dp4a_us(u[r][1], xa.y, d0);
            d0 = dp4a_us(u[r][2], xa.z, d0); d0 = dp4a_us(u[r][3], xa.w, d0);
            d1 = dp4a_us(u[r][4], xb.x, d1); d1 = dp4a_us(u[r][5], xb.y, d1);
            d1 = dp4a_us(u[r][6], xb.z, d1); d1 = dp4a_us(u[r][7], xb.w, d1);
            const uint64_t dots = fadd2(pack2u((uint32_t)d0, (uint32_t)d1), unbias);
            accp[r][m] = ffma2_i8(dots, fmul2(swp[r][j], sx2), accp[r][m]);
        }
    }
}

// FP16 variant: F2FP.E2M1 unpack (free byte select) + HFMA2.  A half2 lane sums 8 products per
// 16-block: multiples of 0.25 bounded by 288, exact in FP16; the two lanes are added in FP32.
__device__ __forceinline__ uint32_t hfma2(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
    return d;
}
__device__ __forceinline__ uint32_t hmul2(uint32_t a, uint32_t b) {
    uint32_t d;
    asm("mul.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}
__device__ __forceinline__ uint32_t hadd2(uint32_t a, uint32_t b) {
    uint32_t d;
    asm("add.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
    return d;
}
__device__ __forceinline__ float2 h2_to_float2(uint32_t h2) {
    float2 r;
    asm("{.reg .b16 lo, hi; mov.b32 {lo, hi}, %2; cvt.f32.f16 %0, lo; cvt.f32.f16 %1, hi;}"
        : "=f"(r.x), "=f"(r.y) : "r"(h2));
    return r;
}
// lo + hi of a half2 in FP32: one f16->f32 conversion and one mixed-precision add (SASS FHADD)
__device__ __forceinline__ float h2_sum_f32(uint32_t h2) {
    float r;
    asm("{.reg .b16 lo, hi; .reg .f32 t; mov.b32 {lo, hi}, %1; cvt.f32.f16 t, lo; add.rn.f32.f16 %0, hi, t;}"
        : "=f"(r) : "r"(h2));
    return r;
}
template <int M, int R>
__device__ __forceinline__ void block_pair_w4a4_h(const uint4 (&wv)[R], const uint8_t* xbp, const uint64_t (&swp)[R][4],
                                                  int j, uint64_t (&accp)[R][M]) {
    uint32_t wh[R][16];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        uint32_t t[4];
        cvt_word_e2m1(wv[r].x, t); wh[r][0] = t[0]; wh[r][1] = t[1]; wh[r][2] = t[2]; wh[r][3] = t[3];
        cvt_word_e2m1(wv[r].y, t); wh[r][4] = t[0]; wh[r][5] = t[1]; wh[r][6] = t[2]; wh[r][7] = t[3];
        cvt_word_e2m1(wv[r].z, t); wh[r][8] = t[0]; wh[r][9] = t[1]; wh[r][10] = t[2]; wh[r][11] = t[3];
        cvt_word_e2m1(wv[r].w, t); wh[r][12] = t[0]; wh[r][13] = t[1]; wh[r][14] = t[2]; wh[r][15] = t[3];
    }
#pragma unroll
    for (int m = 0; m < M; ++m) {
        const uint4* xr = reinterpret_cast<const uint4*>(xbp + m * XBP_W4A4H);
        const uint4 x0 = xr[0], x1 = xr[1], x2 = xr[2], x3 = xr[3];
        const uint2 sxb = *reinterpret_cast<const uint2*>(xbp + m * XBP_W4A4H + 64);
        const uint64_t sx2 = pack2u(sxb.x, sxb.y);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            // two independent 4-deep chains per block, merged by an exact HADD2 (|sums| <= 288)
            uint32_t a0 = hmul2(wh[r][0], x0.x), b0 = hmul2(wh[r][4], x1.x);
            uint32_t a1 = hmul2(wh[r][8], x2.x), b1 = hmul2(wh[r][12], x3.x);
            a0 = hfma2(wh[r][1], x0.y, a0); b0 = hfma2(wh[r][5], x1.y, b0);
            a1 = hfma2(wh[r][9], x2.y, a1); b1 = hfma2(wh[r][13], x3.y, b1);
            a0 = hfma2(wh[r][2], x0.z, a0); b0 = hfma2(wh[r][6], x1.z, b0);
            a1 = hfma2(wh[r][10], x2.z, a1); b1 = hfma2(wh[r][14], x3.z, b1);
            a0 = hfma2(wh[r][3], x0.w, a0); b0 = hfma2(wh[r][7], x1.w, b0);
            a1 = hfma2(wh[r][11], x2.w, a1); b1 = hfma2(wh[r][15], x3.w, b1);
            a0 = hadd2(a0, b0); a1 = hadd2(a1, b1);
            // f32(lo) + f32(hi) per block: exact (|sum| <= 576); the two blocks' sW*sX products and the
            // accumulation ride in packed FP32 (one FMUL2 + one FFMA2 per row, m and block pair)
            const uint64_t dots = pack2u(__float_as_uint(h2_sum_f32(a0)), __float_as_uint(h2_sum_f32(a1)));
            accp[r][m] = ffma2_i8(dots, fmul2(swp[r][j], sx2), accp[r][m]);
        }
    }
}

// W4A16: weights to FP32 pairs (F2FP.E2M1 + two f16->f32), packed FP32 FMA (fma.rn.f32x2: two MACs per
// instruction) against FP32 copies of the BF16 activations; two 4-deep chains per 16-block.
__device__ __forceinline__ uint64_t pack2(float lo, float hi) {
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ uint64_t ffma2(uint64_t a, uint64_t b, uint64_t c) {
    uint64_t d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ float2 unpack2(uint64_t v) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}
template <int M, int R>
__device__ __forceinline__ void block_pair_w4a16(const uint4 (&wv)[R], const uint8_t* xbp, const float (&sw)[R][8],
                                                 int j, float (&acc)[R][M]) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const uint32_t ww[4] = {wv[r].x, wv[r].y, wv[r].z, wv[r].w};
#pragma unroll
        for (int h = 0; h < 2; ++h) {                                      // the two 16-blocks
            uint64_t wp[8];
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                uint32_t hw[4];
                cvt_word_e2m1(ww[h * 2 + q], hw);
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const float2 f = h2_to_float2(hw[b]);
                    wp[q * 4 + b] = pack2(f.x, f.y);
                }
            }
#pragma unroll
            for (int m = 0; m < M; ++m) {
                const ulonglong2* xp = reinterpret_cast<const ulonglong2*>(xbp + m * XBP_W4A16) + h * 4;
                const ulonglong2 x0 = xp[0], x1 = xp[1], x2 = xp[2], x3 = xp[3];
                uint64_t da = ffma2(wp[0], x0.x, 0ull), db = ffma2(wp[4], x2.x, 0ull);
                da = ffma2(wp[1], x0.y, da); db = ffma2(wp[5], x2.y, db);
                da = ffma2(wp[2], x1.x, da); db = ffma2(wp[6], x3.x, db);
                da = ffma2(wp[3], x1.y, da); db = ffma2(wp[7], x3.y, db);
                const float2 fa = unpack2(da), fb = unpack2(db);
                acc[r][m] = fmaf((fa.x + fa.y) + (fb.x + fb.y), sw[r][2 * j + h], acc[r][m]);
            }
        }
    }
}

// ---- shared-memory carve-up: ONE definition for the host (gemv_smem_bytes) and the kernel -----------
struct SmemMap { uint32_t xs, ring, slots, aslots, hand, bars, xbars, hbars, cnt, bstart, astart, misc, total; };
__host__ __device__ inline SmemMap gemv_smem_map(int kmode, int M, int R, int W, int S, int rpt, int ncw_max, int kp,
                                                 int nxb, int base, int nb, int amax, int nhand) {
    SmemMap m;
    uint32_t o = 0;
    const uint32_t slot_bytes = (uint32_t)R * M * rpt * 4;
    m.xs = o;     o += ((uint32_t)ncw_max * CELL_VECS * kp * xvec_stride(kmode, M) + 127u) & ~127u;   // activation records
    m.ring = o;   o += (uint32_t)W * S * R * CELL_BYTES;                   // per-warp bulk-copy rings
    m.slots = o;  o += (uint32_t)W * 2 * slot_bytes;                       // phase B segment partials (two per warp)
    m.aslots = o; o += (uint32_t)amax * slot_bytes;                        // phase A: one partial per leftover cell
    m.hand = o;   o += (uint32_t)nhand * slot_bytes;                       // CTA sums handed to the closer warps
    o = (o + 7u) & ~7u;
    m.bars = o;   o += (uint32_t)W * S * 8;                                // ring mbarriers
    m.xbars = o;  o += (uint32_t)nxb * 8;                                  // staging-batch mbarriers
    m.hbars = o;  o += (uint32_t)(nhand + 1) * 8;                          // hand-off mbarriers + the header-check barrier
    m.cnt = o;    o += (uint32_t)(base + 3) * 4;                           // arrival counters: [0,1] leftover units, [2..] whole units
    m.bstart = o; o += (uint32_t)(W + 1) * 4;                              // phase B: warp share starts
    m.astart = o; o += (uint32_t)2 * (nb + 1) * 4;                         // phase A: CTA share starts, both slice variants
    m.misc = o;   o += (2 + 32) * 4;                                       // [0] fused gX, [1] blob-ok flag, [2..] per-warp amax
    m.total = (o + 15u) & ~15u;
    return m;
}

// CTA-constant context of the work split
struct CtaCtx {
    int ncw;            // cells per unit in this CTA's K slice
    int var;            // slice variant (0: cells_q, 1: cells_q + 1 cells per unit)
    int nb;             // CTAs per slice
    int unit0;          // phase B: global index of this CTA's first whole unit
    int a0, na;         // phase A: this CTA's leftover cells [a0, a0 + na) of the slice's leftover stream
    int qa0, n0;        // first leftover unit touched, and how many of the na cells belong to it
    const int* astart;  // [2][nb + 1] leftover share starts per variant (entries above nba repeat the end)
};

// CTAs of a variant-v slice whose leftover share intersects leftover unit q: [lo, hi].  The starts are
// strictly increasing over the nba participating CTAs; the float estimate is corrected against the table.
__device__ __forceinline__ void contrib_range(const GemvParams& p, const CtaCtx& c, int v, int q, int& lo, int& hi) {
    const int ncw_v = p.cells_q + v, nba = p.nba[v];
    const int* cs = c.astart + v * (c.nb + 1);
    const int x0 = q * ncw_v, x1 = x0 + ncw_v - 1;
    int b = (int)((float)x0 * p.inv_a[v]);
    b = b < 0 ? 0 : (b > nba - 1 ? nba - 1 : b);
    while (b + 1 < nba && cs[b + 1] <= x0) ++b;
    while (cs[b] > x0) --b;
    lo = b;
    while (b + 1 < nba && cs[b + 1] <= x1) ++b;
    hi = b;
}

__device__ __forceinline__ unsigned long long globaltimer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
#ifdef NVFP4_ENABLE_TRACE      // debug builds only (-DNVFP4_ENABLE_TRACE): per-phase %globaltimer stamps, 64 per CTA
#define NVFP4_TRACE(slot) do { if (p.trace) p.trace[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 64 + (slot)] = globaltimer_ns(); } while (0)
#define NVFP4_CLK(i) do { if (threadIdx.x == 0) clk_[i] = clock64(); } while (0)
#define NVFP4_CLK_DECL long long clk_[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}
#define NVFP4_CLK_FLUSH do { if (threadIdx.x == 0 && p.trace) for (int i_ = 0; i_ < 16; ++i_) \
    p.trace[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 64 + 48 + i_] = (unsigned long long)(clk_[i_] ? clk_[i_] - clk_[0] : 0); } while (0)
#else
#define NVFP4_TRACE(slot) do { } while (0)
#define NVFP4_CLK(i) do { } while (0)
#define NVFP4_CLK_DECL do { } while (0)
#define NVFP4_CLK_FLUSH do { } while (0)
#endif

__device__ __forceinline__ void store_y(const GemvParams& p, int m, int n, float v) {
    if (p.y_bf16) static_cast<uint16_t*>(p.y)[(int64_t)m * p.ldy + n] = float_to_bf16_rn(v);
    else          static_cast<float*>(p.y)[(int64_t)m * p.ldy + n] = v;
}

// ---- a7 (closer warps): complete a unit this CTA holds only a part of.  `hand` = the CTA's FP32 sums
// [(r*M + m)*rpt + row].  kind A: leftover unit q (cut between CTAs, and between K slices); kind B: whole unit
// (cut between K slices only).  The partial goes to the workspace; the last CTA to arrive for the unit sums all
// contributions in a fixed order (slice-major, then CTA order) and writes the outputs.
template <int M, int R>
__device__ __forceinline__ void close_unit(const GemvParams& p, const CtaCtx& c, const float* hand, bool kind_a, int idx,
                                           int lane, int rpt, float gs) {
    // idx: kind A -> leftover unit q; kind B -> local whole unit ul
    const int unit = kind_a ? (p.base * c.nb + idx) : (c.unit0 + idx);
    const int prow0 = (kind_a ? idx : unit) * R * rpt;                  // first row inside partials_a / partials_b
    int lo0 = 0, hi0 = -1, lo1 = 0, hi1 = -1;
    const int nvar1 = p.cells_r, nvar0 = p.ksplit - p.cells_r;          // slices per variant
    unsigned int expected = (unsigned int)p.ksplit;
    float* mine;
    if (kind_a) {
        if (nvar0 > 0) contrib_range(p, c, 0, idx, lo0, hi0);
        if (nvar1 > 0) contrib_range(p, c, 1, idx, lo1, hi1);
        expected = (unsigned int)(nvar0 * (hi0 - lo0 + 1) + nvar1 * (hi1 - lo1 + 1));
        mine = p.partials_a + (int64_t)((int)blockIdx.y * p.jmax + ((int)blockIdx.x - (c.var ? lo1 : lo0))) * M * p.npad_a;
    } else {
        mine = p.partials_b + (int64_t)blockIdx.y * M * p.npad_b;
    }
    const int npad = kind_a ? p.npad_a : p.npad_b;
    const int nval = R * M * rpt;
    for (int i = lane; i < nval; i += 32) {
        const int row = i % rpt, rm = i / rpt, m = rm % M, r = rm / M;
        __stcg(mine + (int64_t)m * npad + prow0 + r * rpt + row, hand[i]);
    }
    __threadfence();
    __syncwarp();
    unsigned int last = 0;
    if (lane == 0) {
        const unsigned int old = atomicAdd(p.counters + unit, 1u);
        last = (old == expected - 1u);
        if (last) p.counters[unit] = 0u;                              // leave the workspace clean
    }
    last = __shfl_sync(0xFFFFFFFFu, last, 0);
    if (!last) return;
    __threadfence();
    for (int i = lane; i < nval; i += 32) {
        const int row = i % rpt, rm = i / rpt, m = rm % M, r = rm / M;
        const int n = (unit * R + r) * rpt + row;
        if (unit * R + r >= p.ntiles || n >= p.N) continue;
        float sum = 0.0f;
        for (int ks = 0; ks < p.ksplit; ++ks) {
            if (kind_a) {
                const int nj = ks < p.cells_r ? (hi1 - lo1) : (hi0 - lo0);
                for (int j = 0; j <= nj; ++j)
                    sum += __ldcg(p.partials_a + ((int64_t)(ks * p.jmax + j) * M + m) * npad + prow0 + r * rpt + row);
            } else {
                sum += __ldcg(p.partials_b + ((int64_t)ks * M + m) * npad + prow0 + r * rpt + row);
            }
        }
        store_y(p, m, n, sum * (p.gscale_per_row ? gs * __ldg(p.x_gscale + m) : gs));
    }
}

// K parts of a row are summed by shuffles (lanes of one row are rpt apart)
template <int M, int R>
__device__ __forceinline__ void reduce_parts(float (&acc)[R][M], int rpt) {
    for (int off = rpt; off < 32; off <<= 1) {
#pragma unroll
        for (int r = 0; r < R; ++r)
#pragma unroll
            for (int m = 0; m < M; ++m) acc[r][m] += __shfl_xor_sync(0xFFFFFFFFu, acc[r][m], off);
    }
}
// the CTA's sums of a finished unit: outputs (the CTA holds the whole unit) or hand-off to a closer warp
template <int M, int R>
__device__ __forceinline__ void emit_or_hand(const GemvParams& p, float (&acc)[R][M], bool direct, int unit, float* hand,
                                             uint64_t* hbars, int h, int lane, bool writer, int rsub, int rpt, float gs) {
    if (direct) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int n = (unit * R + r) * rpt + rsub;
            if (writer && unit * R + r < p.ntiles && n < p.N) {
#pragma unroll
                for (int m = 0; m < M; ++m)
                    store_y(p, m, n, acc[r][m] * (p.gscale_per_row ? gs * __ldg(p.x_gscale + m) : gs));
            }
        }
    } else {
        float* dst = hand + (size_t)h * (R * M * rpt);
        if (writer) {
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int m = 0; m < M; ++m) dst[(r * M + m) * rpt + rsub] = acc[r][m];
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(hbars + h));
    }
}
__device__ __forceinline__ int arrive_count(int* cnt_word, int lane) {     // CTA-scope acq_rel arrival; old value to all lanes
    int old = 0;
    __syncwarp();                                   // the writer lanes' slot stores are ordered before the arrival
    if (lane == 0)
        asm volatile("atom.acq_rel.cta.shared::cta.add.u32 %0, [%1], 1;" : "=r"(old) : "r"(smem_u32(cnt_word)) : "memory");
    return __shfl_sync(0xFFFFFFFFu, old, 0);
}

// ---- a6, phase A: a warp finished leftover cell i (0 <= i < na) of this CTA.  Every leftover cell is its own
// segment; its partial goes to aslots[i]; the last cell of a leftover unit to arrive sums the unit's cells in
// index order (deterministic) and hands the CTA's sum to a closer warp (or writes it, if the CTA holds the
// whole unit and K is not sliced).
template <int M, int R>
__device__ __forceinline__ void finish_leftover_cell(const GemvParams& p, const CtaCtx& c, float (&acc)[R][M], float* aslots,
                                                     float* hand, uint64_t* hbars, int* cnt, int i, int lane, int part,
                                                     int rsub, int rpt, float gs) {
    reduce_parts<M, R>(acc, rpt);
    const bool writer = (part == 0);
    const int slot_floats = R * M * rpt;
    const int qa = i < c.n0 ? 0 : 1;                                         // which of the (at most two) leftover units
    const int ilo = qa ? c.n0 : 0, ihi = qa ? c.na - 1 : c.n0 - 1;
    if (ihi > ilo) {
        float* mine = aslots + (size_t)i * slot_floats;
        if (writer) {
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int m = 0; m < M; ++m) mine[(r * M + m) * rpt + rsub] = acc[r][m];
        }
        if (arrive_count(cnt + qa, lane) != ihi - ilo) return;
        if (writer) {
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int m = 0; m < M; ++m) acc[r][m] = 0.0f;
            for (int k = ilo; k <= ihi; ++k) {
                const float* sl = aslots + (size_t)k * slot_floats;
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int m = 0; m < M; ++m) acc[r][m] += *(volatile const float*)(sl + (r * M + m) * rpt + rsub);
            }
        }
    }
    const bool direct = (p.ksplit == 1) && (ihi - ilo + 1 == c.ncw);
    emit_or_hand<M, R>(p, acc, direct, p.base * c.nb + c.qa0 + qa, hand, hbars, qa, lane, writer, rsub, rpt, gs);
}

// ---- a6, phase B: a warp finished its segment of local whole unit `ul`.  A unit shared by several warps is
// combined through shared-memory slots (two per warp: slot 0 = the segment that starts the warp's run,
// slot 1 = its last one; every other segment covers a whole unit) by the LAST warp to arrive, in fixed warp
// order -> deterministic.
template <int M, int R>
__device__ __forceinline__ void finish_segment(const GemvParams& p, const CtaCtx& c, float (&acc)[R][M], float* slots,
                                               float* hand, uint64_t* hbars, int* cnt, const int* bstart, int ul,
                                               bool whole, bool seg_at_run_start, int warp, int lane, int part, int rsub,
                                               int rpt, float gs) {
    reduce_parts<M, R>(acc, rpt);
    const bool writer = (part == 0);
    const int slot_floats = R * M * rpt;
    if (!whole) {
        const int W = p.warps;
        float* mine = slots + (size_t)(warp * 2 + (seg_at_run_start ? 0 : 1)) * slot_floats;
        if (writer) {
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int m = 0; m < M; ++m) mine[(r * M + m) * rpt + rsub] = acc[r][m];
        }
        // contributors of this unit: warps whose run intersects [ul*ncw, (ul+1)*ncw) (every warp has >= 1 cell)
        const int lo = ul * c.ncw, hi = lo + c.ncw - 1;
        int w_first = 0, w_last = 0;
        for (int w = 0; w < W; ++w) {
            const int fs = bstart[w];
            if (fs <= lo) w_first = w;
            if (fs <= hi) w_last = w;
        }
        if (arrive_count(cnt + 2 + ul, lane) != w_last - w_first) return;
        if (writer) {
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int m = 0; m < M; ++m) acc[r][m] = 0.0f;
            for (int w = w_first; w <= w_last; ++w) {
                const float* sl = slots + (size_t)(w * 2 + (bstart[w] >= lo ? 0 : 1)) * slot_floats;
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int m = 0; m < M; ++m) acc[r][m] += *(volatile const float*)(sl + (r * M + m) * rpt + rsub);
            }
        }
    }
    emit_or_hand<M, R>(p, acc, p.ksplit == 1, c.unit0 + ul, hand, hbars, 2 + ul, lane, writer, rsub, rpt, gs);
}

// threads per CTA the instantiation is compiled for (consumer + stager warps): the FP16 path (M = 1) runs up to
// 16 consumer warps at <= 102 registers; the integer and W4A16 paths 12 consumer warps at 128 registers (no
// spills in the main loop: profiles/r02_ptxas.md; 12 warps measured as fast as 16 at M >= 2)
__host__ __device__ constexpr int gemv_max_threads(int kmode, int M, int R) {
    if (kmode == KMODE_W4A4_H) return 640;
    if (kmode == KMODE_W4A4_I8 && M <= 2 && R == 1) return 640;           // 16 consumer warps at <= 102 registers
    return 512;
}

// Persistent and balanced (see the file header).  STAGER_WARPS extra warps help to decode the activations and
// afterwards complete the row tiles this CTA shares with other CTAs.
template <int MODE, int M, int R>
__global__ void __launch_bounds__(gemv_max_threads(MODE, M, R)) gemv_kernel(const GemvParams p) {
    extern __shared__ __align__(128) uint8_t smem[];
    NVFP4_CLK_DECL;
    NVFP4_CLK(0);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int W = p.warps, S = p.stages;
    const int rsub = lane & ((32 >> p.kp_shift) - 1), part = lane >> (5 - p.kp_shift);   // lane = part*rpt + rsub
    const int rpt = 32 >> p.kp_shift;
    constexpr uint32_t STAGE_BYTES = R * CELL_BYTES;
    NVFP4_CLK(1);
    if (threadIdx.x == 0) NVFP4_TRACE(0);
    // a blob that was not repacked for this (N, K, KP, ABI version) must not produce plausible numbers: one thread
    // per CTA (the first stager thread) loads the header right away (a cold DRAM access, kept OFF the staging path)
    // and publishes the verdict through an mbarrier that is checked before the first output is written
    uint4 hdr = make_uint4(0u, 0u, 0u, 0u);
    const bool checker = (threadIdx.x == p.warps * 32);
    if (checker) hdr = __ldg(reinterpret_cast<const uint4*>(p.blob - BLOB_HEADER_BYTES));

    // K slice of this CTA (whole cells of 256*kp k); quotients and remainders come from the host
    const int by = blockIdx.y, bx = blockIdx.x, nb = gridDim.x;
    CtaCtx c;
    c.var = by < p.cells_r ? 1 : 0;
    c.nb = nb;
    const int c0 = by * p.cells_q + (by < p.cells_r ? by : p.cells_r);
    const int ncw = p.cells_q + c.var;
    c.ncw = ncw;
    const int ncw_max = p.cells_q + (p.cells_r > 0 ? 1 : 0);
    // phase A: this CTA's equal share of the leftover units' flat cell stream; phase B: `base` whole units
    {
        const unsigned nba = (unsigned)p.nba[c.var], aq = (unsigned)p.a_q[c.var], ar = (unsigned)p.a_r[c.var];
        unsigned a0 = 0, a1 = 0;
        if ((unsigned)bx < nba) {
            a0 = (unsigned)bx * aq + fastdiv((unsigned)bx * ar, p.fd_nba[c.var]);
            a1 = (unsigned)(bx + 1) * aq + fastdiv((unsigned)(bx + 1) * ar, p.fd_nba[c.var]);
        }
        c.a0 = (int)a0; c.na = (int)(a1 - a0);
        c.qa0 = (int)fastdiv(a0, p.fd_ncw[c.var]);
        const int room = (c.qa0 + 1) * ncw - c.a0;                          // cells left in the first leftover unit
        c.n0 = c.na < room ? c.na : room;
    }
    NVFP4_CLK(2);
    const int my_base = p.base + ((p.whole_units && bx < p.ur) ? 1 : 0);   // whole units of this CTA ...
    c.unit0 = bx * p.base + (p.whole_units ? (bx < p.ur ? bx : p.ur) : 0);  // ... starting at this global unit
    const int Bc = my_base * ncw;                                           // phase B cells of this CTA

    SmemMap map;                                                            // computed by the host (gemv_smem_map)
    map.xs = p.smem_map[0]; map.ring = p.smem_map[1]; map.slots = p.smem_map[2]; map.aslots = p.smem_map[3];
    map.hand = p.smem_map[4]; map.bars = p.smem_map[5]; map.xbars = p.smem_map[6]; map.hbars = p.smem_map[7];
    map.cnt = p.smem_map[8]; map.bstart = p.smem_map[9]; map.astart = p.smem_map[10]; map.misc = p.smem_map[11];
    map.total = p.smem_map[12];
    (void)ncw_max;
    uint8_t* xs = smem + map.xs;                                             // activations
    constexpr int XVS = xvec_stride(MODE, M);
    uint8_t* ring_all = smem + map.ring;
    float* slots = reinterpret_cast<float*>(smem + map.slots);
    float* aslots = reinterpret_cast<float*>(smem + map.aslots);
    float* hand = reinterpret_cast<float*>(smem + map.hand);
    uint64_t* bars_all = reinterpret_cast<uint64_t*>(smem + map.bars);
    uint64_t* xbars = reinterpret_cast<uint64_t*>(smem + map.xbars);
    uint64_t* hbars = reinterpret_cast<uint64_t*>(smem + map.hbars);
    int* cnt = reinterpret_cast<int*>(smem + map.cnt);
    int* bstart = reinterpret_cast<int*>(smem + map.bstart);
    int* astart = reinterpret_cast<int*>(smem + map.astart);
    float* gx_slot = reinterpret_cast<float*>(smem + map.misc);
    volatile int* blob_flag = reinterpret_cast<volatile int*>(smem + map.misc) + 1;
    uint32_t* red = reinterpret_cast<uint32_t*>(smem + map.misc) + 2;
    c.astart = astart;
    const bool fused = (MODE != KMODE_W4A16) && p.fuse_quant;
    const bool records = (MODE == KMODE_W4A4_H) && p.x_records != nullptr;
    // items per staging batch (records: the one bulk copy covers every item)
    const int stage_items = records ? (1 << 28) : fused ? (int)blockDim.x : (int)blockDim.x * STAGE_BATCH;

    // ---- consumer warps: request the first weight cells before anything else (private ring, private barriers) ----
    // warp w: phase A cells i = w, w + W, ... < na (na_w of them), then phase B cells [bs, be) of the CTA's Bc
    const bool consumer = warp < W;
    const int na_w = consumer ? (int)fastdiv((unsigned)(c.na + W - 1 - warp), p.fd_w) : 0;
    const int bs = consumer ? Bc - (int)fastdiv((unsigned)(W - warp) * (unsigned)Bc, p.fd_w) : 0;
    const int be = consumer ? Bc - (int)fastdiv((unsigned)(W - warp - 1) * (unsigned)Bc, p.fd_w) : 0;
    const int total = na_w + (be - bs);
    const int64_t tile_stride = (int64_t)p.nch * CELL_BYTES;
    uint8_t* ring = ring_all + (size_t)(consumer ? warp : 0) * S * STAGE_BYTES;
    uint64_t* bars = bars_all + (consumer ? warp : 0) * S;
    const bool leader = consumer && (lane == 0);
    // producer cursor (used by lane 0 only): next cell to request.  The warp's cells form RUNS of cells that are
    // contiguous in the blob: every leftover cell is a run of one, then one run per whole unit touched.
    int p_left = 0, p_count = 0, p_nv = 0, p_a = 0, p_tile0 = 0;
    bool p_b_started = false;
    uint32_t p_dst = smem_u32(ring), p_bar = smem_u32(bars);
    const uint32_t ring_end = p_dst + (uint32_t)S * STAGE_BYTES;
    const uint8_t* p_src = nullptr;
    const int64_t unit_jump = (int64_t)(R - 1) * tile_stride + (int64_t)(p.nch - ncw) * CELL_BYTES;
    auto next_run = [&]() {
        int tile0;
        if (p_a < na_w) {                                                   // phase A: leftover cell i = warp + p_a*W
            const int fa = c.a0 + warp + p_a * W;
            const int q = (int)fastdiv((unsigned)fa, p.fd_ncw[c.var]), cell = fa - q * ncw;
            tile0 = (p.base * nb + q) * R;
            p_src = p.blob + ((int64_t)tile0 * p.nch + c0 + cell) * CELL_BYTES;
            p_left = 1;
            ++p_a;
        } else if (!p_b_started) {                                          // phase B starts: cell bs of the CTA's whole units
            p_b_started = true;
            const int ul = (int)fastdiv((unsigned)bs, p.fd_ncw[c.var]), cell = bs - ul * ncw;
            tile0 = (c.unit0 + ul) * R;
            p_src = p.blob + ((int64_t)tile0 * p.nch + c0 + cell) * CELL_BYTES;
            p_left = ncw - cell;
        } else {                                                            // next whole unit of the run
            p_src += unit_jump;
            p_left = ncw;
            tile0 = p_tile0 + R;
        }
        p_tile0 = tile0;
        p_nv = p.ntiles - tile0; p_nv = p_nv > R ? R : p_nv;
    };
    auto issue = [&]() {
        mbar_arrive_expect_tx(p_bar, (uint32_t)p_nv * CELL_BYTES);
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (r < p_nv) bulk_g2s(p_dst + r * CELL_BYTES, p_src + r * tile_stride, CELL_BYTES, p_bar);
        ++p_count;
        p_src += CELL_BYTES;
        if (--p_left == 0) next_run();
        p_dst += STAGE_BYTES; p_bar += 8;
        if (p_dst == ring_end) { p_dst -= (uint32_t)S * STAGE_BYTES; p_bar -= (uint32_t)S * 8; }
    };
    NVFP4_CLK(3);
    if (leader) {
        for (int s = 0; s < S; ++s) mbar_init(smem_u32(bars + s), 1);
        mbar_fence_init();
        NVFP4_CLK(4);
        if (total > 0) next_run();
        NVFP4_CLK(5);
        // ONE cell per warp now: a burst of S cells per warp arrives interleaved (every cell lands at the END of the
        // burst) and the activation loads issued after griddepcontrol.wait would queue behind all of it
        if (total > 0) issue();
    }
    NVFP4_CLK(6);
    if (threadIdx.x == 0) NVFP4_TRACE(1);

    // ---- CTA-wide barriers (the tables follow under the latency of the activation loads: `deferred` below) ----
    for (int i = threadIdx.x; i < p.nxb; i += blockDim.x) mbar_init(smem_u32(xbars + i), blockDim.x);
    for (int i = threadIdx.x; i <= p.nhand; i += blockDim.x) mbar_init(smem_u32(hbars + i), 1);
    if (threadIdx.x == 0) mbar_fence_init();
    NVFP4_CLK(7);
    __syncthreads();
    NVFP4_CLK(8);

    // the weight stream is under way; everything below touches data of the previous kernel
    pdl_wait();
    pdl_launch_dependents();
    if (MODE == KMODE_W4A4_H && p.x_records != nullptr && threadIdx.x == 0) {   // activation records: first thing after the wait
        const uint32_t bytes = (uint32_t)(ncw * CELL_VECS * p.kp) * (uint32_t)xvec_stride(MODE, M);
        mbar_arrive_expect_tx(smem_u32(xbars), bytes);
        bulk_g2s(smem_u32(xs), p.x_records + (size_t)(c0 * CELL_VECS * p.kp) * xvec_stride(MODE, M), bytes, smem_u32(xbars));
    }
    NVFP4_CLK(9);
    if (threadIdx.x == 0) NVFP4_TRACE(2);
    // global scales: issue the loads now, combine them only when the first segment is written
    const float gw_raw = __ldg(p.w_gscale);
    const float gx_raw = (MODE == KMODE_W4A16 || fused || p.gscale_per_row) ? 1.0f : __ldg(p.x_gscale);
    // Runs in every thread right after its first activation loads are in flight (or before the fused quantizer):
    // the rest of the ring prefetch, then the CTA-wide tables.  Every thread's stores precede its arrival on the first
    // staging barrier, and every reader has waited on a staging barrier (or on a hand-off that follows one).
    bool deferred_done = false;
    auto deferred = [&]() {
        deferred_done = true;
        if (leader) {
            const int npre = total < S ? total : S;
            while (p_count < npre) issue();
        }
        for (int i = threadIdx.x; i < p.base + 3; i += blockDim.x) cnt[i] = 0;
        if (threadIdx.x <= W) bstart[threadIdx.x] = Bc - (int)fastdiv((unsigned)(W - threadIdx.x) * (unsigned)Bc, p.fd_w);
        if (p.nba[0] | p.nba[1]) {
            for (unsigned b = threadIdx.x; b <= (unsigned)nb; b += blockDim.x) {
#pragma unroll
                for (int v = 0; v < 2; ++v) {
                    const unsigned nba = (unsigned)p.nba[v];
                    const unsigned bb = b < nba ? b : nba;                  // CTAs that take no part repeat the end
                    astart[v * (nb + 1) + b] = nba ? (int)(bb * (unsigned)p.a_q[v] + fastdiv(bb * (unsigned)p.a_r[v], p.fd_nba[v])) : 0;
                }
            }
        }
    };
    // activation staging: every thread of the CTA takes its share
    if (records) {
        // the quantizer wrote the records (32 f16 values + two FP32 block scales per 32 k, padded K zero): one bulk copy of
        // this CTA's K range, completion on the first staging barrier together with every thread's arrival
        // (requested right behind griddepcontrol.wait, above)
        deferred();
        if (threadIdx.x != 0) mbar_arrive(smem_u32(xbars));
    } else if (MODE == KMODE_W4A16) stage_x_w4a16<M>(p, xs, c0, ncw, threadIdx.x, blockDim.x, xbars, deferred);
    else if (fused) {
        deferred();
        stage_x_fused<M, MODE == KMODE_W4A4_H>(p, xs, c0, ncw, threadIdx.x, blockDim.x, xbars, red, gx_slot);
    } else stage_x_w4a4<M, MODE == KMODE_W4A4_H>(p, xs, c0, ncw, threadIdx.x, blockDim.x, xbars, deferred);
    if (!deferred_done) deferred();
    NVFP4_CLK(10);
    if (threadIdx.x == W * 32) NVFP4_TRACE(9);
    const uint32_t hdr_bar = smem_u32(hbars + p.nhand);
    if (checker) {                                                          // after this thread's share of the staging
        *blob_flag = (hdr.x == p.hdr_expect.x) && (hdr.y == p.hdr_expect.y) && (hdr.z == p.hdr_expect.z) &&
                     (hdr.w == p.hdr_expect.w);
        mbar_arrive(hdr_bar);
    }

    if (!consumer) {                                                        // ---- closer warps ----
        // units this CTA holds only a part of: the (at most two) leftover units, and with K slices every whole unit
        const int sw = warp - W, nsw = (int)(blockDim.x >> 5) - W;
        const int njobs = 2 + (p.ksplit > 1 ? my_base : 0);
        for (int j = sw; j < njobs; j += nsw) {
            if (j == 0 && (c.n0 == 0 || (p.ksplit == 1 && c.n0 == ncw))) continue;
            if (j == 1 && c.na - c.n0 == 0) continue;                       // (a second leftover unit is never whole)
            mbar_wait(smem_u32(hbars + j), 0u);
            mbar_wait(hdr_bar, 0u);
            float g = gw_raw;
            if (MODE != KMODE_W4A16) {
                g = g * (fused ? *reinterpret_cast<volatile float*>(gx_slot) : gx_raw);
                if (MODE == KMODE_W4A4_I8) g *= 0.25f;                       // ints are 2*e (exact scaling)
            }
            if (!*blob_flag) g = __int_as_float(0x7FC00000);
            if (lane == 0) NVFP4_TRACE(10 + (j & 1) * 2);
            close_unit<M, R>(p, c, hand + (size_t)j * (R * M * rpt), j < 2, j < 2 ? c.qa0 + j : j - 2, lane, rpt, g);
            if (lane == 0) NVFP4_TRACE(11 + (j & 1) * 2);
        }
        return;
    }

    // ---- consumer warps ----
    float acc[R][M];
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int m = 0; m < M; ++m) acc[r][m] = 0.0f;

    uint64_t accp[R][M];                       // W4A4 paths: packed {even blocks, odd blocks} partial sums
#pragma unroll
    for (int r = 0; r < R; ++r)
#pragma unroll
        for (int m = 0; m < M; ++m) accp[r][m] = 0ull;

    const WLut lut = make_wlut((uint32_t)p.zero);
    // this lane's activation records: vector (cell*8 + j)*kp + part  ->  stride between j steps = kp records
    const size_t xstep = (size_t)p.kp * XVS;
    const uint8_t* xlane0 = xs + (size_t)part * XVS;
    constexpr int ITEMS_PER_CELL_KP = M * CELL_VECS * ((MODE == KMODE_W4A16) ? 4 : 2); // staging items per cell and K part
    const int x_items_cell = p.kp * ITEMS_PER_CELL_KP;
    // loop state kept incremental: consumer stage pointer and barrier, cells left in the current segment,
    // staging items this lane's next cell depends on
    const uint8_t* st = ring;
    const uint8_t* const st_end = ring + (size_t)S * STAGE_BYTES;
    uint32_t bar = smem_u32(bars);
    uint32_t phase = 0;
    // segments: a leftover cell (phase A) is a segment of its own; in phase B a segment ends with its unit
    int c_ul = 0, seg_left = 0, seg_cell0 = 0, seg_len = 0, a_k = 0;
    bool seg_first = true, seg_in_a = false, b_started = false, hdr_known = false;
    const uint8_t* xlane = xlane0;
    int x_need = 0;
    int x_have = 0;                                                         // items known to be staged
    uint32_t xbar = smem_u32(xbars);
    auto next_segment = [&](int left) {                                     // left = cells of this warp still to do (> 0)
        int cell;
        if (a_k < na_w) {
            const int fa = c.a0 + warp + a_k * W;
            cell = fa - (int)fastdiv((unsigned)fa, p.fd_ncw[c.var]) * ncw;
            seg_in_a = true; seg_len = 1;
        } else if (!b_started) {
            b_started = true; seg_in_a = false;
            c_ul = (int)fastdiv((unsigned)bs, p.fd_ncw[c.var]);
            cell = bs - c_ul * ncw;
            seg_len = ncw - cell < left ? ncw - cell : left;
        } else {
            ++c_ul; cell = 0;
            seg_len = ncw < left ? ncw : left;
        }
        seg_cell0 = cell; seg_left = seg_len;
        xlane = xlane0 + (size_t)cell * CELL_VECS * xstep;
        x_need = (cell + 1) * x_items_cell;
    };
    if (total > 0) next_segment(total);
    for (int f = 0; f < total; ++f) {
        while (x_have < x_need) { mbar_wait(xbar, 0u); xbar += 8; x_have += stage_items; }
        if (threadIdx.x == 0 && f == 0) NVFP4_TRACE(3);
        if (f == 0) NVFP4_CLK(11);
        mbar_wait(bar, phase);
        if (f == 0) NVFP4_CLK(12);

        if (threadIdx.x == 0 && f < 3) NVFP4_TRACE(4 + f);
        if (lane == 0 && f == 1) NVFP4_TRACE(40 + warp);

#pragma unroll
        for (int hc = 0; hc < CELL_VECS / 4; ++hc) {                       // half cells: 8 scales, 4 vectors
            float sw[R][8];
            uint64_t swp[R][4];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const uint2 sc = *reinterpret_cast<const uint2*>(st + r * CELL_BYTES + CELL_CODES + lane * (2 * CELL_VECS) + hc * 8);
                const float2 f0s = e4m3x2_to_float2((uint16_t)(sc.x & 0xFFFFu));
                const float2 f1s = e4m3x2_to_float2((uint16_t)(sc.x >> 16));
                const float2 f2s = e4m3x2_to_float2((uint16_t)(sc.y & 0xFFFFu));
                const float2 f3s = e4m3x2_to_float2((uint16_t)(sc.y >> 16));
                sw[r][0] = f0s.x; sw[r][1] = f0s.y; sw[r][2] = f1s.x; sw[r][3] = f1s.y;
                sw[r][4] = f2s.x; sw[r][5] = f2s.y; sw[r][6] = f3s.x; sw[r][7] = f3s.y;
                if (MODE != KMODE_W4A16) {
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        swp[r][q] = pack2u(__float_as_uint(sw[r][2 * q]), __float_as_uint(sw[r][2 * q + 1]));
                }
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {                                  // 32-k vectors of this lane
                uint4 wv[R];
#pragma unroll
                for (int r = 0; r < R; ++r)
                    wv[r] = *reinterpret_cast<const uint4*>(st + r * CELL_BYTES + (hc * 4 + j) * 512 + lane * 16);
                const uint8_t* xbp = xlane + (size_t)(hc * 4 + j) * xstep;
                if (MODE == KMODE_W4A4_I8)     block_pair_w4a4<M, R>(lut, wv, xbp, swp, j, accp);
                else if (MODE == KMODE_W4A4_H) block_pair_w4a4_h<M, R>(wv, xbp, swp, j, accp);
                else                           block_pair_w4a16<M, R>(wv, xbp, sw, j, acc);
            }
        }
        xlane += CELL_VECS * xstep;
        x_need += x_items_cell;

        // every lane has read the stage -> lane 0 requests the next cell of the share into it
        __syncwarp();
        if (leader && p_count < total) issue();
        st += STAGE_BYTES; bar += 8;
        if (st == st_end) { st = ring; bar -= (uint32_t)S * 8; phase ^= 1u; }

        if (--seg_left == 0) {                                              // segment finished
            if (MODE != KMODE_W4A16) {
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int m = 0; m < M; ++m) {
                        const float2 two = unpack2(accp[r][m]);
                        acc[r][m] = two.x + two.y;
                        accp[r][m] = 0ull;
                    }
            }
            float gs = gw_raw;
            if (MODE == KMODE_W4A4_I8) gs = (gs * (fused ? *reinterpret_cast<volatile float*>(gx_slot) : gx_raw)) * 0.25f;   // ints are 2*e
            if (MODE == KMODE_W4A4_H)  gs = gs * (fused ? *reinterpret_cast<volatile float*>(gx_slot) : gx_raw);
            if (!hdr_known) { mbar_wait(hdr_bar, 0u); hdr_known = true; }   // (long complete by now)
            if (!*blob_flag) gs = __int_as_float(0x7FC00000);
            const int left = total - f - 1;
            if (seg_in_a) {
                finish_leftover_cell<M, R>(p, c, acc, aslots, hand, hbars, cnt, warp + a_k * W, lane, part, rsub, rpt, gs);
                ++a_k;
            } else {
                const bool whole = (seg_cell0 == 0) && (seg_len == ncw);
                finish_segment<M, R>(p, c, acc, slots, hand, hbars, cnt, bstart, c_ul, whole, seg_first,
                                     warp, lane, part, rsub, rpt, gs);
                seg_first = false;
            }
            if (left > 0) next_segment(left);
#pragma unroll
            for (int r = 0; r < R; ++r)
#pragma unroll
                for (int m = 0; m < M; ++m) acc[r][m] = 0.0f;
        }
    }
    NVFP4_CLK(14);
    NVFP4_CLK_FLUSH;
    if (lane == 0 && (warp == 0 || warp == W - 1)) NVFP4_TRACE(warp == 0 ? 7 : 14);
    if (lane == 0) NVFP4_TRACE(16 + warp);
}

}  // namespace nvfp4
