// nvfp4_common.cuh -- device helpers shared by the sm_100a kernels of this library
// (PRODUCT code: shares nothing with oracle/).
//
// Format (PAPER.md:344-349 Table 7, :359): E2M1 4-bit elements, one E4M3 scale per
// 16 consecutive K, one FP32 global scale per tensor.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/nvfp4.h"

#if defined(__CUDA_ARCH__) && !defined(__CUDA_ARCH_FEAT_SM100_ALL) && !defined(__CUDA_ARCH_FEAT_SM101_ALL) && !defined(__CUDA_ARCH_FEAT_SM103_ALL)
#error "compile with -gencode arch=compute_100a,code=sm_100a"
#endif

namespace nvfp4 {

// ---- repacked weight blob geometry -------------------------
// A "cell" = 32 weight rows (one per lane) x 128 consecutive k:
//   bytes [0,2048)    codes:  vector j (0..3), lane l -> 16 B = k in [32j, 32j+32) of row l
//   bytes [2048,2304) scales: lane l -> 8 B = the 8 E4M3 block scales of row l
// Blob = cells in [tile = n/32][chunk = k/128] order, so one warp streams a contiguous run.
constexpr int TILE_ROWS   = 32;
constexpr int CHUNK_K     = 128;
constexpr int CELL_CODES  = TILE_ROWS * CHUNK_K / 2;   // 2048
constexpr int CELL_SCALES = TILE_ROWS * CHUNK_K / 16;  // 256
constexpr int CELL_BYTES  = CELL_CODES + CELL_SCALES;  // 2304

__host__ __device__ inline int n_tiles(int N)  { return (N + TILE_ROWS - 1) / TILE_ROWS; }
__host__ __device__ inline int n_chunks(int K) { return (K + CHUNK_K - 1) / CHUNK_K; }

// ---- conversions ------------------------------------------------------------------------
// E4M3 byte pair -> two FP32 (exact): F2FP.E4M3.UNPACK then two f16->f32.
__device__ __forceinline__ float2 e4m3x2_to_float2(uint16_t v) {
    uint32_t h2;
    asm("cvt.rn.f16x2.e4m3x2 %0, %1;" : "=r"(h2) : "h"(v));
    float2 r;
    asm("{.reg .b16 lo, hi; mov.b32 {lo, hi}, %2; cvt.f32.f16 %0, lo; cvt.f32.f16 %1, hi;}"
        : "=f"(r.x), "=f"(r.y) : "r"(h2));
    return r;
}
__device__ __forceinline__ float e4m3_to_float(uint8_t v) {
    return e4m3x2_to_float2((uint16_t)v).x;
}

// FP32 -> E4M3 byte, round-to-nearest-even, saturating at 448 (input must be >= 0, not NaN).
__device__ __forceinline__ uint8_t float_to_e4m3_rn_sat(float u) {
    uint16_t r;
    asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(0.0f), "f"(u));
    return (uint8_t)(r & 0xFF);
}

// two FP32 -> one byte of two E2M1 codes (lo in the low nibble), RNE, saturating at +-6.
__device__ __forceinline__ uint8_t float2_to_e2m1x2(float lo, float hi) {
    uint16_t r;
    asm("{.reg .b8 t; cvt.rn.satfinite.e2m1x2.f32 t, %1, %2; cvt.u16.u8 %0, t;}"
        : "=h"(r) : "f"(hi), "f"(lo));
    return (uint8_t)r;
}

// one byte of two E2M1 codes -> f16x2 (lo nibble in the low half), exact.
__device__ __forceinline__ uint32_t e2m1x2_to_f16x2(uint32_t byte) {
    uint32_t r;
    asm("{.reg .b8 t; cvt.u8.u32 t, %1; cvt.rn.f16x2.e2m1x2 %0, t;}" : "=r"(r) : "r"(byte));
    return r;
}

__device__ __forceinline__ float bf16_bits_to_float(uint16_t b) {
    return __uint_as_float(((uint32_t)b) << 16);
}
// FP32 -> BF16 bits, round-to-nearest-even (finite inputs).
__device__ __forceinline__ uint16_t float_to_bf16_rn(float f) {
    uint16_t r;
    asm("cvt.rn.bf16.f32 %0, %1;" : "=h"(r) : "f"(f));
    return r;
}

// ---- mbarrier / bulk-copy (TMA) wrappers ------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// 1-D bulk copy global -> shared, completion counted in bytes on `bar` (SASS: UBLKCP).
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

}  // namespace nvfp4
