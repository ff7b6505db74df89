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
// A lane of the GEMV owns (row r, K part p): lane = p*(32/KP) + r (lanes of one K part are adjacent,
// so their activation loads hit one address per part), KP = 2^i K parts per row inside a warp
// (chosen per weight shape by layout_kparts, or given explicitly to nvfp4_repack_weight_kp).
// A "cell" is what one warp consumes in CELL_VECS = 8 128-bit loads per lane: 32/KP weight rows x
// 256*KP consecutive k:
//   bytes [0,4096)    codes:  vector j (0..7), lane (r,p) -> 16 B = the 32 k starting at
//                             cell_k0 + (j*KP + p)*32 of row tile_row0 + r
//   bytes [4096,4608) scales: lane (r,p) -> 16 B = the E4M3 scales of those 8 x 2 blocks (j-major)
// Blob = 128-byte header, then the cells in [tile = n/(32/KP)][cell = k/(256*KP)] order, so one warp
// streams a contiguous run.
constexpr int CELL_VECS   = 8;                          // 128-bit code vectors per lane and cell
constexpr int CELL_CODES  = CELL_VECS * 512;            // 4096
constexpr int CELL_SCALES = CELL_VECS * 64;             // 512
constexpr int CELL_BYTES  = CELL_CODES + CELL_SCALES;   // 4608 = 0.5625 B per weight

// Versioned blob header (the only persistent artefact of the library).  The GEMV
// compares the first four words with what its launch expects and writes NaN outputs on a mismatch.
constexpr int      BLOB_HEADER_BYTES = 128;             // keeps the cells 128-byte aligned (512 measured no faster)
constexpr uint32_t BLOB_MAGIC        = 0x3446564Eu;     // "NVF4"
struct BlobHeader {
    uint32_t magic;          // BLOB_MAGIC
    uint32_t version_kp;     // NVFP4_ABI_VERSION << 16 | KP
    uint32_t N, K;
    uint32_t cell_bytes, ntiles, ncells, reserved;
};
__host__ __device__ inline uint4 blob_header_words(int N, int K, int kp) {
    return make_uint4(BLOB_MAGIC, ((uint32_t)NVFP4_ABI_VERSION << 16) | (uint32_t)kp, (uint32_t)N, (uint32_t)K);
}

struct Layout {
    int kp;         // K parts per row inside a warp (1, 2, 4, 8, 16 or 32)
    int rpt;        // weight rows per tile = 32 / kp
    int cell_k;     // k per cell = 32 * CELL_VECS * kp
    int ntiles;     // ceil(N / rpt)
    int ncells;     // ceil(K / cell_k)
};

__host__ __device__ inline Layout make_layout(int N, int K, int kp) {
    Layout L;
    L.kp = kp; L.rpt = 32 / kp; L.cell_k = 32 * CELL_VECS * kp;
    L.ntiles = (N + L.rpt - 1) / L.rpt;
    L.ncells = (K + L.cell_k - 1) / L.cell_k;
    return L;
}

// Default K parts for a weight shape: the smallest power of two that yields >= 296 (= 2 per SM) tiles of
// at most 32 cells each, among those whose K padding costs at most 3% more than KP = 1 does.  (Balance
// across and inside the SMs comes from the flat-stream split of the GEMV, so few K parts are needed;
// fewer parts = more uniform activation loads.)
__host__ __device__ inline int layout_kparts(int N, int K) {
    const long long ck1 = 32 * CELL_VECS;
    const long long pad1 = ((K + ck1 - 1) / ck1) * ck1;
    int best = 1;
    for (int kp = 1; kp <= 32; kp *= 2) {
        const long long ck = ck1 * kp;
        const long long padk = ((K + ck - 1) / ck) * ck;
        if (padk * 100 > pad1 * 103) break;
        best = kp;
        // enough tiles (2 per SM), and rows short enough (<= 32 cells) that a row tile is shared by few warps
        if ((long long)N * kp >= 296LL * 32 && padk / ck <= 32) break;
    }
    return best;
}

// ---- division by a launch-constant divisor without the ~25-instruction udiv sequence ----------------------------------
// q = floor(n / d) for 0 <= n < 2^31:  mul = ceil(2^(31+L) / d), L = ceil(log2 d);  q = (n * mul) >> (31 + L).
// (n*mul/2^(31+L) = n/d + n*e/2^(31+L) with 0 <= e < 1, and n*e/2^(31+L) < 2^-L <= 1/d: the floor cannot move.)
struct FastDiv { uint32_t mul; uint32_t sh; };
__host__ __device__ inline FastDiv fastdiv_make(uint32_t d) {
    FastDiv f;
    if (d == 0) d = 1;
    uint32_t L = 0;
    while ((1ull << L) < d) ++L;
    f.mul = (uint32_t)(((1ull << (31 + L)) + d - 1) / d);
    f.sh = 31 + L;
    return f;
}
__host__ __device__ __forceinline__ uint32_t fastdiv(uint32_t n, const FastDiv& f) {
    return (uint32_t)(((unsigned long long)n * f.mul) >> f.sh);
}

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

// one 32-bit word of eight E2M1 codes -> four f16x2 (codes 0,1 | 2,3 | 4,5 | 6,7), exact.  The vector mov lets the
// conversions take their source byte through the instruction's byte selector (F2FP ... R.B1): no shift / mask per byte.
__device__ __forceinline__ void cvt_word_e2m1(uint32_t w, uint32_t (&h)[4]) {
    asm("{.reg .b8 t0,t1,t2,t3; mov.b32 {t0,t1,t2,t3}, %4;\n"
        "cvt.rn.f16x2.e2m1x2 %0, t0; cvt.rn.f16x2.e2m1x2 %1, t1; cvt.rn.f16x2.e2m1x2 %2, t2; cvt.rn.f16x2.e2m1x2 %3, t3;}"
        : "=r"(h[0]), "=r"(h[1]), "=r"(h[2]), "=r"(h[3]) : "r"(w));
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

// ---- programmatic dependent launch (PDL) --------------------------------------------------
// Every kernel of the path is launched with cudaLaunchAttributeProgrammaticStreamSerialization, so
// it may start while its stream predecessor is still running.  pdl_wait() blocks until the
// predecessor grid has completed and its writes are visible: it must precede every access to
// memory the predecessor may write or read-before-overwrite (activations, outputs, workspace).
// Work on constant data (the repacked weights) is issued BEFORE it, which is the point.
// pdl_launch_dependents() is called only AFTER pdl_wait(), so at most two consecutive kernels overlap.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

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
