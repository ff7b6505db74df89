// tc_common.cuh -- pieces shared by the tensor-core kernels (gemm_tc.cu: W4A4 block-scaled MMA; gemm_tc16.cu: W4A16):
// geometry of the tensor-core weight blob and thin wrappers around the tcgen05 / TMEM PTX instructions.
#pragma once
#include "nvfp4_common.cuh"

namespace nvfp4 {

constexpr int TC_TILE_N      = 128;                     // weight rows per tile = TMEM lanes
constexpr int TC_STAGE_K     = 256;                     // k per stage = 4 MMAs of K = 64
constexpr int TC_CODE_BYTES  = TC_TILE_N * TC_STAGE_K / 2;            // 16384
constexpr int TC_SF_BYTES    = 4 * 512;                               // 2048
constexpr int TC_STAGE_BYTES = TC_CODE_BYTES + TC_SF_BYTES;           // 18432
constexpr uint32_t TC_BLOB_MAGIC = 0x5446564Eu;         // "NVFT"

__host__ __device__ inline int tc_tiles(int N) { return (N + TC_TILE_N - 1) / TC_TILE_N; }
__host__ __device__ inline int tc_xrec_bytes(int MT) { return MT * 128 + TC_SF_BYTES; }
// `interleaved` (fused gate_up weights, N = 2I): tile t holds gate rows [64t, 64t+64) in its rows 0..63 and the matching up
// rows [I + 64t, I + 64t + 64) in its rows 64..127, so that one tile's epilogue owns both factors of SiLU(gate) * up
__host__ __device__ inline uint4 tc_header_words(int N, int K, int interleaved = 0) {
    return make_uint4(TC_BLOB_MAGIC, ((uint32_t)NVFP4_ABI_VERSION << 16) | (interleaved ? 0x7Du : 0x7Cu), (uint32_t)N, (uint32_t)K);
}
// canonical weight row held by row r of tile `tile`
__host__ __device__ inline int tc_source_row(int tile, int r, int N, int interleaved) {
    if (!interleaved) return tile * TC_TILE_N + r;
    return r < 64 ? tile * 64 + r : N / 2 + tile * 64 + (r - 64);
}

// ---- tcgen05 / TMEM wrappers (PTX ISA "tcgen05" family; B200 guide sec. 1-2) ---------------------------------------
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {           // whole warp
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {            // whole warp
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// arrives on `bar` once every tcgen05 operation issued so far by this thread has completed
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// 32 rows x 16 bytes of shared memory -> 4 TMEM columns, replicated into the four 32-lane sub-partitions
__device__ __forceinline__ void tc_cp_sf(uint32_t taddr, uint64_t sdesc) {
    asm volatile("tcgen05.cp.cta_group::1.32x128b.warpx4 [%0], %1;" ::"r"(taddr), "l"(sdesc) : "memory");
}
__device__ __forceinline__ void tc_mma_nvf4(uint32_t d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t sfa,
                                            uint32_t sfb, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %6, 0;\n"
        "tcgen05.mma.cta_group::1.kind::mxf4nvf4.block_scale.scale_vec::4X [%0], %1, %2, %3, [%4], [%5], p;\n"
        "}\n" ::"r"(d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(sfa), "r"(sfb), "r"(accumulate) : "memory");
}
// this thread's TMEM lane (32*(warp%4) + lane), 8 consecutive 32-bit columns
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_plain(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// shared-memory matrix descriptor, no swizzle, K-major: core matrix = 8 rows x 16 bytes (128 contiguous bytes);
// SBO = byte distance between 8-row groups, LBO = byte distance between 16-byte chunks along K
__device__ __forceinline__ uint64_t tc_smem_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) |
           (1ull << 46);                                 // bits [46,48) = descriptor version 1 (sm_100)
}
__device__ __forceinline__ uint64_t tc_desc(uint32_t lo, uint32_t hi) {
    uint64_t d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "r"(lo), "r"(hi));
    return d;
}
__device__ __forceinline__ bool elect_one() {                 // one lane of the (converged) warp
    uint32_t pred;
    asm volatile("{\n.reg .pred p;\nelect.sync _|p, 0xffffffff;\nselp.u32 %0, 1, 0, p;\n}\n" : "=r"(pred));
    return pred != 0;
}
}  // namespace nvfp4
