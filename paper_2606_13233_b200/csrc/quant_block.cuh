// quant_block.cuh -- the per-block arithmetic of the NVFP4 activation quantizer (R1/R2), shared by
// quantize.cu (canonical codes + scales) and by the GEMV's fused-quantization stagers (f16 records).
// Every op is ONE binary32 RNE operation; never compile with -use_fast_math.
#pragma once
#include "nvfp4_common.cuh"

namespace nvfp4 {

__device__ __forceinline__ uint32_t absmax_bits16(const uint4& a, const uint4& b) {
    // max over the sixteen 15-bit magnitudes (BF16 magnitudes order like integers)
    uint32_t m = 0;
    const uint32_t w[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        uint32_t v = w[i] & 0x7FFF7FFFu;
        m = max(m, max(v & 0xFFFFu, v >> 16));
    }
    return m;
}

// scale byte and divisor of a block: t = a_b/6; u = t/g; sc = E4M3_RNE(min(u, 448)); d = g * dec(sc)
__device__ __forceinline__ void block_scale(uint32_t ab_bits, float g, uint8_t& sc, float& d) {
    const float a_b = __uint_as_float(ab_bits << 16);
    const float t = __fdiv_rn(a_b, 6.0f);
    const float u = __fdiv_rn(t, g);
    sc = float_to_e4m3_rn_sat(fminf(u, 448.0f));
    d = __fmul_rn(g, e4m3_to_float(sc));
}

}  // namespace nvfp4
