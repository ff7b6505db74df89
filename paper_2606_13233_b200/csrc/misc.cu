// misc.cu -- SiLU*mul glue of the decode chain (step a8, BASELINE.json configs[4]; not part of
// the paper's kernel):  h[m,j] = silu(gu[m,j]) * gu[m,I+j],  FP32 math, BF16 RNE output.
#include "nvfp4_common.cuh"
#include "nvfp4_internal.h"

namespace nvfp4 {

__global__ void __launch_bounds__(256) silu_mul_kernel(const uint16_t* __restrict__ gu, int M, int I,
                                                       uint16_t* __restrict__ h) {
    const int vec_per_row = I >> 3;                                  // 8 BF16 per 16-byte vector
    const int total = M * vec_per_row;
    for (int v = blockIdx.x * blockDim.x + threadIdx.x; v < total; v += gridDim.x * blockDim.x) {
        const int m = v / vec_per_row, j = (v - m * vec_per_row) * 8;
        const uint4 g = __ldg(reinterpret_cast<const uint4*>(gu + (int64_t)m * 2 * I + j));
        const uint4 u = __ldg(reinterpret_cast<const uint4*>(gu + (int64_t)m * 2 * I + I + j));
        const uint32_t gw[4] = {g.x, g.y, g.z, g.w}, uw[4] = {u.x, u.y, u.z, u.w};
        uint32_t out[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float g0 = __uint_as_float(gw[i] << 16), g1 = __uint_as_float(gw[i] & 0xFFFF0000u);
            const float u0 = __uint_as_float(uw[i] << 16), u1 = __uint_as_float(uw[i] & 0xFFFF0000u);
            const float h0 = __fdiv_rn(g0, 1.0f + expf(-g0)) * u0;
            const float h1 = __fdiv_rn(g1, 1.0f + expf(-g1)) * u1;
            out[i] = (uint32_t)float_to_bf16_rn(h0) | ((uint32_t)float_to_bf16_rn(h1) << 16);
        }
        *reinterpret_cast<uint4*>(h + (int64_t)m * I + j) = make_uint4(out[0], out[1], out[2], out[3]);
    }
}

cudaError_t launch_silu_mul(const void* gu, int M, int I, void* h, cudaStream_t st) {
    const int total = M * (I / 8);
    int grid = (total + 255) / 256;
    if (grid > 148 * 8) grid = 148 * 8;
    if (grid < 1) grid = 1;
    silu_mul_kernel<<<grid, 256, 0, st>>>(static_cast<const uint16_t*>(gu), M, I, static_cast<uint16_t*>(h));
    return cudaGetLastError();
}

}  // namespace nvfp4
