// repack.cu -- offline weight repack (step a0) and its exact inverse.  Pure byte permutation:
// canonical codes[N,K/2] + scales[N,K/16]  <->  blob = 128-byte versioned header + 4608-byte cells
// (nvfp4_common.cuh; the K-part count KP of the layout is recorded in the header).
// Padding rows (n >= N) and padding k (k >= K) are zero codes / zero scales.
//
// Both launches end with an empty, ordinary (non-PDL) kernel: the GEMV is launched with programmatic
// stream serialization and starts reading the blob BEFORE its griddepcontrol.wait, so its stream
// predecessor must never be the kernel that writes the blob.  With the empty kernel in between, the
// GEMV's predecessor starts only after the repack has completed and flushed.
#include "nvfp4_common.cuh"
#include "nvfp4_internal.h"

namespace nvfp4 {

// one thread per 16-byte code vector of the blob, one per 16-byte scale group
template <bool TO_BLOB>
__global__ void __launch_bounds__(256) repack_kernel(uint8_t* __restrict__ codes, uint8_t* __restrict__ scales,
                                                     int N, int K, Layout L, uint8_t* __restrict__ blob) {
    const int64_t ncells = (int64_t)L.ntiles * L.ncells;
    constexpr int EPC = CELL_VECS * 32 + 32;                // code vectors + scale groups per cell
    const int64_t nvec = ncells * EPC;
    const int64_t rowb = K / 2, rows = K / 16;
    if (TO_BLOB && blockIdx.x == 0 && threadIdx.x < BLOB_HEADER_BYTES / 4) {          // versioned header
        const uint4 w = blob_header_words(N, K, L.kp);
        const uint32_t h[8] = {w.x, w.y, w.z, w.w, (uint32_t)CELL_BYTES, (uint32_t)L.ntiles, (uint32_t)L.ncells, 0u};
        reinterpret_cast<uint32_t*>(blob)[threadIdx.x] = threadIdx.x < 8 ? h[threadIdx.x] : 0u;
    }
    for (int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; v < nvec; v += (int64_t)gridDim.x * blockDim.x) {
        const int64_t cell = v / EPC;
        const int e = (int)(v - cell * EPC);
        const int tile = (int)(cell / L.ncells), ci = (int)(cell - (int64_t)tile * L.ncells);
        uint8_t* cellp = blob + BLOB_HEADER_BYTES + cell * CELL_BYTES;
        const int lane = e & 31;
        const int n = tile * L.rpt + lane % L.rpt, part = lane / L.rpt;      // lane = part * rpt + row
        if (e < CELL_VECS * 32) {
            const int j = e >> 5;
            const int64_t k0 = (int64_t)ci * L.cell_k + (int64_t)(j * L.kp + part) * 32;
            const int64_t b0 = k0 / 2;                          // byte offset inside the canonical row
            uint8_t* bp = cellp + j * 512 + lane * 16;
            for (int i = 0; i < 16; ++i) {
                const bool valid = (n < N) && (b0 + i < rowb);
                if (TO_BLOB) bp[i] = valid ? codes[(int64_t)n * rowb + b0 + i] : (uint8_t)0;
                else if (valid) codes[(int64_t)n * rowb + b0 + i] = bp[i];
            }
        } else {
            uint8_t* sp = cellp + CELL_CODES + lane * (2 * CELL_VECS);
            for (int i = 0; i < 2 * CELL_VECS; ++i) {
                const int j = i >> 1;
                const int64_t s0 = ((int64_t)ci * L.cell_k + (int64_t)(j * L.kp + part) * 32) / 16 + (i & 1);
                const bool valid = (n < N) && (s0 < rows);
                if (TO_BLOB) sp[i] = valid ? scales[(int64_t)n * rows + s0] : (uint8_t)0;
                else if (valid) scales[(int64_t)n * rows + s0] = sp[i];
            }
        }
    }
}

static int repack_grid(const Layout& L) {
    const int64_t nvec = (int64_t)L.ntiles * L.ncells * (CELL_VECS * 32 + 32);
    int64_t g = (nvec + 255) / 256;
    if (g > 148 * 32) g = 148 * 32;
    return (int)g;
}

__global__ void pdl_fence_kernel() {}

cudaError_t launch_repack(const uint8_t* codes, const uint8_t* scales, int N, int K, int kp, void* blob, cudaStream_t st) {
    const Layout L = make_layout(N, K, kp);
    repack_kernel<true><<<repack_grid(L), 256, 0, st>>>(const_cast<uint8_t*>(codes), const_cast<uint8_t*>(scales),
                                                        N, K, L, static_cast<uint8_t*>(blob));
    pdl_fence_kernel<<<1, 32, 0, st>>>();
    return cudaGetLastError();
}

cudaError_t launch_unpack(const void* blob, int N, int K, int kp, uint8_t* codes, uint8_t* scales, cudaStream_t st) {
    const Layout L = make_layout(N, K, kp);
    repack_kernel<false><<<repack_grid(L), 256, 0, st>>>(codes, scales, N, K, L,
                                                         static_cast<uint8_t*>(const_cast<void*>(blob)));
    pdl_fence_kernel<<<1, 32, 0, st>>>();
    return cudaGetLastError();
}

}  // namespace nvfp4
