// pack_weights.cu -- offline re-layout of one layer's weights (step a0; PAPER.md L123:
// all transforms and weight formats are "pre-processed offline").  Not on the timed path.
//
// Blob sections (each 256-byte aligned; offsets from packed_layout.h):
//   R4   [N][K/2] u8    two INT4 codes per byte, low nibble = even k (two's complement)
//   swT  [K/G][N] f32   group scales transposed, so an epilogue warp reads 32 consecutive n
//   L1T  [r][K]   f16   L1 transposed (K-major A operand of the stage-1 MMA)
//   L2T  [N][r]   f16   L2 transposed (K-major A operand of the stage-2 MMA, reduction over r)
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "packed_layout.h"

namespace twq {

__global__ void pack_codes_kernel(const int8_t* __restrict__ Rq, uint8_t* __restrict__ R4, long long n_words) {
    // one thread: 8 codes (8 bytes in) -> 4 bytes out
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < n_words;
         i += static_cast<long long>(gridDim.x) * blockDim.x) {
        const uint2 v = __ldg(reinterpret_cast<const uint2*>(Rq) + i);
        uint32_t out = 0;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            out |= ((v.x >> (8 * b)) & 0xFu) << (4 * b);
            out |= ((v.y >> (8 * b)) & 0xFu) << (16 + 4 * b);
        }
        reinterpret_cast<uint32_t*>(R4)[i] = out;
    }
}

__global__ void pack_scales_kernel(const __half* __restrict__ sw, float* __restrict__ swT, int N, int ng) {
    __shared__ float tile[32][33];
    const int n0 = blockIdx.x * 32, g0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {
        const int n = n0 + j, g = g0 + threadIdx.x;
        if (n < N && g < ng) tile[j][threadIdx.x] = __half2float(sw[static_cast<size_t>(n) * ng + g]);
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {
        const int g = g0 + j, n = n0 + threadIdx.x;
        if (n < N && g < ng) swT[static_cast<size_t>(g) * N + n] = tile[threadIdx.x][j];
    }
}

// out[c][r] = in[r][c] for 16-bit elements
__global__ void transpose16_kernel(const uint16_t* __restrict__ in, uint16_t* __restrict__ out, int rows, int cols) {
    __shared__ uint16_t tile[32][34];
    const int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {
        const int r = r0 + j, c = c0 + threadIdx.x;
        if (r < rows && c < cols) tile[j][threadIdx.x] = in[static_cast<size_t>(r) * cols + c];
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += blockDim.y) {
        const int c = c0 + j, r = r0 + threadIdx.x;
        if (r < rows && c < cols) out[static_cast<size_t>(c) * rows + r] = tile[threadIdx.x][j];
    }
}

cudaError_t launch_pack_weights(const int8_t* Rq, const void* sw, const void* L1, const void* L2, int N, int K, int r,
                                int G, void* packed, cudaStream_t stream, int* launches) {
    const PackedLayout lay = packed_layout(N, K, r, G);
    uint8_t* base = static_cast<uint8_t*>(packed);
    const long long n_words = static_cast<long long>(N) * K / 8;
    long long blocks = (n_words + 255) / 256;
    if (blocks > 148 * 32) blocks = 148 * 32;
    pack_codes_kernel<<<static_cast<unsigned>(blocks), 256, 0, stream>>>(Rq, base + lay.off_r4, n_words);
    const int ng = K / G;
    dim3 tb(32, 8);
    pack_scales_kernel<<<dim3((N + 31) / 32, (ng + 31) / 32), tb, 0, stream>>>(
        static_cast<const __half*>(sw), reinterpret_cast<float*>(base + lay.off_swT), N, ng);
    int n = 2;
    if (r > 0) {
        // L1 [K][r] -> L1T [r][K]
        transpose16_kernel<<<dim3((r + 31) / 32, (K + 31) / 32), tb, 0, stream>>>(
            static_cast<const uint16_t*>(L1), reinterpret_cast<uint16_t*>(base + lay.off_l1t), K, r);
        // L2 [r][N] -> L2T [N][r]
        transpose16_kernel<<<dim3((N + 31) / 32, (r + 31) / 32), tb, 0, stream>>>(
            static_cast<const uint16_t*>(L2), reinterpret_cast<uint16_t*>(base + lay.off_l2t), r, N);
        n += 2;
    }
    if (launches) *launches = n;
    return cudaGetLastError();
}

}  // namespace twq
