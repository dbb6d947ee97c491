// pack_weights.cu -- offline re-layout of one layer's weights (step a0; PAPER.md L123:
// all transforms and weight formats are "pre-processed offline").  Not on the timed path.
// Blob sections and their reasons: packed_layout.h.
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "packed_layout.h"

namespace twq {

// one thread: 8 codes of one row (8 bytes in) -> 4 bytes of the (n/8, g) block, row n%8
__global__ void pack_codes_kernel(const int8_t* __restrict__ Rq, uint8_t* __restrict__ R4, int N, int K, int G) {
    const long long n_words = static_cast<long long>(N) * (K / 8);
    const int wpr = K / 8, ng = K / G;
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < n_words;
         i += static_cast<long long>(gridDim.x) * blockDim.x) {
        const uint2 v = __ldg(reinterpret_cast<const uint2*>(Rq) + i);
        uint32_t out = 0;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            out |= ((v.x >> (8 * b)) & 0xFu) << (4 * b);
            out |= ((v.y >> (8 * b)) & 0xFu) << (16 + 4 * b);
        }
        const int n = static_cast<int>(i / wpr), k0 = static_cast<int>(i - static_cast<long long>(n) * wpr) * 8;
        const int g = k0 / G, b0 = (k0 - g * G) >> 1;
        const size_t o = (static_cast<size_t>(n >> 3) * ng + g) * (4 * static_cast<size_t>(G)) + (n & 7) * (G / 2) + b0;
        *reinterpret_cast<uint32_t*>(R4 + o) = out;
    }
}

// sw [N][ng] f16 -> sw16 [N/8][ng][8] f16
__global__ void pack_scales_kernel(const __half* __restrict__ sw, __half* __restrict__ sw16, int N, int ng) {
    const long long total = static_cast<long long>(N) * ng;
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < total;
         i += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int n = static_cast<int>(i / ng), g = static_cast<int>(i - static_cast<long long>(n) * ng);
        sw16[(static_cast<size_t>(n >> 3) * ng + g) * 8 + (n & 7)] = sw[i];
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

// L1 [K][r] f16 -> L1D [K/32][r][32] f16 (a 32 x 32 tile transpose per block: both sides coalesced)
__global__ void slab_l1_kernel(const uint16_t* __restrict__ L1, uint16_t* __restrict__ L1D, int K, int r) {
    __shared__ uint16_t tile[32][34];
    const int j0 = blockIdx.x * 32, k0 = blockIdx.y * 32;      // K % 32 == 0; r % 16 == 0
    for (int kk = threadIdx.y; kk < 32; kk += blockDim.y) {
        const int j = j0 + threadIdx.x;
        if (j < r) tile[kk][threadIdx.x] = L1[static_cast<size_t>(k0 + kk) * r + j];
    }
    __syncthreads();
    for (int jj = threadIdx.y; jj < 32; jj += blockDim.y) {
        const int j = j0 + jj;
        if (j < r) L1D[(static_cast<size_t>(k0 >> 5) * r + j) * 32 + threadIdx.x] = tile[threadIdx.x][jj];
    }
}

cudaError_t launch_pack_weights(const int8_t* Rq, const void* sw, const void* L1, const void* L2, int N, int K, int r,
                                int G, void* packed, cudaStream_t stream, int* launches) {
    const PackedLayout lay = packed_layout(N, K, r, G);
    uint8_t* base = static_cast<uint8_t*>(packed);
    const long long n_words = static_cast<long long>(N) * K / 8;
    long long blocks = (n_words + 255) / 256;
    if (blocks > 148 * 32) blocks = 148 * 32;
    pack_codes_kernel<<<static_cast<unsigned>(blocks), 256, 0, stream>>>(Rq, base + lay.off_r4, N, K, G);
    const int ng = K / G;
    long long sblocks = (static_cast<long long>(N) * ng + 255) / 256;
    if (sblocks > 148 * 32) sblocks = 148 * 32;
    pack_scales_kernel<<<static_cast<unsigned>(sblocks), 256, 0, stream>>>(
        static_cast<const __half*>(sw), reinterpret_cast<__half*>(base + lay.off_sw16), N, ng);
    int n = 2;
    if (r > 0) {
        dim3 tb(32, 8);
        // L1 [K][r] -> L1T [r][K]
        transpose16_kernel<<<dim3((r + 31) / 32, (K + 31) / 32), tb, 0, stream>>>(
            static_cast<const uint16_t*>(L1), reinterpret_cast<uint16_t*>(base + lay.off_l1t), K, r);
        // L1 [K][r] -> L1D [K/32][r][32]
        slab_l1_kernel<<<dim3((r + 31) / 32, K / 32), tb, 0, stream>>>(
            static_cast<const uint16_t*>(L1), reinterpret_cast<uint16_t*>(base + lay.off_l1d), K, r);
        // L2 [r][N] -> L2T [N][r]
        transpose16_kernel<<<dim3((N + 31) / 32, (r + 31) / 32), tb, 0, stream>>>(
            static_cast<const uint16_t*>(L2), reinterpret_cast<uint16_t*>(base + lay.off_l2t), r, N);
        n += 3;
    }
    if (launches) *launches = n;
    return cudaGetLastError();
}

// ---- q4lr blob (both low-rank factors 4-bit): U and V sections of packed_layout.h
// one thread: one byte (two codes) of U.  Uq [r][K] int8 -> U [K/G][r][G/2] (+ r scales behind each group)
__global__ void pack_u_kernel(const int8_t* __restrict__ Uq, const __half* __restrict__ su, uint8_t* __restrict__ U,
                              int r, int K, int G) {
    const int ng = K / G;
    const size_t gb = static_cast<size_t>(r) * (G / 2) + static_cast<size_t>(r) * 2;
    const long long total = static_cast<long long>(r) * (K / 2);
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < total;
         i += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int j = static_cast<int>(i / (K / 2)), kb = static_cast<int>(i - static_cast<long long>(j) * (K / 2));
        const int g = kb / (G / 2), b = kb - g * (G / 2);
        const int8_t lo = Uq[static_cast<size_t>(j) * K + 2 * kb], hi = Uq[static_cast<size_t>(j) * K + 2 * kb + 1];
        U[g * gb + static_cast<size_t>(j) * (G / 2) + b] = static_cast<uint8_t>((lo & 0xF) | ((hi & 0xF) << 4));
    }
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < static_cast<long long>(r) * ng;
         i += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int j = static_cast<int>(i / ng), g = static_cast<int>(i - static_cast<long long>(j) * ng);
        reinterpret_cast<__half*>(U + g * gb + static_cast<size_t>(r) * (G / 2))[j] = su[i];
    }
}

// one thread: one stored byte of V.  Vq [N][r] int8 -> V [N/8][nh][8][grs/2], zero beyond gr codes; sv [N][nh] -> [N/8][nh][8]
__global__ void pack_v_kernel(const int8_t* __restrict__ Vq, const __half* __restrict__ sv, uint8_t* __restrict__ V,
                              __half* __restrict__ sv16, int N, int r, int gr, int grs, int nh) {
    const int rb = grs / 2;
    const long long total = static_cast<long long>(N) * nh * rb;
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < total;
         i += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int b = static_cast<int>(i % rb);
        const long long row = i / rb;                       // (tile, h, c)
        const int c = static_cast<int>(row & 7), h = static_cast<int>((row >> 3) % nh), t = static_cast<int>((row >> 3) / nh);
        uint8_t out = 0;
        if (2 * b < gr) {
            const int8_t* src = Vq + static_cast<size_t>(t * 8 + c) * r + h * gr + 2 * b;
            out = static_cast<uint8_t>((src[0] & 0xF) | ((src[1] & 0xF) << 4));
        }
        V[i] = out;
    }
    for (long long i = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; i < static_cast<long long>(N) * nh;
         i += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int n = static_cast<int>(i / nh), h = static_cast<int>(i - static_cast<long long>(n) * nh);
        sv16[(static_cast<size_t>(n >> 3) * nh + h) * 8 + (n & 7)] = sv[i];
    }
}

cudaError_t launch_pack_weights_q4lr(const int8_t* Rq, const void* sw, const int8_t* Uq, const void* su, const int8_t* Vq,
                                     const void* sv, int N, int K, int r, int G, void* packed, cudaStream_t stream,
                                     int* launches) {
    const PackedLayoutQ4 lay = packed_layout_q4lr(N, K, r, G);
    uint8_t* base = static_cast<uint8_t*>(packed);
    const long long n_words = static_cast<long long>(N) * K / 8;
    long long blocks = (n_words + 255) / 256;
    if (blocks > 148 * 32) blocks = 148 * 32;
    pack_codes_kernel<<<static_cast<unsigned>(blocks), 256, 0, stream>>>(Rq, base + lay.off_r4, N, K, G);
    const int ng = K / G;
    long long sblocks = (static_cast<long long>(N) * ng + 255) / 256;
    if (sblocks > 148 * 32) sblocks = 148 * 32;
    pack_scales_kernel<<<static_cast<unsigned>(sblocks), 256, 0, stream>>>(
        static_cast<const __half*>(sw), reinterpret_cast<__half*>(base + lay.off_sw16), N, ng);
    long long ub = (static_cast<long long>(r) * (K / 2) + 255) / 256;
    if (ub > 148 * 32) ub = 148 * 32;
    pack_u_kernel<<<static_cast<unsigned>(ub), 256, 0, stream>>>(Uq, static_cast<const __half*>(su), base + lay.off_u, r, K, G);
    long long vb = (static_cast<long long>(N) * lay.nh * (lay.grs / 2) + 255) / 256;
    if (vb > 148 * 32) vb = 148 * 32;
    pack_v_kernel<<<static_cast<unsigned>(vb), 256, 0, stream>>>(Vq, static_cast<const __half*>(sv), base + lay.off_v,
                                                                 reinterpret_cast<__half*>(base + lay.off_sv16), N, r, lay.gr,
                                                                 lay.grs, lay.nh);
    if (launches) *launches = 4;
    return cudaGetLastError();
}

}  // namespace twq
