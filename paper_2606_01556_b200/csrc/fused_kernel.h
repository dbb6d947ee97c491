// fused_kernel.h -- host-side interface between the C ABI (twq_api.cu) and the fused
// dual-branch kernel (fused_kernel.cu).  Plain structs; all launch planning is host arithmetic.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace twq {

// Work decomposition and shared-memory plan of one twq_dual_linear call (host-computed).
struct FusedPlan {
    int TN;                  // tokens per tile (MMA N): 16 / 32 / 64 / 128
    int cs;                  // CTAs per cluster; the cluster shares the stage-1 product H through DSMEM
    int splits;              // K splits (decode-shaped calls)
    int g_per_split;         // residual groups per split
    int n_tiles, m_tiles;    // 128-channel tiles, TN-token tiles
    int n_blocks;            // n_tiles / cs
    int units;               // splits * m_tiles * n_blocks  (one unit = cs n-tiles of one m-tile, one K split)
    int nclusters;           // persistent clusters; cluster c owns units [c*units/nclusters, (c+1)*units/nclusters)
    int nsp, nsu, ns1;       // ring depths: packed (TMA), expanded (MMA operands), stage-1
    int alias;               // 1: the stage-1 ring and the FP32 H partial overlay the residual rings
    int pair;                // 1: CTA pairs (cta_group::2): ranks 2i / 2i+1 of a cluster share one M = 256 MMA
    int ystage;              // 1: the epilogue parks the finished tile in shared memory and bulk-copies it out (async)
    int off_H, off_L2T, off_U, off_P, off_S1, off_Hpart, off_sx, off_bar, off_Y;
    int smem_bytes;
    int tmem_cols;           // 256 or 512
};

struct FusedParams {
    int M, N, K, r, ng;
    int ldy, ydt;            // ydt: 0 bf16, 1 fp16, 2 fp32
    const float* sx;         // [M][ng] activation group scales
    const float* swT;        // [ng][N] weight group scales (FP32, transposed)
    void* Y;                 // [M][ldy]
    int32_t* dbgP;           // NULL or [M][ng][N]
    float* ws_part;          // split-K partials [splits][M][N] (splits > 1 only)
    unsigned* ws_ctr;        // split-K tile counters [m_tiles][n_tiles], zero between calls
    FusedPlan plan;
};

struct FusedMaps {
    CUtensorMap W, Xq, X, L1T, L2T, Y;
};


// Decode-shaped calls (M <= 16): parameters and plan of decode_kernel.cu (host-computed).
struct DecodeParams {
    int M, N, K, r, ng;
    int ldx, ldy, ydt;       // ydt: 0 bf16, 1 fp16, 2 fp32
    int n_tiles;             // N / 16
    int cs, grid;            // CTAs per cluster, CTAs in the grid (a multiple of cs)
    int T, P;                // 16-channel tiles per CTA, K-parts per tile
    int off_res, off_hpart, off_h, off_ylr, off_sx, off_xs, smem_bytes;
    int ncl_k;               // > 1: stage 1 splits K over ALL ncl_k clusters (L1T read once per call); partials meet in ws_h
    float* ws_h;             // [ncl_k][16][r] FP32 cluster-level partials of H (caller's workspace)
    unsigned* ws_ctr;        // grid barrier counter (zero between calls)
    const uint8_t* R4;       // [N][K/2]
    const float* swT;        // [ng][N]
    const void* L1T;         // [r][K] f16
    const void* L2T;         // [N][r] f16
    const void* X;           // [M][ldx] bf16
    const uint8_t* Xq;       // [M][K/2]
    const float* sx;         // [M][ng]
    void* Y;
    int32_t* dbgP;
};
bool decode_make_plan(int M, int N, int K, int r, int G, int num_sms, DecodeParams* out);
inline size_t decode_workspace_bytes(const DecodeParams& p) {
    return p.ncl_k > 1 ? 256 + ((static_cast<size_t>(p.ncl_k) * 16 * p.r * sizeof(float) + 255) & ~static_cast<size_t>(255)) : 0;
}
cudaError_t launch_decode(const DecodeParams& p, int G, cudaStream_t stream);

// Fills `plan` for a shape; returns false if the shape cannot be planned (never for valid ABI shapes).
bool fused_make_plan(int M, int N, int K, int r, int G, int num_sms, FusedPlan* plan);
cudaError_t launch_fused(const FusedMaps& maps, const FusedParams& p, int G, cudaStream_t stream);

cudaError_t launch_quantize_act(const void* X, int M, int K, int ldx, const float* tinv, int G, uint8_t* Xq,
                                float* sx, cudaStream_t stream);
cudaError_t launch_pack_weights(const int8_t* Rq, const void* sw, const void* L1, const void* L2, int N, int K, int r,
                                int G, void* packed, cudaStream_t stream, int* launches);

}  // namespace twq
