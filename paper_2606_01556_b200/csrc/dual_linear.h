// dual_linear.h -- host-side interface between the C ABI (twq_api.cu) and the fused kernel.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace twq {

struct DualParams {
    int M, N, K, r, ng;
    int ldy, ydt;            // ydt: 0 bf16, 1 fp16, 2 fp32
    int g_per_split;         // residual groups handled by one split (grid.z)
    const float* sx;         // [M][ng] activation group scales
    const float* swT;        // [ng][N] weight group scales (FP32, transposed)
    void* Y;                 // [M][ldy]
    int32_t* dbgP;           // NULL or [M][ng][N]
    float* ws_part;          // split-K partials [splits][M][N] (splits > 1 only)
    unsigned* ws_ctr;        // split-K tile counters, zero between calls
};

struct DualMaps {
    CUtensorMap W, Xq, X, L1T, L2T;
};

int dual_pick_tn(int M);
cudaError_t launch_dual_linear(const DualMaps& maps, const DualParams& p, int TN, int G, int splits,
                               cudaStream_t stream);

cudaError_t launch_quantize_act(const void* X, int M, int K, int ldx, const float* tinv, int G, uint8_t* Xq,
                                float* sx, cudaStream_t stream);
cudaError_t launch_pack_weights(const int8_t* Rq, const void* sw, const void* L1, const void* L2, int N, int K, int r,
                                int G, void* packed, cudaStream_t stream, int* launches);

}  // namespace twq
