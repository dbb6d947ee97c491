// fused_kernel.h -- host-side interface between the C ABI (twq_api.cu) and the fused
// dual-branch kernel (fused_kernel.cu).  Plain structs; all launch planning is host arithmetic.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cuda_fp16.h>
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
    const __half* sw16;      // [N/8][ng][8] weight group scales (FP16, tiled like R4)
    void* Y;                 // [M][ldy]
    int32_t* dbgP;           // NULL or [M][ng][N]
    float* ws_part;          // split-K partials [splits][M][N] (splits > 1 only)
    unsigned* ws_ctr;        // split-K tile counters [m_tiles][n_tiles], zero between calls
    unsigned long long* trace;   // NULL, or the timeline buffer of a -DTWQ_TRACE build (trace.cuh)
    FusedPlan plan;
};

struct FusedMaps {
    CUtensorMap W, Xq, X, L1T, L2T, Y;
};


// Small-batch calls (M <= kDecodeMaxM): parameters and plan of decode_kernel.cu (host-computed).
constexpr int kDecodeMaxM = 64;
struct DecodeParams {
    int M, N, K, r, ng;
    int ldx, ldy, ydt;       // ydt: 0 bf16, 1 fp16, 2 fp32
    int n_tiles;             // N / 8 (8-channel tiles)
    int cs, grid;            // CTAs per cluster, CTAs in the grid (a multiple of cs)
    int mt, mp;              // 16-token MMA tiles, padded tokens (16 * mt)
    int lrw;                 // warps running the low-rank chain (0 when r == 0); the other compute warps stream the residual
    int tmax;                // most 8-channel tiles any CTA owns
    int gc, nchunks, nslots; // residual ring: K-groups per chunk, chunks per call, ring depth
    int slot_bytes, xq_off;  // bytes of one ring slot; offset of the Xq box inside it
    int sc, l1_slots;        // stage-1 ring: 32-wide K slabs per chunk, ring depth
    int nu_max;              // most K slabs of stage 1 any CTA multiplies
    int xs_stride;           // halves per token row of the staged FP16 X slice
    int xrows;               // token rows staged (8 when M <= 8, else mp)
    int off_ring, off_l1, off_sw, off_xs, off_hpart, off_h, off_ylr, off_sx, off_xq, off_res, off_bar, smem_bytes;
    int quant;               // 1: the activation quantizer runs inside the kernel (twq_dual_linear_x);
                             // 2: the same with the 4-bit low-rank branch (twq_dual_linear_q4lr_x): then L1D / L2T point to the
                             //    U / V sections of a q4lr blob, "slab" means one K-group of U, and off_h holds FP32 H
    int gr, grs, nh;         // q4lr: group of the re-quantized H along r, its stored size (rounded up to 32 codes), r / gr
    int off_qh, off_sh;      // q4lr: packed Q_H [nh][mp][grs/2], scales s_H * 2^-8 [nh][mp]
    const __half* sv16;      // q4lr: [N/8][nh][8]
    float* dbgH;             // q4lr: NULL, or [M][r] FP32 H before re-quantization (parity evidence)
    int8_t* dbgQH;           // q4lr: NULL, or [M][r] codes of the re-quantized H
    float* dbgSH;            // q4lr: NULL, or [M][nh] scales s_H
    const float* tinv;       // quant: [K] diagonal transform or NULL
    uint8_t* xq_out;         // quant: NULL, or [M][K/2] copy of the codes (parity evidence)
    float* sx_out;           // quant: NULL, or [M][K/G] copy of the scales
    const uint8_t* R4;       // [N/8][ng][8][G/2]
    const __half* sw16;      // [N/8][ng][8]
    const void* L1D;         // [K/32][r][32] f16
    const void* L2T;         // [N][r] f16
    const void* X;           // [M][ldx] bf16
    const float* sx;         // [M][ng]
    void* Y;
    int32_t* dbgP;
    unsigned long long* trace;   // NULL, or the timeline buffer of a -DTWQ_TRACE build (trace.cuh)
};
bool decode_make_plan(int M, int N, int K, int r, int G, int num_sms, int quant, DecodeParams* out);
cudaError_t launch_decode(const CUtensorMap& tmXq, const DecodeParams& p, int G, cudaStream_t stream);

// Planner overrides for tests (include/twq_testing.h, twq_testing_set_plan_flags): a process-wide word, never the
// environment.  0 in production.
enum : unsigned {
    kPlanNoSplit = 1u,       // fused kernel: no K split for shapes with few tiles (small shapes then take the unsplit / CTA-pair path)
    kPlanNoPair = 2u,        // fused kernel: no CTA pairs
    kPlanNoYStage = 4u,      // fused kernel: finished tiles are stored from registers (no staged TMA store)
    kPlanNoAlias2 = 8u,      // fused kernel: the stage-1 ring may not overlay the L2T tile
    kPlanNoDecode = 16u,     // small-batch calls go to the tcgen05 kernel too
    kPlanFusedCsShift = 8,   // bits 8..11: forced cluster size of the fused kernel (0 = planner's choice)
    kPlanDecodeCsShift = 12, // bits 12..16: forced cluster size of the decode kernel (0 = planner's choice)
    kPlanFusedTnShift = 17,  // bits 17..18: token tile of the fused kernel: 0 = planner's choice, 1 = at most 64, 2 = at most 32
};
size_t workspace_counter_bytes(int M, int N, int K, int r, int G);   // twq_api.cu: zero-on-entry prefix of a workspace
unsigned plan_flags();
void set_plan_flags(unsigned f);
float measure_i8_tops(int iters, int reps, cudaStream_t stream);   // peak_i8.cu (bench measurement aid)
cudaError_t launch_cold_fill(const void* src, size_t stride, int bytes, int mode, int ctas, unsigned long long* tout,
                             cudaStream_t stream);          // cold_fill.cu (bench measurement aid)
unsigned long long* trace_buffer();   // set by twq_testing_set_trace_buffer; only read by -DTWQ_TRACE builds

// Fills `plan` for a shape; returns false if the shape cannot be planned (never for valid ABI shapes).
bool fused_make_plan(int M, int N, int K, int r, int G, int num_sms, FusedPlan* plan);
cudaError_t launch_fused(const FusedMaps& maps, const FusedParams& p, int G, cudaStream_t stream);

cudaError_t launch_quantize_act(const void* X, int M, int K, int ldx, const float* tinv, int G, uint8_t* Xq,
                                float* sx, cudaStream_t stream);
cudaError_t launch_pack_weights(const int8_t* Rq, const void* sw, const void* L1, const void* L2, int N, int K, int r,
                                int G, void* packed, cudaStream_t stream, int* launches);
cudaError_t launch_pack_weights_q4lr(const int8_t* Rq, const void* sw, const int8_t* Uq, const void* su, const int8_t* Vq,
                                     const void* sv, int N, int K, int r, int G, void* packed, cudaStream_t stream,
                                     int* launches);

}  // namespace twq
