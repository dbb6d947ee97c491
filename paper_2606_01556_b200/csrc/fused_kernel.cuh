// fused_kernel.cuh -- the fused dual-branch kernel template (steps a3-a7), sm_100a only.
// Instantiated per (TN, G, debug) in fused_inst_*.cu; planned and dispatched by fused_kernel.cu.
//
//   Y[m,n] = sum_g sx[m,g]*sw[n,g]*P[m,g,n]  +  sum_j H[m,j]*L2[j,n],
//   P[m,g,n] = sum_{k in g} qx[m,k]*qw[n,k] (exact int32),   H = X*L1 (FP32 accumulate)
//   PAPER.md Eq. 2 (L49-50), Eq. 3 (L62), L177-181 (section 4.3), L193 (groups of G).
//
// Orientation: a CTA computes Y^T for 128 output channels (TMEM lanes = n, the MMA M
// dimension; weights are the A operand) x TN tokens (TMEM columns = m, the MMA N dimension;
// activations are the B operand).  Decode-shaped calls run N = 16 MMAs.
//
// Persistent clusters.  A cluster of `cs` CTAs owns `cs` adjacent n-tiles and walks a list of
// units (K split, m-tile, n-block) with the m-tile changing slowest, so the stage-1 product
// H = X*L1 of an m-tile is computed once per cluster, cooperatively: every CTA multiplies
// 1/cs of the K range, the FP32 partials are reduce-scattered and the FP16 result all-gathered
// through distributed shared memory.  H never leaves the chip.
//
// Warp roles (640 threads; registers re-balanced per role with setmaxnreg):
//   warps 0-7   operand preparation.  All: BF16->FP16 rewrite of the X tile (kind::f16 needs one
//               16-bit format for both operands).  INT4 -> int8 expansion: each nibble c becomes
//               the byte 16*c (one shift/and per word, sign for free; sm_100 has no INT4 MMA).
//               Warps 0-3: weight rows, registers -> TMEM (the MMA reads A from TMEM, so expanded
//               weights never touch shared memory).  Warps 4-7: activation rows -> swizzled smem
//               tile (B operand), and the activation group scales.
//   warps 8-15  epilogue: per group, tcgen05.ld the int32 accumulator, fold both scales in
//               FP32 (two packed f32x2 FMAs per pair), accumulate in registers; add Ylr; store.
//   warp 16     TMA producer: stage-1 tiles (X, L1T), L2T tile, packed INT4 tiles (R4, Xq)
//   warp 17     MMA issuer (the warp runs converged, one elected lane issues): kind::f16 stage 1 /
//               stage 2, kind::i8 residual
//   warp 18     TMEM allocator
//
// CTA pairs (kPair, 128-token tiles in an even cluster): ranks 2i / 2i+1 share ONE tcgen05.mma of M = 256
// (cta_group::2).  Each CTA keeps its own 128 weight rows in its TMEM and expands only HALF of the token
// rows (B rows [rank*64, rank*64+64)), which halves the activation-side shared-memory traffic and
// expansion work; the even CTA issues after both CTAs' preparation warps and epilogues have arrived on
// ITS barriers (relaxed remote arrives: the data is already fenced locally; a release at cluster scope
// costs ~800 cycles per warp here) and multicasts the completion to both CTAs' barriers.  The odd CTA's
// issuer still runs its own stage-1 / stage-2 MMAs (cta_group::1) and follows the leader use by use.
// The single-thread roles keep stage indices and phases in counters (no division in any loop).
//
// Accumulator trick: each P buffer is pre-filled with the bit pattern of 1.5*2^23, and the
// group's MMAs accumulate 256*P onto it (|256*P| < 2^22), so tcgen05.ld returns the float
// 1.5*2^23 + 256*P directly: no int->float conversion instruction in the hot loop.
//
// Three P buffers rotate (MMA -> commit -> epilogue -> refill costs several hundred cycles of
// latency per hand-off; two buffers cannot cover it).  The low-rank product Ylr = H*L2 of a tile
// is accumulated (FP32) into the next P buffer at the START of the tile and becomes the initial
// value of the epilogue's register accumulators, so it needs no TMEM columns of its own.
// Group scales are staged ahead of use: the preparation warps fetch sx for 8 groups at a time,
// one block ahead; the epilogue warps fetch sw two groups ahead.
//
// Store of a finished tile (a thread owns one channel x TN/2 tokens): 128-token tiles of 16-bit outputs are
// written into a 128B-swizzled shared-memory tile and leave through two asynchronous TMA stores while the
// next tile is computed; other 16-bit cases transpose 8 x 8 among lanes to 16-byte stores; FP32 outputs and
// split-K partials pair neighbouring lanes (8-byte stores).  Split-K calls (one unit per cluster, whole grid
// resident): the CTAs holding the splits of a tile meet on the tile counter and each sums a share of the rows.
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <type_traits>

#include "fused_kernel.h"
#include "sm100_ptx.cuh"
#include "trace.cuh"

namespace twq {

namespace {

constexpr int kThreads = 640;
constexpr int kPrepWarps = 8;           // warps 4..7 expand weight rows, warps 8..11 expand activation rows
constexpr int kPrepThreads = kPrepWarps * 32;
constexpr int kEpiWarp0 = 8;            // first epilogue warp (a multiple of 4: TMEM lane quarter = warp % 4)
// The single-thread roles get the HIGHEST warp ids: the warp scheduler of a sub-partition favours higher warp
// ids, and with the issuer in warp 1 every step of its loop waited ~300 cycles for an issue slot behind the
// spinning / streaming warps of its sub-partition (in-kernel timeline, r01b).
constexpr int kCtlWarp0 = 16;           // 16 TMA producer, 17 MMA issuer, 18 TMEM allocator, 19 idle
constexpr int kEpiWarps = 8;            // warps 12..19
// register budgets after setmaxnreg: the pool is what the CTA was launched with (640 x 96 = 61440);
// 128*40 + 256*56 + 256*160 = 60416
constexpr int kRegsCtl = 40, kRegsPrep = 56, kRegsEpi = 160;
constexpr int kTileN = 128;             // output channels per CTA (MMA M)
constexpr int kSxSlots = 16;            // per-group activation-scale slots (two blocks of 8 groups)
constexpr int kNB = 3;                  // P accumulator buffers in rotation
constexpr int kMaxNS1 = 5, kMaxNSP = 8, kMaxNSU = 4;
constexpr int kL1Chunk = 128 * 128;     // 128 rows x 64 fp16 (one 128B-swizzled tile)
constexpr uint32_t kMagic = 0x4B400000u;  // bits of 1.5 * 2^23
constexpr int kMaxDynSmem = 232448 - 64;

// barrier slots (uint64 each)
enum : int {
    B_FULL1 = 0,
    B_EMPTY1 = B_FULL1 + kMaxNS1,
    B_XCONV = B_EMPTY1 + kMaxNS1,
    B_PFULL = B_XCONV + kMaxNS1,
    B_PEMPTY = B_PFULL + kMaxNSP,
    B_UFULL = B_PEMPTY + kMaxNSP,
    B_UEMPTY = B_UFULL + kMaxNSU,
    B_TFULL = B_UEMPTY + kMaxNSU,
    B_TEMPTY = B_TFULL + kNB,
    B_HFULL = B_TEMPTY + kNB,   // stage-1 MMAs of this CTA complete
    B_HDRAINED,                 // epilogue read H^T out of TMEM and re-initialised the P buffers
    B_HREADY,                   // full FP16 H is in this CTA's shared memory
    B_X1,                       // cluster: every CTA's FP32 partial is in its shared memory
    B_X2,                       // cluster: every CTA finished reading partials and writing H
    B_L2FULL,
    B_L2EMPTY,
    B_RESID,                    // all residual MMAs of a tile complete
    // CTA pairs (cta_group::2): barriers of the pair's leader that BOTH CTAs arrive on
    B_TEMPTY2,                  // + kNB: P buffer drained by the epilogues of both CTAs
    B_UFULL2 = B_TEMPTY2 + kNB, // + kMaxNSU: expanded operands of both CTAs ready
    B_HDRAINED2 = B_UFULL2 + kMaxNSU,
    B_COUNT
};

template <int TN, int G, bool kPair = false>
struct Cfg {
    static constexpr int kXChunk = TN * 128;          // X tile: TN rows x 64 bf16
    static constexpr int kXR = kPair ? TN / 2 : TN;   // activation rows this CTA expands (a pair splits the B rows)
    static constexpr int kWB = kTileN * (G / 2);      // packed weight rows of one group
    static constexpr int kXB = kXR * (G / 2);         // packed activation rows of one group
    static constexpr int kUB = kXR * G;               // expanded activation tile of one group
    static constexpr int kColP = 0;                   // P buffer b at b*TN; H^T block rb at rb*TN
    static constexpr int kColA = (kNB * TN + 31) / 32 * 32;   // expanded weight rows (A operand), 32 cols / stage
    static constexpr int kTmemCols = kColA + kMaxNSU * 32 <= 256 ? 256 : 512;
    static constexpr int kCW = TN >= 32 ? TN / 2 : 16;   // token columns per epilogue warp
    static constexpr int kCPW = kCW / 16;                // 16-column chunks per epilogue warp
    static_assert(kColA + kMaxNSU * 32 <= 512, "TMEM budget");
};

__device__ __forceinline__ uint32_t nib_lo16(uint32_t w) { return (w << 4) & 0xF0F0F0F0u; }  // 16*code, even k
__device__ __forceinline__ uint32_t nib_hi16(uint32_t w) { return w & 0xF0F0F0F0u; }         // 16*code, odd k

// Position of 16-byte chunk `c` of row `row` in a packed tile whose rows are G/2 bytes
// (TMA SWIZZLE_64B for G = 128, SWIZZLE_32B for G = 64).
template <int G>
__device__ __forceinline__ uint32_t packed_chunk_offset(uint32_t row, uint32_t c) {
    if constexpr (G == 128) return row * 64u + ((c ^ ((row >> 1) & 3u)) << 4);
    else return row * 32u + ((c ^ ((row >> 2) & 1u)) << 4);
}

// uses of P buffer b among the first q uses of the rotation
__device__ __forceinline__ int buf_uses(int q, int b) { return (q + kNB - 1 - b) / kNB; }

struct Unit {
    int n0, m0, g_begin, g_end, ctx, ks;
};

__device__ __forceinline__ Unit decode_unit(const FusedParams& p, int u, int rank) {
    const FusedPlan& pl = p.plan;
    Unit t;
    const int nb = u % pl.n_blocks;
    t.ctx = u / pl.n_blocks;
    const int mt = t.ctx % pl.m_tiles;
    t.ks = t.ctx / pl.m_tiles;
    t.n0 = (nb * pl.cs + rank) * kTileN;
    t.m0 = mt * pl.TN;
    t.g_begin = t.ks * pl.g_per_split;
    t.g_end = min(p.ng, t.g_begin + pl.g_per_split);
    return t;
}

// 64-wide K chunks of stage 1 this CTA multiplies for a unit's context: 1/cs of the split's K range.
template <int G>
__device__ __forceinline__ void s1_range(const FusedParams& p, const Unit& t, int rank, int& kc0, int& kc1) {
    const int b = t.g_begin * (G / 64), e = t.g_end * (G / 64);
    const int per = (e - b + p.plan.cs - 1) / p.plan.cs;
    kc0 = min(e, b + rank * per);
    kc1 = min(e, kc0 + per);
}

template <int TN, int G, bool kDbg, bool kPair = false>
__global__ void __launch_bounds__(kThreads, 1)
fused_dual_linear_kernel(const __grid_constant__ CUtensorMap tmW, const __grid_constant__ CUtensorMap tmXq,
                         const __grid_constant__ CUtensorMap tmX, const __grid_constant__ CUtensorMap tmL1T,
                         const __grid_constant__ CUtensorMap tmL2T, const __grid_constant__ CUtensorMap tmY,
                         const __grid_constant__ FusedParams p) {
    using C = Cfg<TN, G, kPair>;
    const FusedPlan& pl = p.plan;
    extern __shared__ uint8_t smem_raw[];
    // identical offset in every CTA of the cluster (DSMEM addresses are formed from local ones)
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint8_t* sH = smem + pl.off_H;          // H[m, j] fp16, K-major, 64-wide k-blocks of TN x 128 B
    uint8_t* sL2T = smem + pl.off_L2T;      // L2T tile: k-blocks of 128 x 128 B
    uint8_t* sU = smem + pl.off_U;          // expanded activation tiles [nsu][TN x G]
    uint8_t* sP = smem + pl.off_P;          // packed tiles [nsp][W 128 x G/2 | Xq TN x G/2]
    uint8_t* sS1 = smem + pl.off_S1;        // stage-1 ring [ns1][X TN x 128 | L1T nrb x 16 KB]
    float* sHpart = reinterpret_cast<float*>(smem + pl.off_Hpart);   // FP32 partial H[m][r]
    float* sSx = reinterpret_cast<float*>(smem + pl.off_sx);
    uint8_t* sY = smem + pl.off_Y;          // output staging (only when pl.ystage): 2 x [TN][64 channels], 128B-swizzled
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + pl.off_bar);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + B_COUNT);

    TWQ_TG(0);
    // through a shuffle: the compiler then knows the warp index, the role branches and their loop bounds are warp-uniform
    const int warp = __shfl_sync(0xffffffffu, static_cast<int>(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const int r = p.r;
    const int nrb = (r + 127) >> 7;          // 128-row blocks of L1T / H^T
    const int nkb = (r + 63) >> 6;           // 64-wide k-blocks of H / L2T
    const int cs = pl.cs;
    const int rank = cs > 1 ? static_cast<int>(cluster_ctarank()) : 0;
    const int cid = cs > 1 ? static_cast<int>(cluster_id_x()) : static_cast<int>(blockIdx.x);
    const int u_begin = static_cast<int>(static_cast<long long>(cid) * pl.units / pl.nclusters);
    const int u_end = static_cast<int>(static_cast<long long>(cid + 1) * pl.units / pl.nclusters);
    const int s1_stage_bytes = C::kXChunk + nrb * kL1Chunk;
    const int p_stage_bytes = C::kWB + C::kXB;

    if (threadIdx.x == 0) {
        for (int i = 0; i < kMaxNS1; ++i) {
            mbar_init(&bars[B_FULL1 + i], 1);
            mbar_init(&bars[B_EMPTY1 + i], 1);
            mbar_init(&bars[B_XCONV + i], kPrepWarps);
        }
        for (int i = 0; i < kMaxNSP; ++i) { mbar_init(&bars[B_PFULL + i], 1); mbar_init(&bars[B_PEMPTY + i], kPrepWarps); }
        for (int i = 0; i < kMaxNSU; ++i) { mbar_init(&bars[B_UFULL + i], kPrepWarps); mbar_init(&bars[B_UEMPTY + i], 1); }
        for (int i = 0; i < kNB; ++i) { mbar_init(&bars[B_TFULL + i], 1); mbar_init(&bars[B_TEMPTY + i], kEpiWarps); }
        mbar_init(&bars[B_HFULL], 1);
        mbar_init(&bars[B_HDRAINED], kEpiWarps);
        mbar_init(&bars[B_HREADY], kEpiWarps);
        mbar_init(&bars[B_X1], kEpiWarps * cs);
        mbar_init(&bars[B_X2], kEpiWarps * cs);
        mbar_init(&bars[B_L2FULL], 1);
        mbar_init(&bars[B_L2EMPTY], 1);
        mbar_init(&bars[B_RESID], 1);
        for (int i = 0; i < kNB; ++i) mbar_init(&bars[B_TEMPTY2 + i], 2 * kEpiWarps);
        for (int i = 0; i < kMaxNSU; ++i) mbar_init(&bars[B_UFULL2 + i], 2 * kPrepWarps);
        mbar_init(&bars[B_HDRAINED2], 2 * kEpiWarps);
        fence_mbar_init();
    }
    if (warp == kCtlWarp0 && lane == 0) {
        tma_prefetch_desc(&tmW);
        tma_prefetch_desc(&tmXq);
        if (r > 0) { tma_prefetch_desc(&tmX); tma_prefetch_desc(&tmL1T); tma_prefetch_desc(&tmL2T); }
    }
    if (threadIdx.x < 32) tmem_slot[8 + threadIdx.x] = kMagic;   // read back by the epilogue warps (see kfill)
    if (warp == kCtlWarp0 + 2) {
        if (kPair) tmem_alloc_pair<C::kTmemCols>(tmem_slot);
        else tmem_alloc<C::kTmemCols>(tmem_slot);
    }
    tc_fence_before();
    __syncthreads();
    if (cs > 1) cluster_sync_all();   // peers' barriers are initialised before any remote arrive
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t bar0 = smem_u32(bars);   // shared-window address of barrier slot 0 (slot i at bar0 + 8*i)
#define TWQ_BAR(i) (bar0 + 8u * static_cast<uint32_t>(i))
    // pair mode: the same barrier slots in the pair's leader (even rank), as shared::cluster addresses
    const uint32_t lbar0 = kPair ? mapa_u32(bar0, static_cast<uint32_t>(rank & ~1)) : bar0;
#define TWQ_LBAR(i) (lbar0 + 8u * static_cast<uint32_t>(i))
    const bool leader = !kPair || (rank & 1) == 0;
    pdl_launch_dependents();          // the next kernel may start its own prologue / weight prefetch
    TWQ_TG(1);

    if (warp >= kCtlWarp0) {
        reg_dec<kRegsCtl>();
    if (warp == kCtlWarp0) {
        // ================================================================ TMA producer
        if (lane == 0) {
            int tile_n = 0, ctx_n = 0, cur_ctx = -1;
            int s1 = 0, ph1 = 0;          // stage-1 ring position / phase
            int sp = 0, php = 0;          // packed ring position / phase
            bool waited = false;
            const uint32_t sP_a = smem_u32(sP);
#ifdef TWQ_TRACE
            int trn = 0;
#endif
            for (int u = u_begin; u < u_end; ++u) {
                const Unit t = decode_unit(p, u, rank);
                if (r > 0 && t.ctx != cur_ctx) {
                    cur_ctx = t.ctx;
                    // the stage-1 ring overlays the residual rings: every residual MMA must be done
                    if (pl.alias && tile_n > 0) mbar_wait(&bars[B_RESID], (tile_n - 1) & 1, 10);
                    int kc0, kc1;
                    s1_range<G>(p, t, rank, kc0, kc1);
                    if (!waited && kc0 < kc1) { pdl_wait(); waited = true; }   // X comes from the previous kernel
                    for (int kc = kc0; kc < kc1; ++kc) {
                        mbar_wait(&bars[B_EMPTY1 + s1], ph1 ^ 1, 11);
                        uint8_t* st = sS1 + s1 * s1_stage_bytes;
                        mbar_arrive_expect_tx(&bars[B_FULL1 + s1], s1_stage_bytes);
                        tma_load_2d(st, &tmX, &bars[B_FULL1 + s1], kc * 64, t.m0);
                        for (int rb = 0; rb < nrb; ++rb)
                            tma_load_2d(st + C::kXChunk + rb * kL1Chunk, &tmL1T, &bars[B_FULL1 + s1], kc * 64, rb * 128);
                        if (++s1 == pl.ns1) { s1 = 0; ph1 ^= 1; }
                    }
                    // overlay: stage-1 MMAs done and the H exchange finished before residual tiles land
                    if (pl.alias) mbar_wait(&bars[B_HREADY], ctx_n & 1, 12);
                    ++ctx_n;
                }
                if (r > 0) {
                    mbar_wait(&bars[B_L2EMPTY], (tile_n & 1) ^ 1, 13);
                    mbar_arrive_expect_tx(&bars[B_L2FULL], nkb * kL1Chunk);
                    for (int kb = 0; kb < nkb; ++kb)
                        tma_load_2d(sL2T + kb * kL1Chunk, &tmL2T, &bars[B_L2FULL], kb * 64, t.n0);
                }
                int c0 = t.g_begin * (G / 2);
                for (int g = t.g_begin; g < t.g_end; ++g, c0 += G / 2) {
                    TWQ_TR(0, trn, 1);
                    mbar_wait_a(TWQ_BAR(B_PEMPTY + sp), php ^ 1);
                    TWQ_TR(0, trn, 2);
                    const uint32_t st = sP_a + sp * p_stage_bytes;
                    mbar_arrive_expect_tx_a(TWQ_BAR(B_PFULL + sp), p_stage_bytes);
                    tma_load_4d_a(st, &tmW, TWQ_BAR(B_PFULL + sp), 0, 0, g, t.n0 >> 3);   // 16 blocks of (8 channels x G/2 bytes)
                    if (!waited) { pdl_wait(); waited = true; }               // Xq comes from the quantizer
                    tma_load_2d_a(st + C::kWB, &tmXq, TWQ_BAR(B_PFULL + sp), c0, t.m0 + (kPair ? (rank & 1) * C::kXR : 0));
                    if (++sp == pl.nsp) { sp = 0; php ^= 1; }
                }
                ++tile_n;
            }
        }
    } else if (warp == kCtlWarp0 + 1) {
        // ================================================================ MMA issuer
        // The whole warp runs the loop converged and one elected lane issues: inside an `if (lane == 0)` region
        // the compiler wraps EVERY tcgen05 instruction in its own elect / branch loop (~50 cycles each), which
        // together with two dependent barrier polls (~150 cycles each even when already complete) made the
        // issuer itself the slowest stage of the pipeline (in-kernel timeline + micro-benchmark, r01b).
        {
            const uint32_t idesc_lr = umma_idesc(1, 0, 0, 128, TN);  // D f32, A f16, B f16
            const uint32_t idesc_i8 = umma_idesc(2, 1, 1, 128, TN);  // D s32, A s8, B s8
            const uint32_t idesc_i8_pair = umma_idesc(2, 1, 1, 256, TN);
            (void)idesc_i8_pair;
            int tile_n = 0, ctx_n = 0, cur_ctx = -1;
            int s1 = 0, ph1 = 0;          // stage-1 ring position / phase
            int su = 0, phu = 0;          // expanded-operand ring position / phase
            int b = 0, pb = 0;            // next P buffer of the rotation / parity of its use count
            bool h_waited = true;
            const uint64_t udesc0 = umma_smem_desc<G>(smem_u32(sU));   // + stage * kUB/16 + k-step * 2
#ifdef TWQ_TRACE
            int trn = 0;
#endif
            for (int u = u_begin; u < u_end; ++u) {
                const Unit t = decode_unit(p, u, rank);
                if (r > 0 && t.ctx != cur_ctx) {
                    cur_ctx = t.ctx;
                    int kc0, kc1;
                    s1_range<G>(p, t, rank, kc0, kc1);
                    if (kc0 < kc1) {
                        // H^T accumulates in the columns of P buffers 0..nrb-1: all their uses must be drained
                        for (int bb = 0; bb < nrb; ++bb) mbar_wait(&bars[B_TEMPTY + bb], bb < b ? (pb ^ 1) : pb, 20);
                        tc_fence_after();
                        for (int kc = kc0; kc < kc1; ++kc) {
                            mbar_wait(&bars[B_XCONV + s1], ph1, 21);
                            tc_fence_after();
                            const uint32_t xb = smem_u32(sS1 + s1 * s1_stage_bytes);
                            const uint32_t lb = xb + C::kXChunk;
                            if (elect_one()) {
#pragma unroll
                                for (int ks = 0; ks < 4; ++ks)
                                    for (int rb = 0; rb < nrb; ++rb)
                                        umma_f16(tmem + C::kColP + rb * TN, umma_smem_desc<128>(lb + rb * kL1Chunk + ks * 32),
                                                 umma_smem_desc<128>(xb + ks * 32), idesc_lr, (kc != kc0 || ks != 0) ? 1u : 0u);
                                tc_commit(&bars[B_EMPTY1 + s1]);
                            }
                            __syncwarp();
                            if (++s1 == pl.ns1) { s1 = 0; ph1 ^= 1; }
                        }
                        if (elect_one()) tc_commit(&bars[B_HFULL]);
                        __syncwarp();
                    } else {
                        if (elect_one()) mbar_arrive(&bars[B_HFULL]);   // empty K share: the epilogue contributes zeros
                        __syncwarp();
                    }
                    mbar_wait(&bars[B_HDRAINED], ctx_n & 1, 22);
                    // pair leader: its MMAs also write the peer's P buffers, where the peer's H^T partial lives
                    if (kPair && leader) mbar_wait_cluster_a(TWQ_BAR(B_HDRAINED2), ctx_n & 1);
                    tc_fence_after();
                    h_waited = false;
                }
                if (r > 0) {
                    // stage 2 first: Ylr^T = L2T * H^T (FP32) into the next P buffer; the epilogue takes it
                    // as the initial value of its accumulators
                    if (!h_waited) { mbar_wait(&bars[B_HREADY], ctx_n & 1, 25); h_waited = true; ++ctx_n; }
                    mbar_wait(&bars[B_L2FULL], tile_n & 1, 26 + 100 * tile_n + 10000 * (rank & 1));
                    mbar_wait(&bars[B_TEMPTY + b], pb, 27);
                    tc_fence_after();
                    const uint32_t l2b = smem_u32(sL2T), hb = smem_u32(sH);
                    const int nks = (r + 15) >> 4;
                    if (elect_one()) {
                        for (int ks = 0; ks < nks; ++ks) {
                            const int kb = ks >> 2, kk = ks & 3;
                            umma_f16(tmem + C::kColP + b * TN, umma_smem_desc<128>(l2b + kb * kL1Chunk + kk * 32),
                                     umma_smem_desc<128>(hb + kb * (TN * 128) + kk * 32), idesc_lr, ks != 0 ? 1u : 0u);
                        }
                        tc_commit(&bars[B_L2EMPTY]);
                        tc_commit(&bars[B_TFULL + b]);
                    }
                    __syncwarp();
                    if (++b == kNB) { b = 0; pb ^= 1; }
                }
                const int ngr = t.g_end - t.g_begin;
                for (int gi = 0; gi < ngr; ++gi) {
                    TWQ_TR(1, trn, 1);
                    if (!kPair) {
                        {   // both polls in flight together
                            const bool ok1 = mbar_try_wait_a(TWQ_BAR(B_TEMPTY + b), pb);
                            const bool ok2 = mbar_try_wait_a(TWQ_BAR(B_UFULL + su), phu);
                            if (!ok1) mbar_wait_a(TWQ_BAR(B_TEMPTY + b), pb);
                            TWQ_TR(1, trn, 2);
                            if (!ok2) mbar_wait_a(TWQ_BAR(B_UFULL + su), phu);
                        }
                        TWQ_TR(1, trn, 3);
                        tc_fence_after();
                        const uint64_t ud = udesc0 + static_cast<uint64_t>(su * (C::kUB >> 4));
                        const uint32_t ta = tmem + C::kColA + su * 32;
                        const uint32_t td = tmem + C::kColP + b * TN;
                        if (elect_one()) {
#pragma unroll
                            for (int ks = 0; ks < G / 32; ++ks)   // accumulate onto the pre-filled 1.5*2^23 pattern
                                umma_i8_ts(td, ta + ks * 8, ud + static_cast<uint64_t>(ks * 2), idesc_i8, 1u);
                            tc_commit_a(TWQ_BAR(B_UEMPTY + su));
                            tc_commit_a(TWQ_BAR(B_TFULL + b));
                        }
                        __syncwarp();
                    } else if (leader) {
                        // one M = 256 MMA per K-step for the pair: both epilogues drained buffer b, both CTAs'
                        // operands of stage su are in place; completion is multicast to both CTAs' barriers
                        {   // both polls in flight together
                            const bool ok1 = mbar_try_wait_cluster_a(TWQ_BAR(B_TEMPTY2 + b), pb);
                            const bool ok2 = mbar_try_wait_cluster_a(TWQ_BAR(B_UFULL2 + su), phu);
                            if (!ok1) mbar_wait_cluster_a(TWQ_BAR(B_TEMPTY2 + b), pb);
                            TWQ_TR(1, trn, 2);
                            if (!ok2) mbar_wait_cluster_a(TWQ_BAR(B_UFULL2 + su), phu);
                        }
                        TWQ_TR(1, trn, 3);
                        tc_fence_after();
                        const uint64_t ud = udesc0 + static_cast<uint64_t>(su * (C::kUB >> 4));
                        const uint32_t ta = tmem + C::kColA + su * 32;
                        const uint32_t td = tmem + C::kColP + b * TN;
                        if (elect_one()) {
#pragma unroll
                            for (int ks = 0; ks < G / 32; ++ks)
                                umma_i8_ts_pair(td, ta + ks * 8, ud + static_cast<uint64_t>(ks * 2), idesc_i8_pair, 1u);
                            const uint16_t mask = static_cast<uint16_t>(3u << (rank & ~1));
                            tc_commit_pair_a(TWQ_BAR(B_UEMPTY + su), mask);
                            tc_commit_pair_a(TWQ_BAR(B_TFULL + b), mask);
                        }
                        __syncwarp();
                    } else {
                        // the peer's issuer follows the leader use by use (a parity wait may only be one phase
                        // ahead of its barrier): it waits for the leader's completion of this group
                        mbar_wait_a(TWQ_BAR(B_TFULL + b), pb);
                    }
                    TWQ_TR(1, trn, 4);
                    if (++su == pl.nsu) { su = 0; phu ^= 1; }
                    if (++b == kNB) { b = 0; pb ^= 1; }
                }
                // all residual MMAs of the tile complete (alias mode: the stage-1 ring may overwrite the rings);
                // in a pair the leader's commit covers both CTAs' operands
                if (elect_one()) {
                    if (!kPair) tc_commit(&bars[B_RESID]);
                    else if (leader) tc_commit_pair_a(TWQ_BAR(B_RESID), static_cast<uint16_t>(3u << (rank & ~1)));
                }
                __syncwarp();
                ++tile_n;
            }
        }
    }
    }  // control warps
    else if (warp < kEpiWarp0) {
        // ================================================================ operand preparation warps
        reg_dec<kRegsPrep>();
        const bool w_role = warp < 4;                 // warps 0-3: weight rows -> TMEM; warps 4-7: activation rows -> smem
        const int c_tid = threadIdx.x;                // 0..255, stage-1 conversion index
        const int u_tid = threadIdx.x & 127;          // index inside the role
        const int qd = warp & 3;                      // TMEM lane quarter a weight warp may write
        const uint32_t arow = qd * 32 + lane;         // weight row (output channel) of this thread
        const uint32_t tlane = tmem + (static_cast<uint32_t>(qd * 32) << 16);
        constexpr int kCPR = (G / 2) / 16;            // 16-byte packed chunks per row
        // activation rows: kTPR threads share a row, each expands kXC of its kCPR chunks
        constexpr int kTPR = (128 / C::kXR) < kCPR ? (128 / C::kXR) : kCPR;
        constexpr int kXC = kCPR / kTPR;
        const uint32_t xrow = u_tid % C::kXR;
        const uint32_t xpart = u_tid / C::kXR;
        const bool x_on = xpart < kTPR;
        uint32_t in_off[kCPR];                        // packed chunk offsets (weight role: all; activation role: first kXC)
        uint32_t out_off[2 * kXC];
        if (w_role) {
#pragma unroll
            for (int c = 0; c < kCPR; ++c) in_off[c] = packed_chunk_offset<G>(arow, c);
        } else {
#pragma unroll
            for (int j = 0; j < kXC; ++j) {
                const uint32_t ch = xpart + j * kTPR;
                in_off[j] = C::kWB + packed_chunk_offset<G>(xrow, ch);
                out_off[2 * j] = swizzled_chunk_offset<G>(xrow, 2 * ch);
                out_off[2 * j + 1] = swizzled_chunk_offset<G>(xrow, 2 * ch + 1);
            }
        }
        pdl_wait();                                   // reads sx (quantizer output)
        int cur_ctx = -1, itp = 0;
        int s1 = 0, ph1 = 0, sp = 0, php = 0, su = 0, phu = 0;
#ifdef TWQ_TRACE
        int trn = (warp == 4 && lane == 0) ? 0 : 4096;
#endif
        float sxv[8];                                 // scales of the next block of 8 groups for token row u_tid
        // scales of the unit the last fetch came from: row pointer (at the unit's first group) and validity.  A fetch
        // inside the same unit only advances along the row; decode_unit (integer divisions, ~500 cycles) runs once per unit.
        const float* fx_row = p.sx;
        bool fx_ok = false;
        auto fetch_sx = [&](const float* src, int left) {
            if (fx_ok && left >= 8 && (reinterpret_cast<uintptr_t>(src) & 15u) == 0) {
                // sx is written by the stream predecessor, which may still have been running when this kernel started
                // (programmatic dependent launch): coherent loads, not the read-only (.nc) path
                const float4 a = __ldcg(reinterpret_cast<const float4*>(src)), c = __ldcg(reinterpret_cast<const float4*>(src) + 1);
                sxv[0] = a.x; sxv[1] = a.y; sxv[2] = a.z; sxv[3] = a.w;
                sxv[4] = c.x; sxv[5] = c.y; sxv[6] = c.z; sxv[7] = c.w;
            } else {
#pragma unroll
                for (int j = 0; j < 8; ++j) sxv[j] = (fx_ok && j < left) ? __ldcg(src + j) : 0.0f;
            }
        };
        {
#pragma unroll
            for (int j = 0; j < 8; ++j) sxv[j] = 0.0f;
            if (!w_role && u_begin < u_end) {
                const Unit t0 = decode_unit(p, u_begin, rank);
                const int m = t0.m0 + u_tid;
                fx_ok = u_tid < TN && m < p.M;
                fx_row = p.sx + static_cast<size_t>(fx_ok ? m : 0) * p.ng + t0.g_begin;
                fetch_sx(fx_row, t0.g_end - t0.g_begin);
            }
        }
        for (int u = u_begin; u < u_end; ++u) {
            const Unit t = decode_unit(p, u, rank);
            if (r > 0 && t.ctx != cur_ctx) {
                cur_ctx = t.ctx;
                // kind::f16 needs A and B in ONE 16-bit format and L1 is FP16: rewrite the BF16 X tile in
                // place as FP16 (exact for 2^-14 <= |x| <= 65504, saturating above).  Elementwise, so the
                // swizzled layout TMA wrote is untouched.
                int kc0, kc1;
                s1_range<G>(p, t, rank, kc0, kc1);
                for (int kc = kc0; kc < kc1; ++kc) {
                    mbar_wait(&bars[B_FULL1 + s1], ph1, 30);
                    uint4* xt = reinterpret_cast<uint4*>(sS1 + s1 * s1_stage_bytes);
                    for (int i = c_tid; i < C::kXChunk / 16; i += kPrepThreads) {
                        uint4 w = xt[i];
                        uint32_t* wp = reinterpret_cast<uint32_t*>(&w);
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            float lo = __uint_as_float(wp[e] << 16), hi = __uint_as_float(wp[e] & 0xFFFF0000u);
                            lo = fminf(fmaxf(lo, -65504.0f), 65504.0f);
                            hi = fminf(fmaxf(hi, -65504.0f), 65504.0f);
                            const __half2 h2 = __floats2half2_rn(lo, hi);
                            wp[e] = *reinterpret_cast<const uint32_t*>(&h2);
                        }
                        xt[i] = w;
                    }
                    fence_proxy_async_smem();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&bars[B_XCONV + s1]);
                    if (++s1 == pl.ns1) { s1 = 0; ph1 ^= 1; }
                }
            }
            const int ngr = t.g_end - t.g_begin;
            for (int gi = 0; gi < ngr; ++gi, ++itp) {
                if (!w_role && (gi & 7) == 0) {
                    // activation scales of groups gi..gi+7 (fetched one block ahead), pre-multiplied by 2^-8
                    // (the MMA operands are 16*code); then start the fetch of the next block
                    if (u_tid < TN) {
#pragma unroll
                        for (int j = 0; j < 8; ++j) sSx[((itp + j) & (kSxSlots - 1)) * TN + u_tid] = sxv[j] * 0x1p-8f;
                    }
                    if (gi + 8 < ngr) {
                        fetch_sx(fx_row + gi + 8, ngr - gi - 8);          // same unit: fx_row is this unit's row
                    } else if (u + 1 < u_end) {
                        const Unit tn = decode_unit(p, u + 1, rank);
                        const int m = tn.m0 + u_tid;
                        fx_ok = u_tid < TN && m < p.M;
                        fx_row = p.sx + static_cast<size_t>(fx_ok ? m : 0) * p.ng + tn.g_begin;
                        fetch_sx(fx_row, tn.g_end - tn.g_begin);
                    }
                }
                TWQ_TR(2, trn, 1);
                // both barrier polls in flight together (a poll costs ~150 cycles even when the phase is complete)
                const bool pf_ok = mbar_try_wait_a(TWQ_BAR(B_PFULL + sp), php);
                const bool ue_ok = mbar_try_wait_a(TWQ_BAR(B_UEMPTY + su), phu ^ 1);
                if (!pf_ok) mbar_wait_a(TWQ_BAR(B_PFULL + sp), php);
                TWQ_TR(2, trn, 2);
                const uint8_t* pw = sP + sp * p_stage_bytes;
                if (w_role) {
                    // weight row -> registers -> 16*code bytes -> TMEM (A operand): 16 int8 words per packed chunk pair
                    uint4 wv[kCPR];
#pragma unroll
                    for (int c = 0; c < kCPR; ++c) wv[c] = *reinterpret_cast<const uint4*>(pw + in_off[c]);
                    if (!ue_ok) mbar_wait_a(TWQ_BAR(B_UEMPTY + su), phu ^ 1);
                    tc_fence_after();
#pragma unroll
                    for (int c = 0; c < kCPR; c += 2) {
                        uint32_t o[16];
                        const uint32_t wi[8] = {wv[c].x, wv[c].y, wv[c].z, wv[c].w, wv[c + 1].x, wv[c + 1].y, wv[c + 1].z, wv[c + 1].w};
#pragma unroll
                        for (int i = 0; i < 8; ++i) { o[2 * i] = nib_lo16(wi[i]); o[2 * i + 1] = nib_hi16(wi[i]); }
                        tmem_st16(tlane + C::kColA + su * 32 + c * 8, o);
                    }
                    tmem_st_wait();
                    tc_fence_before();
                } else {
                    // activation rows -> swizzled K-major smem tile (B operand)
                    uint4 xv[kXC];
                    if (x_on) {
#pragma unroll
                        for (int j = 0; j < kXC; ++j) xv[j] = *reinterpret_cast<const uint4*>(pw + in_off[j]);
                    }
                    if (!ue_ok) mbar_wait_a(TWQ_BAR(B_UEMPTY + su), phu ^ 1);
                    TWQ_TR(2, trn, 3);
                    if (x_on) {
                        uint8_t* ub = sU + su * C::kUB;
#pragma unroll
                        for (int j = 0; j < kXC; ++j) {
                            const uint4 w = xv[j];
                            *reinterpret_cast<uint4*>(ub + out_off[2 * j]) =
                                make_uint4(nib_lo16(w.x), nib_hi16(w.x), nib_lo16(w.y), nib_hi16(w.y));
                            *reinterpret_cast<uint4*>(ub + out_off[2 * j + 1]) =
                                make_uint4(nib_lo16(w.z), nib_hi16(w.z), nib_lo16(w.w), nib_hi16(w.w));
                        }
                    }
                    fence_proxy_async_smem();  // generic-proxy writes -> visible to the tensor core (async proxy)
                }
                __syncwarp();
                if (lane == 0) {
                    if (kPair) mbar_arrive_remote_relaxed(TWQ_LBAR(B_UFULL2 + su));   // release.cluster, on the pair leader
                    else mbar_arrive_a(TWQ_BAR(B_UFULL + su));
                    mbar_arrive_a(TWQ_BAR(B_PEMPTY + sp));
                }
                TWQ_TR(2, trn, 4);
                if (++sp == pl.nsp) { sp = 0; php ^= 1; }
                if (++su == pl.nsu) { su = 0; phu ^= 1; }
            }
        }
    }
    else {
        // ================================================================ epilogue warps
        reg_inc<kRegsEpi>();
        const int qd = warp & 3;             // TMEM lane quarter this warp may access
        const int h = (warp - kEpiWarp0) >> 2;   // which half of the token columns
        const bool active = TN >= 32 || h == 0;
        const int col0 = h * C::kCW;
        const int row = qd * 32 + lane;
        const int et = threadIdx.x - kEpiWarp0 * 32;    // 0..255
        const uint32_t tlane = tmem + (static_cast<uint32_t>(qd * 32) << 16);
        constexpr int kNA = C::kCPW * 8;     // accumulator pairs per thread
        bool y_pending = false;              // first epilogue warp: bulk stores of the previous tile in flight
        uint64_t acc[kNA];
        // the 1.5*2^23 pattern in 16 registers that stay allocated (a tcgen05.st source is a register vector;
        // opaque to the compiler so that it is not re-materialised per store)
        uint32_t kfill[16];
        {
            // one word per lane, so that the values are not warp-uniform to the compiler (uniform registers
            // would be copied into a fresh vector before every store)
            const volatile uint32_t* mg = reinterpret_cast<const volatile uint32_t*>(tmem_slot + 8) + lane;
#pragma unroll
            for (int i = 0; i < 16; ++i) kfill[i] = *mg;
        }
#ifdef TWQ_TRACE
        int trn = 0;
        const bool trw = warp == kEpiWarp0 && lane == 0;
#endif

        // pre-fill this warp's slices of the P buffers with the 1.5*2^23 pattern
        if (active) {
#pragma unroll
            for (int b = 0; b < kNB; ++b)
#pragma unroll
                for (int i = 0; i < C::kCPW; ++i) tmem_st16(tlane + C::kColP + b * TN + col0 + i * 16, kfill);
            tmem_st_wait();
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
#pragma unroll
            for (int b = 0; b < kNB; ++b) {
                mbar_arrive(&bars[B_TEMPTY + b]);
                if (kPair) mbar_arrive_remote_relaxed(TWQ_LBAR(B_TEMPTY2 + b));
            }
        }
        pdl_wait();                          // Y / workspace writes must follow the previous kernel
        TWQ_TG(2);

        int itp = 0, ctx_n = 0, cur_ctx = -1;
        int b = 0, pb = 0;                   // next P buffer / parity of its use count (same rotation as the MMA issuer)
        for (int u = u_begin; u < u_end; ++u) {
            const Unit t = decode_unit(p, u, rank);
            const int n = t.n0 + row;
            const bool n_ok = n < p.N;
            // FP16 group scales, tiled [N/8][ng][8]: channel n of group g at ((n >> 3) * ng + g) * 8 + (n & 7)
            const __half* swp = p.sw16 + (n_ok ? (static_cast<size_t>(n >> 3) * p.ng * 8 + (n & 7)) : 0);
            // weight scales two groups ahead of use; the raw FP16 bits wait in the registers and are converted at use
            // (a conversion right behind the load would make the warp wait for the load it just issued)
            const unsigned short* swu = reinterpret_cast<const unsigned short*>(swp);
            unsigned short sw0 = n_ok ? __ldg(swu + static_cast<size_t>(t.g_begin) * 8) : static_cast<unsigned short>(0);
            unsigned short sw1 = (n_ok && t.g_begin + 1 < t.g_end) ? __ldg(swu + static_cast<size_t>(t.g_begin + 1) * 8) : static_cast<unsigned short>(0);
            if (r > 0 && t.ctx != cur_ctx) {
                cur_ctx = t.ctx;
                int kc0, kc1;
                s1_range<G>(p, t, rank, kc0, kc1);
                const bool has_s1 = kc0 < kc1;
                mbar_wait(&bars[B_HFULL], ctx_n & 1, 40);
                TWQ_TG(12);
                tc_fence_after();
                if (active) {
                    for (int rb = 0; rb < nrb; ++rb) {
                        const int j = rb * 128 + row;
#pragma unroll
                        for (int i = 0; i < C::kCPW; ++i) {
                            uint32_t v[16];
                            if (has_s1) {
                                tmem_ld16(tlane + C::kColP + rb * TN + col0 + i * 16, v);
                                tmem_ld_wait();
                            } else {
#pragma unroll
                                for (int c = 0; c < 16; ++c) v[c] = 0u;
                            }
                            if (j < r) {
                                if (cs == 1) {
                                    uint8_t* hk = sH + (j >> 6) * (TN * 128) + (j & 7) * 2;
                                    const uint32_t chunk = (j & 63) >> 3;
#pragma unroll
                                    for (int c = 0; c < 16; ++c) {
                                        const uint32_t m = col0 + i * 16 + c;
                                        const float hv = fminf(fmaxf(__uint_as_float(v[c]), -65504.0f), 65504.0f);
                                        *reinterpret_cast<__half*>(hk + swizzled_chunk_offset<128>(m, chunk)) = __float2half_rn(hv);
                                    }
                                } else {
#pragma unroll
                                    for (int c = 0; c < 16; ++c) sHpart[(col0 + i * 16 + c) * r + j] = __uint_as_float(v[c]);
                                }
                            }
                        }
                    }
                    // the H^T columns are P buffers 0..nrb-1: restore their pre-fill
                    for (int bb = 0; bb < nrb; ++bb)
#pragma unroll
                        for (int i = 0; i < C::kCPW; ++i) tmem_st16(tlane + C::kColP + bb * TN + col0 + i * 16, kfill);
                    tmem_st_wait();
                }
                tc_fence_before();
                __syncwarp();
                TWQ_TG(13);
                if (lane == 0) {
                    mbar_arrive(&bars[B_HDRAINED]);
                    if (kPair) mbar_arrive_remote_relaxed(TWQ_LBAR(B_HDRAINED2));
                }
                if (cs > 1) {
                    // ---- reduce-scatter the FP32 partials, all-gather the FP16 result (DSMEM)
                    if (lane < cs) mbar_arrive_remote(mapa_u32(smem_u32(&bars[B_X1]), lane));
                    mbar_wait_cluster(&bars[B_X1], ctx_n & 1, 41);
                    TWQ_TG(14);
                    const int jcs = r >> 3;                     // 8-wide column chunks of H
                    const int total = TN * jcs;
                    for (int i = rank + cs * et; i < total; i += cs * 256) {
                        const int m = i / jcs, jc = i - m * jcs;
                        const uint32_t src = smem_u32(sHpart + m * r + jc * 8);
                        float s[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
                        // the remote loads of two peers in flight together (one at a time was a chain of cs round trips per
                        // element: 6400 cycles of the split-K call at M = 128, r02); fixed order: every CTA sees identical H
                        // the CTA's own partial is read with plain shared loads: distributed shared memory moves ~20 bytes per
                        // cycle, and through it the own half cost as much as the peer's
                        const float* own = sHpart + m * r + jc * 8;
                        for (int pr = 0; pr < cs; pr += 2) {
                            const int p1 = pr + 1 < cs ? pr + 1 : pr;
                            const uint32_t a0 = mapa_u32(src, pr), a1 = mapa_u32(src, p1);
                            const float4 x0 = pr == rank ? *reinterpret_cast<const float4*>(own) : ld_dsmem_f4(a0);
                            const float4 x1 = pr == rank ? *reinterpret_cast<const float4*>(own + 4) : ld_dsmem_f4(a0 + 16);
                            float4 y0 = p1 == rank ? *reinterpret_cast<const float4*>(own) : ld_dsmem_f4(a1);
                            float4 y1 = p1 == rank ? *reinterpret_cast<const float4*>(own + 4) : ld_dsmem_f4(a1 + 16);
                            if (pr + 1 >= cs) { y0 = make_float4(0.f, 0.f, 0.f, 0.f); y1 = y0; }
                            s[0] += x0.x; s[1] += x0.y; s[2] += x0.z; s[3] += x0.w;
                            s[4] += x1.x; s[5] += x1.y; s[6] += x1.z; s[7] += x1.w;
                            s[0] += y0.x; s[1] += y0.y; s[2] += y0.z; s[3] += y0.w;
                            s[4] += y1.x; s[5] += y1.y; s[6] += y1.z; s[7] += y1.w;
                        }
                        uint32_t hw[4];
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const float lo = fminf(fmaxf(s[2 * e], -65504.0f), 65504.0f);
                            const float hi = fminf(fmaxf(s[2 * e + 1], -65504.0f), 65504.0f);
                            const __half2 h2 = __floats2half2_rn(lo, hi);
                            hw[e] = *reinterpret_cast<const uint32_t*>(&h2);
                        }
                        uint8_t* dloc = sH + (jc >> 3) * (TN * 128) + swizzled_chunk_offset<128>(m, jc & 7);
                        const uint32_t dst = smem_u32(dloc);
                        for (int pr = 0; pr < cs; ++pr) {
                            if (pr == rank) *reinterpret_cast<uint4*>(dloc) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
                            else st_dsmem_u4(mapa_u32(dst, pr), make_uint4(hw[0], hw[1], hw[2], hw[3]));
                        }
                    }
                    TWQ_TG(15);
                    fence_proxy_async_all();
                    __syncwarp();
                    if (lane < cs) mbar_arrive_remote(mapa_u32(smem_u32(&bars[B_X2]), lane));
                    mbar_wait_cluster(&bars[B_X2], ctx_n & 1, 42);
                }
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars[B_HREADY]);
                TWQ_TG(3);
                ++ctx_n;
            }

            if (r > 0) {
                // Ylr of this tile (FP32) is the initial value of the accumulators
                mbar_wait(&bars[B_TFULL + b], pb, 44);
                tc_fence_after();
                if (active) {
                    // all loads in flight, one wait (the accumulator registers are free at this point)
                    uint32_t v[C::kCPW][16];
#pragma unroll
                    for (int i = 0; i < C::kCPW; ++i) tmem_ld16(tlane + C::kColP + b * TN + col0 + i * 16, v[i]);
                    tmem_ld_wait();
#pragma unroll
                    for (int i = 0; i < C::kCPW; ++i) tmem_st16(tlane + C::kColP + b * TN + col0 + i * 16, kfill);
#pragma unroll
                    for (int i = 0; i < C::kCPW; ++i) {
#pragma unroll
                        for (int c2 = 0; c2 < 8; ++c2)
                            acc[i * 8 + c2] = (static_cast<uint64_t>(v[i][2 * c2 + 1]) << 32) | v[i][2 * c2];
                    }
                    tmem_st_wait();
                }
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(&bars[B_TEMPTY + b]);
                    if (kPair) mbar_arrive_remote_relaxed(TWQ_LBAR(B_TEMPTY2 + b));
                }
                if (++b == kNB) { b = 0; pb ^= 1; }
#ifdef TWQ_TRACE
                if (trw) TWQ_TR(3, trn, 7);
#endif
            } else {
#pragma unroll
                for (int i = 0; i < kNA; ++i) acc[i] = 0ull;
            }

            for (int g = t.g_begin; g < t.g_end; ++g, ++itp) {
                const float swn = __half2float(__ushort_as_half(sw0));
                sw0 = sw1;
                sw1 = (n_ok && g + 2 < t.g_end) ? __ldg(swu + static_cast<size_t>(g + 2) * 8) : static_cast<unsigned short>(0);
                const float cm = __fmul_rn(12582912.0f, swn);   // exact: sw has an 11-bit significand
                const uint64_t sw2 = pack_f2(swn, swn), ncm2 = pack_f2(-cm, -cm);
#ifdef TWQ_TRACE
                if (trw) TWQ_TR(3, trn, 1);
#endif
                mbar_wait_a(TWQ_BAR(B_TFULL + b), pb);
#ifdef TWQ_TRACE
                if (trw) TWQ_TR(3, trn, 2);
#endif
                tc_fence_after();
                if (active) {
                    const float* cs_ = sSx + (itp & (kSxSlots - 1)) * TN + col0;
                    const uint32_t tcol = tlane + C::kColP + b * TN + col0;
                    constexpr int kBatch = C::kCPW >= 2 ? 2 : 1;   // two 16-column loads per tcgen05.wait::ld
#pragma unroll
                    for (int i0 = 0; i0 < C::kCPW; i0 += kBatch) {
                        uint32_t v[kBatch][16];
#pragma unroll
                        for (int bi = 0; bi < kBatch; ++bi) tmem_ld16(tcol + (i0 + bi) * 16, v[bi]);
                        tmem_ld_wait();
#pragma unroll
                        for (int bi = 0; bi < kBatch; ++bi) tmem_st16(tcol + (i0 + bi) * 16, kfill);
                        if (i0 + kBatch >= C::kCPW) {    // last batch: hand the buffer back before the arithmetic
                            tmem_st_wait();
                            tc_fence_before();
                            __syncwarp();
                            if (lane == 0) {
                                mbar_arrive_a(TWQ_BAR(B_TEMPTY + b));
                                if (kPair) mbar_arrive_remote_relaxed(TWQ_LBAR(B_TEMPTY2 + b));
                            }
#ifdef TWQ_TRACE
                            if (trw) TWQ_TR(3, trn, 3);
#endif
                        }
#pragma unroll
                        for (int bi = 0; bi < kBatch; ++bi) {
#pragma unroll
                            for (int c4 = 0; c4 < 4; ++c4) {
                                const float4 s4 = *reinterpret_cast<const float4*>(cs_ + (i0 + bi) * 16 + c4 * 4);
                                // v = bits(1.5*2^23 + 256*P): one FMA gives RN(256*P * sw), the next accumulates * sx*2^-8
                                const uint64_t f01 = (static_cast<uint64_t>(v[bi][c4 * 4 + 1]) << 32) | v[bi][c4 * 4];
                                const uint64_t f23 = (static_cast<uint64_t>(v[bi][c4 * 4 + 3]) << 32) | v[bi][c4 * 4 + 2];
                                const uint64_t t01 = fma2(f01, sw2, ncm2), t23 = fma2(f23, sw2, ncm2);
                                const int a = (i0 + bi) * 8 + c4 * 2;
                                acc[a] = fma2(t01, pack_f2(s4.x, s4.y), acc[a]);
                                acc[a + 1] = fma2(t23, pack_f2(s4.z, s4.w), acc[a + 1]);
                            }
                            if (kDbg) {
                                if (p.dbgP != nullptr && n_ok) {
#pragma unroll
                                    for (int c = 0; c < 16; ++c) {
                                        const int m = t.m0 + col0 + (i0 + bi) * 16 + c;
                                        if (m < p.M)
                                            p.dbgP[(static_cast<size_t>(m) * p.ng + g) * p.N + n] =
                                                static_cast<int32_t>(v[bi][c] - kMagic) >> 8;
                                    }
                                }
                            }
                        }
                    }
                } else {
                    __syncwarp();
                    if (lane == 0) {
                        mbar_arrive_a(TWQ_BAR(B_TEMPTY + b));
                        if (kPair) mbar_arrive_remote_relaxed(TWQ_LBAR(B_TEMPTY2 + b));
                    }
                }
#ifdef TWQ_TRACE
                if (trw) TWQ_TR(3, trn, 4);
#endif
                if (++b == kNB) { b = 0; pb ^= 1; }
            }

#ifdef TWQ_TRACE
            if (trw) TWQ_TR(3, trn, 5);
#endif
#ifndef TWQ_EXP_NOSTORE
            if (active && pl.splits == 1 && p.ydt <= 1 && (p.ldy & 7) == 0) {
                const bool staged = pl.ystage != 0;
                if (staged) {
                    // the bulk copies of the previous tile have read the staging tile (issued a whole tile ago)
                    if (warp == kEpiWarp0 && y_pending) bulk_wait_read0();
                    named_bar_sync(1, kEpiWarps * 32);
                }
#ifdef TWQ_TRACE
                if (trw) TWQ_TR(3, trn, 8);
#endif
                // 16-bit outputs, 16-byte aligned rows.  Lane = output channel, register = token: an 8 x 8 transpose
                // among groups of 8 lanes (three butterfly rounds, 8 shuffles per 8 tokens) leaves each lane with 8
                // consecutive channels of ONE token: 8 16-byte stores per thread instead of 64 2-byte ones (a store
                // instruction cost ~115 cycles per warp here whatever its width: 7500 cycles per tile before).
                const bool b0 = lane & 1, b1 = lane & 2, b2 = lane & 4;
                const int n8 = t.n0 + qd * 32 + (lane & 24);
                const bool n8_ok = n8 < p.N;                      // N is a multiple of 16
                // one straight-line copy per (format, staged) case: with the two uniform branches inside the loop the
                // eight blocks ran one after the other, each a chain of three shuffle latencies (2200 cycles per tile)
                auto store16 = [&](auto kBf16, auto kStaged) {
#pragma unroll
                for (int blk = 0; blk < kNA / 4; ++blk) {
                    uint32_t rA[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        float y0, y1;
                        unpack_f2(acc[blk * 4 + k], y0, y1);
                        uint32_t w;                               // [token 2k | token 2k+1] of the own channel
                        if (decltype(kBf16)::value) { const __nv_bfloat162 v = __floats2bfloat162_rn(y0, y1); w = *reinterpret_cast<const uint32_t*>(&v); }
                        else { const __half2 v = __floats2half2_rn(y0, y1); w = *reinterpret_cast<const uint32_t*>(&v); }
                        const uint32_t got = __shfl_xor_sync(0xffffffffu, w, 1);
                        // even lane: token 2k, channels (own, partner); odd lane: token 2k+1, channels (partner, own)
                        rA[k] = b0 ? __byte_perm(got, w, 0x7632) : __byte_perm(w, got, 0x5410);
                    }
                    // round 2: lane bit 1 <-> token bit 1 (k & 1); two channel pairs per token
                    uint32_t rB[2][2];
#pragma unroll
                    for (int s2 = 0; s2 < 2; ++s2) {
                        const uint32_t keep = b1 ? rA[2 * s2 + 1] : rA[2 * s2], send = b1 ? rA[2 * s2] : rA[2 * s2 + 1];
                        const uint32_t got = __shfl_xor_sync(0xffffffffu, send, 2);
                        rB[s2][0] = b1 ? got : keep;
                        rB[s2][1] = b1 ? keep : got;
                    }
                    // round 3: lane bit 2 <-> token bit 2; four channel pairs of one token
                    uint32_t o4[4];
                    {
                        const uint32_t k0 = b2 ? rB[1][0] : rB[0][0], k1 = b2 ? rB[1][1] : rB[0][1];
                        const uint32_t s0 = b2 ? rB[0][0] : rB[1][0], s1 = b2 ? rB[0][1] : rB[1][1];
                        const uint32_t g0 = __shfl_xor_sync(0xffffffffu, s0, 4), g1 = __shfl_xor_sync(0xffffffffu, s1, 4);
                        o4[0] = b2 ? g0 : k0; o4[1] = b2 ? g1 : k1;
                        o4[2] = b2 ? k0 : g0; o4[3] = b2 ? k1 : g1;
                    }
                    const int mrow = col0 + blk * 8 + (lane & 7);
                    const int m = t.m0 + mrow;
                    if (decltype(kStaged)::value) {
                        // channel half (qd >> 1), row of 128 bytes, 16-byte chunk XOR (row & 7): the layout TMA expects
                        const int c16 = ((qd & 1) * 32 + (lane & 24)) >> 3;
                        *reinterpret_cast<uint4*>(sY + (qd >> 1) * (TN * 128) + mrow * 128 + ((c16 ^ (mrow & 7)) << 4)) =
                            make_uint4(o4[0], o4[1], o4[2], o4[3]);
                    } else if (n8_ok && m < p.M) {
                        uint8_t* dst = static_cast<uint8_t*>(p.Y) + (static_cast<size_t>(m) * p.ldy + n8) * 2;
                        *reinterpret_cast<uint4*>(dst) = make_uint4(o4[0], o4[1], o4[2], o4[3]);
                    }
                }
                };
                // Staged tiles need no transpose: the lane writes its own 2-byte elements into the swizzled tile (a warp
                // covers 64 contiguous bytes of one token row: one wavefront), 64 stores and no shuffle chains.
                auto stage16 = [&](auto kBf16) {
                    // byte address of this lane's channel in a row with (row & 7) == j; rows are col0 + 2i + e
                    const int chan = (qd & 1) * 32 + lane;                 // channel inside the 64-channel half
                    uint8_t* const half = sY + (qd >> 1) * (TN * 128) + col0 * 128 + (chan & 7) * 2;
                    uint8_t* rowp[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) rowp[j] = half + ((((chan >> 3) ^ j) & 7) << 4);
#pragma unroll
                    for (int i = 0; i < kNA; ++i) {
                        float y0, y1;
                        unpack_f2(acc[i], y0, y1);
                        uint32_t w;
                        if (decltype(kBf16)::value) { const __nv_bfloat162 v = __floats2bfloat162_rn(y0, y1); w = *reinterpret_cast<const uint32_t*>(&v); }
                        else { const __half2 v = __floats2half2_rn(y0, y1); w = *reinterpret_cast<const uint32_t*>(&v); }
                        *reinterpret_cast<uint16_t*>(rowp[(2 * i) & 7] + (2 * i) * 128) = static_cast<uint16_t>(w);
                        *reinterpret_cast<uint16_t*>(rowp[(2 * i + 1) & 7] + (2 * i + 1) * 128) = static_cast<uint16_t>(w >> 16);
                    }
                };
                using TrueT = std::integral_constant<bool, true>;
                using FalseT = std::integral_constant<bool, false>;
                if (staged) { if (p.ydt == 0) stage16(TrueT{}); else stage16(FalseT{}); }
                else if (p.ydt == 0) store16(TrueT{}, FalseT{});
                else store16(FalseT{}, FalseT{});
#ifdef TWQ_TRACE
                if (trw) TWQ_TR(3, trn, 9);
#endif
                if (staged) {
                    // Asynchronous store: the memory system takes ~2900 cycles to absorb the 32 KB every SM writes at a
                    // tile boundary (all SMs at once); two TMA stores drain that while the next tile is computed.
                    // Rows beyond M and channels beyond N are clipped by the tensor map.
                    fence_proxy_async_smem();
                    named_bar_sync(1, kEpiWarps * 32);
#ifdef TWQ_TRACE
                    if (trw) TWQ_TR(3, trn, 10);
#endif
                    if (warp == kEpiWarp0) {
                        if (lane == 0) {
                            tma_store_2d(&tmY, smem_u32(sY), t.n0, t.m0);
                            if (t.n0 + 64 < p.N) tma_store_2d(&tmY, smem_u32(sY + TN * 128), t.n0 + 64, t.m0);
                            bulk_commit();
                        }
                        y_pending = true;
                    }
                }
            } else if (active && (pl.splits > 1 || (p.ldy & 1) == 0)) {
                // Lane = output channel, register = token: neighbouring lanes trade one value per token pair, so the
                // even lane holds channels (n, n+1) of token 2i and the odd lane channels (n-1, n) of token 2i+1 --
                // half as many store instructions, each lane a 4-byte (FP32 output: 8-byte) word.  N is even.
                // Split-K partials (FP32, workspace [ks][M][N]) take the FP32 form of it.
                const bool odd = lane & 1;
                const int nn = n - (odd ? 1 : 0);
                const bool part = pl.splits > 1;
                float* const y32 = part ? p.ws_part + static_cast<size_t>(t.ks) * p.M * p.N : static_cast<float*>(p.Y);
                const int ld32 = part ? p.N : p.ldy;
                // one straight-line copy per format; the shuffles of eight token pairs are issued together, ahead of
                // the (predicated) stores: with a branch per pair each store waited for its own shuffle (~130 cycles)
                auto store_pairs = [&](auto kKind) {
                    constexpr int kind = decltype(kKind)::value;   // 0 bf16, 1 fp16, 2 fp32
#pragma unroll
                    for (int i0 = 0; i0 < kNA; i0 += 8) {
                        float lo[8], hi[8];
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            float y0, y1;
                            unpack_f2(acc[i0 + j], y0, y1);
                            const float got = __shfl_xor_sync(0xffffffffu, odd ? y0 : y1, 1);
                            lo[j] = odd ? got : y0;               // channels nn, nn + 1
                            hi[j] = odd ? y1 : got;
                        }
#pragma unroll
                        for (int j = 0; j < 8; ++j) {
                            const int m = t.m0 + col0 + (i0 + j) * 2 + (odd ? 1 : 0);
                            if (n_ok && m < p.M) {
                                if (kind == 2) {
                                    *reinterpret_cast<float2*>(y32 + static_cast<size_t>(m) * ld32 + nn) = make_float2(lo[j], hi[j]);
                                } else if (kind == 0) {
                                    *reinterpret_cast<__nv_bfloat162*>(static_cast<__nv_bfloat16*>(p.Y) + static_cast<size_t>(m) * p.ldy + nn) =
                                        __floats2bfloat162_rn(lo[j], hi[j]);
                                } else {
                                    *reinterpret_cast<__half2*>(static_cast<__half*>(p.Y) + static_cast<size_t>(m) * p.ldy + nn) =
                                        __floats2half2_rn(lo[j], hi[j]);
                                }
                            }
                        }
                    }
                };
                if (part || p.ydt == 2) store_pairs(std::integral_constant<int, 2>{});
                else if (p.ydt == 0) store_pairs(std::integral_constant<int, 0>{});
                else store_pairs(std::integral_constant<int, 1>{});
            } else if (active && n_ok) {   // odd row pitch: element stores
#pragma unroll
                for (int i = 0; i < kNA; ++i) {
                    float y2[2];
                    unpack_f2(acc[i], y2[0], y2[1]);
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        const int m = t.m0 + col0 + i * 2 + e;
                        if (m >= p.M) continue;
                        const size_t o = static_cast<size_t>(m) * p.ldy + n;
                        if (p.ydt == 0) static_cast<__nv_bfloat16*>(p.Y)[o] = __float2bfloat16_rn(y2[e]);
                        else if (p.ydt == 1) static_cast<__half*>(p.Y)[o] = __float2half_rn(y2[e]);
                        else static_cast<float*>(p.Y)[o] = y2[e];
                    }
                }
            }
#endif
#ifdef TWQ_TRACE
            if (trw) TWQ_TR(3, trn, 6);
#endif
        }
        TWQ_TG(4);
        if (y_pending) bulk_wait_all0();     // the staged tiles are in global memory before the CTA goes away
    }

    // ---------------------------------------------------------------- teardown
    tc_fence_before();
    __syncthreads();
    TWQ_TG(5);
    if (kPair) cluster_sync_all();   // the leader's MMAs write the peer's TMEM: both CTAs are done before either frees
    if (warp == kCtlWarp0 + 2) {
        tc_fence_after();
        if (kPair) tmem_dealloc_pair<C::kTmemCols>(tmem);
        else tmem_dealloc<C::kTmemCols>(tmem);
    }

    if (pl.splits > 1) {
        // Deterministic split-K fix-up (one unit per cluster when splits > 1, so every CTA of the grid is resident):
        // the CTAs that hold the K splits of one (n-tile, m-tile) wait for one another on the tile counter, then each
        // sums a share of the rows over all partials in split order and writes Y.  The counter runs 0 .. splits
        // (partials parked) .. 2*splits (shares written) and the last CTA leaves it at zero for the next call.
        const Unit t = decode_unit(p, u_begin, rank);
        unsigned* ctr = p.ws_ctr + (t.m0 / TN) * pl.n_tiles + t.n0 / kTileN;
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) {
            atomicAdd(ctr, 1u);
            // the launch is cooperative (every CTA of the grid is resident), so the wait is bounded; a protocol bug
            // becomes a trap (reported as a launch failure), not a hung device
            unsigned seen, spins = 0;
            do {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(ctr) : "memory");
                if (seen < static_cast<unsigned>(pl.splits)) {
                    __nanosleep(64);
                    if (++spins > (1u << 24)) __trap();
                }
            } while (seen < static_cast<unsigned>(pl.splits));
            __threadfence();
        }
        __syncthreads();
        TWQ_TG(6);
        {
            const int rows = min(TN, p.M - t.m0);
            const int r0 = rows * t.ks / pl.splits, r1 = rows * (t.ks + 1) / pl.splits;
            // four channels per thread and step (N is a multiple of 16, the workspace 256-byte aligned): the
            // loads of all splits are independent, the sum is in split order
            for (int idx = threadIdx.x; idx < (r1 - r0) * (kTileN / 4); idx += kThreads) {
                const int mm = t.m0 + r0 + idx / (kTileN / 4), nn = t.n0 + (idx % (kTileN / 4)) * 4;
                if (nn >= p.N) continue;
                float4 y = make_float4(0.f, 0.f, 0.f, 0.f);
                // the loads of all splits in flight together (four at a time), the sum in split order
                for (int z0 = 0; z0 < pl.splits; z0 += 4) {
                    float4 v[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        v[q] = z0 + q < pl.splits
                                   ? __ldcg(reinterpret_cast<const float4*>(p.ws_part + (static_cast<size_t>(z0 + q) * p.M + mm) * p.N + nn))
                                   : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                    for (int q = 0; q < 4; ++q) { y.x += v[q].x; y.y += v[q].y; y.z += v[q].z; y.w += v[q].w; }
                    if (z0 == 0 && idx == threadIdx.x) TWQ_TG(11);
                }
                const size_t o = static_cast<size_t>(mm) * p.ldy + nn;
                if (p.ydt == 2 && (p.ldy & 3) == 0) {
                    *reinterpret_cast<float4*>(static_cast<float*>(p.Y) + o) = y;
                } else if (p.ydt <= 1 && (p.ldy & 3) == 0) {
                    uint2 w;
                    if (p.ydt == 0) {
                        const __nv_bfloat162 a = __floats2bfloat162_rn(y.x, y.y), c = __floats2bfloat162_rn(y.z, y.w);
                        w = make_uint2(*reinterpret_cast<const uint32_t*>(&a), *reinterpret_cast<const uint32_t*>(&c));
                    } else {
                        const __half2 a = __floats2half2_rn(y.x, y.y), c = __floats2half2_rn(y.z, y.w);
                        w = make_uint2(*reinterpret_cast<const uint32_t*>(&a), *reinterpret_cast<const uint32_t*>(&c));
                    }
                    *reinterpret_cast<uint2*>(static_cast<uint8_t*>(p.Y) + o * 2) = w;
                } else {
                    const float yv[4] = {y.x, y.y, y.z, y.w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        if (p.ydt == 0) static_cast<__nv_bfloat16*>(p.Y)[o + e] = __float2bfloat16_rn(yv[e]);
                        else if (p.ydt == 1) static_cast<__half*>(p.Y)[o + e] = __float2half_rn(yv[e]);
                        else static_cast<float*>(p.Y)[o + e] = yv[e];
                    }
                }
            }
        }
        TWQ_TG(9);
        __syncthreads();
        TWQ_TG(10);
        if (threadIdx.x == 0) {
            const unsigned prev = atomicAdd(ctr, 1u);
            if (prev == static_cast<unsigned>(2 * pl.splits - 1)) atomicExch(ctr, 0u);
        }
    }
    TWQ_TG(7);
    if (cs > 1) cluster_sync_all();   // no CTA exits while a peer may still touch its shared memory
    TWQ_TG(8);
}


}  // namespace

template <int TN, int G, bool kDbg, bool kPair = false>
cudaError_t launch_fused_inst(const FusedMaps& maps, const FusedParams& p, cudaStream_t stream) {
    auto kern = fused_dual_linear_kernel<TN, G, kDbg, kPair>;
    constexpr int kMaxDevices = 64;
    static bool attr_done[kMaxDevices] = {};      // function attributes are per device
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices || !attr_done[dev]) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < kMaxDevices) attr_done[dev] = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(p.plan.nclusters * p.plan.cs));
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = static_cast<size_t>(p.plan.smem_bytes);
    cfg.stream = stream;
    cudaLaunchAttribute attrs[3];
    int na = 0;
    if (p.plan.cs > 1) {
        attrs[na].id = cudaLaunchAttributeClusterDimension;
        attrs[na].val.clusterDim.x = static_cast<unsigned>(p.plan.cs);
        attrs[na].val.clusterDim.y = 1;
        attrs[na].val.clusterDim.z = 1;
        ++na;
    }
    if (p.plan.splits > 1) {
        // The split-K fix-up waits for the other CTAs of its tile: a cooperative launch makes the driver guarantee
        // that the whole grid is co-resident (or refuse the launch) whatever else runs on the device.
        attrs[na].id = cudaLaunchAttributeCooperative;
        attrs[na].val.cooperative = 1;
        ++na;
    } else {
        attrs[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attrs[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    cfg.attrs = attrs;
    cfg.numAttrs = static_cast<unsigned>(na);
    return cudaLaunchKernelEx(&cfg, kern, maps.W, maps.Xq, maps.X, maps.L1T, maps.L2T, maps.Y, p);
}

// How many clusters of `cs` CTAs (one CTA per SM) the device can hold at once; 0 on failure.
template <int TN, int G, bool kDbg>
int max_active_clusters_inst(int cs, int num_sms) {
    auto kern = fused_dual_linear_kernel<TN, G, kDbg>;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxDynSmem) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(num_sms / cs * cs));
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = kMaxDynSmem;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = static_cast<unsigned>(cs);
    attr.val.clusterDim.y = 1;
    attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return n;
}


// Explicit instantiations live in fused_inst_tn*.cu (one file per token-tile size, compiled in parallel).
#define TWQ_EXTERN_INST(tn)                                                                                         \
    extern template cudaError_t launch_fused_inst<tn, 128, false>(const FusedMaps&, const FusedParams&, cudaStream_t); \
    extern template cudaError_t launch_fused_inst<tn, 128, true>(const FusedMaps&, const FusedParams&, cudaStream_t);  \
    extern template cudaError_t launch_fused_inst<tn, 64, false>(const FusedMaps&, const FusedParams&, cudaStream_t);  \
    extern template cudaError_t launch_fused_inst<tn, 64, true>(const FusedMaps&, const FusedParams&, cudaStream_t);
TWQ_EXTERN_INST(16)
TWQ_EXTERN_INST(32)
TWQ_EXTERN_INST(64)
TWQ_EXTERN_INST(128)
extern template int max_active_clusters_inst<128, 128, false>(int, int);
extern template cudaError_t launch_fused_inst<128, 128, false, true>(const FusedMaps&, const FusedParams&, cudaStream_t);
extern template cudaError_t launch_fused_inst<128, 128, true, true>(const FusedMaps&, const FusedParams&, cudaStream_t);
extern template cudaError_t launch_fused_inst<128, 64, false, true>(const FusedMaps&, const FusedParams&, cudaStream_t);
extern template cudaError_t launch_fused_inst<128, 64, true, true>(const FusedMaps&, const FusedParams&, cudaStream_t);
#define TWQ_DEFINE_INST(tn)                                                                                  \
    template cudaError_t launch_fused_inst<tn, 128, false>(const FusedMaps&, const FusedParams&, cudaStream_t); \
    template cudaError_t launch_fused_inst<tn, 128, true>(const FusedMaps&, const FusedParams&, cudaStream_t);  \
    template cudaError_t launch_fused_inst<tn, 64, false>(const FusedMaps&, const FusedParams&, cudaStream_t);  \
    template cudaError_t launch_fused_inst<tn, 64, true>(const FusedMaps&, const FusedParams&, cudaStream_t);

}  // namespace twq
