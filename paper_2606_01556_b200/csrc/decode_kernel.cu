// decode_kernel.cu -- the fused dual-branch layer for small batches (M <= kDecodeMaxM tokens), sm_100a.
//
//   Y[m,n] = sum_g sx[m,g]*sw[n,g]*P[m,g,n]  +  sum_j H[m,j]*L2[j,n],
//   P[m,g,n] = sum_{k in g} qx[m,k]*qw[n,k] (exact int32),   H = X*L1 (FP32 accumulate)
//   PAPER.md Eq. 2 (L49-50), Eq. 3 (L62), L177-181 (section 4.3), L193 (groups of G).
//
// At these M the layer streams its weights once: the roofline is HBM bandwidth, and what separates a kernel from
// it is latency -- launch, DRAM round trips, and the dependent chain X*L1 -> (exchange) -> H*L2.
// Everything that does not depend on the activations is therefore in flight from the first instruction, as
// asynchronous bulk copies (TMA, cp.async.bulk) into shared memory that complete on mbarriers:
//
//   W compute warps (14 up to two token tiles, 18 for four) + two producer warps; warp ids in this order:
//   residual     (W - lrw warps) per ring chunk, INT4 -> int8 (each code c becomes the byte 16*c: one shift / and per word,
//                sign for free), warp-level int8 MMAs (activations are the 16-row operand, so a tile is 8 channels),
//                int32 = 256*P folded with both group scales in FP32.  When the CTA has fewer tiles than residual warps
//                the K-groups of a tile are dealt round-robin to P warps and summed in fixed order.
//   warp W       activation-side producer: the Xq boxes of the ring's first lap (one 3-D tensor-map box per chunk = the
//                chunk's K-groups of all tokens, rows beyond M zero-filled by the TMA unit), right after
//                griddepcontrol.wait; idle when the quantizer runs inside the kernel.
//   warp W + 1   producer of everything that does not depend on the activations, issued BEFORE griddepcontrol.wait: first
//                this cluster rank's K slice of L1 (slab layout [K/32][r][32]: one contiguous range) through its own
//                ring, then the residual ring -- the CTA owns `ntile` consecutive 8-channel tiles and R4 is stored
//                tile-major ([N/8][K/G][8][G/2]), so the K-groups [c*gc, (c+1)*gc) of a tile are one contiguous range and
//                chunk c = those ranges of all tiles (1-D bulk copies); also pulls the CTA's rows of L2T into L2.
//   lrw warps    the low-rank chain: X slice -> FP16 shared memory, H partial (FP16 warp MMA, FP32 accumulate),
//                reduce-scatter of the FP32 partials and all-gather of the FP16 result through distributed shared
//                memory (fixed order; mbarriers with cluster-scope release / acquire), then Ylr = H * L2T rows.
//                H never leaves the chip (L177-179).
//   all          single epilogue: sum of the K-parts + Ylr, one rounding, one store (L181).
//
// The two branches only meet in the epilogue, so the weight stream, the low-rank chain and the cluster exchange
// overlap instead of following one another.  Nothing here needs a workspace or a grid-wide barrier.
//
// K order inside an MMA is a free permutation as long as both operands use the same one: a thread takes 16
// consecutive bytes of a row (32 codes, or 8 halves) and uses word s of them in K-step s, for the weights and for
// the activations alike, so every shared-memory read is a 128-bit load of contiguous bytes.
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdio.h>

#include <type_traits>

#include "fused_kernel.h"
#include "sm100_ptx.cuh"
#include "trace.cuh"

namespace twq {

namespace {

// Compute warps per CTA, + the producer warp and the activation-side producer: 14 + 2 = 16 warps, the largest CTA that gets
// 128 registers per thread -- the MT = 1 instantiations need 109-116 and were at the 96-register limit of the 20-warp CTA
// this kernel started with, where ptxas' allocation decided the result (lessons 16 and 20):
// M = 1 / 16 / 32 went 8.9 / 9.9 / 14.8 -> 8.6 / 9.5 / 14.1 us.  The wide variant (18 + 2 warps, 96 registers) remains for
// four token tiles at r > 128, where eight low-rank warps would leave six residual warps (M = 64, r = 256: 33.1 vs 35.0 us;
// at r = 128 the narrow CTA wins, 20.4 vs 21.0 us, and so it does in the 4-bit low-rank mode, 28.1 vs 34.0 us).
__host__ __device__ constexpr int dec_warps(bool wide) { return wide ? 18 : 14; }
__host__ __device__ constexpr int dec_threads(bool wide) { return (dec_warps(wide) + 2) * 32; }
inline bool dec_is_wide(int mt, int r, int quant) { return mt == 4 && r > 128 && quant != 2; }
constexpr int kMaxSlots = 8, kMaxL1Slots = 4;
constexpr int kTB = 3;                              // tiles whose MMA chains a residual warp interleaves
constexpr int kJT = 8;                              // 8-wide j tiles of H one low-rank warp can own
constexpr int kDecSmemMax = 232448 - 1024;

enum : int { D_FULL = 0, D_EMPTY = D_FULL + kMaxSlots, D_L1FULL = D_EMPTY + kMaxSlots, D_L1EMPTY = D_L1FULL + kMaxL1Slots,
             D_X1 = D_L1EMPTY + kMaxL1Slots, D_X2, D_XQ, D_COUNT };

__device__ __forceinline__ uint32_t d_lo16(uint32_t w) { return (w << 4) & 0xF0F0F0F0u; }  // 16*code, even k
__device__ __forceinline__ uint32_t d_hi16(uint32_t w) { return w & 0xF0F0F0F0u; }         // 16*code, odd k

// D[16x8] (s32) += A[16x32] (s8, row) * B[32x8] (s8, col)
__device__ __forceinline__ void imma_16832(int (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                           uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+r"(d[0]), "+r"(d[1]), "+r"(d[2]), "+r"(d[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// D[16x8] (s32) = A * B (zero accumulator: the first K-step of a chain; saves the four moves that clear D)
__device__ __forceinline__ void imma_16832_z(int (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                             uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%10,%10,%10};"
        : "=r"(d[0]), "=r"(d[1]), "=r"(d[2]), "=r"(d[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1), "r"(0));
}
// D[16x8] (f32) += A[16x16] (f16, row) * B[16x8] (f16, col)
__device__ __forceinline__ void hmma_16816(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                           uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

__device__ __forceinline__ uint4 ldg_nc(const void* p) {
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
    return v;
}
// plain (coherent) 128-bit global load: for buffers the previous kernel of the stream wrote (X)
__device__ __forceinline__ uint4 ldg_v4(const void* p) {
    uint4 v;
    asm volatile("ld.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ float ldg_f32(const float* p) {
    float v;
    asm volatile("ld.global.f32 %0, [%1];" : "=f"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ uint4 lds_v4(uint32_t a) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ uint2 lds_v2(uint32_t a) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t a) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}

// two BF16 (packed) -> two FP16 (packed), exact for 2^-14 <= |x| <= 65504, saturating above
__device__ __forceinline__ uint32_t bf2_to_h2(uint32_t w) {
    float lo = __uint_as_float(w << 16), hi = __uint_as_float(w & 0xFFFF0000u);
    lo = fminf(fmaxf(lo, -65504.0f), 65504.0f);
    hi = fminf(fmaxf(hi, -65504.0f), 65504.0f);
    const __half2 h2 = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<const uint32_t*>(&h2);
}

__device__ __forceinline__ float ld_dsmem_f(uint32_t cluster_addr) {
    float v;
    asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(cluster_addr) : "memory");
    return v;
}
__device__ __forceinline__ void st_dsmem_u16(uint32_t cluster_addr, uint16_t v) {
    asm volatile("st.shared::cluster.u16 [%0], %1;" ::"r"(cluster_addr), "h"(v) : "memory");
}
__device__ __forceinline__ void st_dsmem_u32(uint32_t cluster_addr, uint32_t v) {
    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(cluster_addr), "r"(v) : "memory");
}
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

template <int kW>
__device__ __forceinline__ void lds_words(uint32_t (&dst)[kW], uint32_t a) {
    if constexpr (kW == 4) {
        const uint4 v = lds_v4(a);
        dst[0] = v.x; dst[1] = v.y; dst[2] = v.z; dst[3] = v.w;
    } else {
        const uint2 v = lds_v2(a);
        dst[0] = v.x; dst[1] = v.y;
    }
}

}  // namespace

// The in-kernel activation quantizer and its all-gather (kMode >= 1), run by the residual warps.
template <int G, int MT, bool kL4>
__device__ __forceinline__ void decode_quantize_share(const DecodeParams& p, uint8_t* dsm, int rank, int cs, int rw, int lane, int nrw,
                                                   int lrw, bool xq_bulk) {
    // (rank, cs) = the cluster rank and size, or (0, 1) in local mode: one or two tokens, where every CTA quantizes the whole
    // row block itself (M x K elements, L2-resident after the first cluster) and nothing is exchanged -- the all-gather's skew
    // and remote latency (~1 us) cost more than the extra items.  Local mode runs the bulk branch with no peer to copy to.
    constexpr int kMp = 16 * MT;
    const int ng = p.ng;
    float* sSx = reinterpret_cast<float*>(dsm + p.off_sx);
    const uint32_t bar0 = smem_u32(dsm + p.off_bar);
#define DBAR(i) (bar0 + 8u * static_cast<uint32_t>(i))
    // ---- steps a1-a2 inside the kernel (Eq. 1; the FP32 operation order of
    // include/twq.h, bit for bit the codes and scales twq_quantize_act writes).  Cluster rank q quantizes the
    // K-groups [ng*q/cs, ng*(q+1)/cs) of every token and stores codes and scales into EVERY peer's shared memory
    // ([g][token][G/2], the layout the MMA fragments read without bank conflicts): the activation tile is
    // quantized once per cluster and reused by all its CTAs and tiles (L179).
    uint8_t* sXq = dsm + p.off_xq;
    // Rows beyond M are written by nobody and stay whatever the shared memory held: row m of the MMA's activation
    // operand only reaches row m of its result, and no result row >= M is ever read (clearing the 32 KB tile cost
    // 1.1 us at the head of the critical path; in-kernel timeline, r02).
    const int gq0 = static_cast<int>(static_cast<unsigned>(ng) * rank / cs);
    const int ngq = static_cast<int>(static_cast<unsigned>(ng) * (rank + 1) / cs) - gq0;
    const int items = p.M * ngq;
    const uint16_t* X = static_cast<const uint16_t*>(p.X);
    TWQ_DSTAMP(21);
    // This loop heads the critical path of the call and is one dependent chain per warp: every instruction in it is paid in
    // full (a software prefetch of four passes with its index divisions cost 0.6 us at M = 1; measured, r02).
    bool waited = cs <= 1;
    TWQ_DCLK(4);
    // One pass of the residual warps covers nrw * 32 / (G/8) items with 8 elements per lane.  Where that is not enough
    // (M >= 16 at 16 ranks) a lane takes 16 elements instead: one pass where there were two, and every pass is a DRAM round
    // trip plus ~150 dependent instructions at the head of the critical path (M = 16: 3.0 -> 1.9 us; in-kernel timeline, r02).
    auto pass = [&](auto epl_c) {
        constexpr int EPL = decltype(epl_c)::value;          // elements per lane: 8 or 16
        constexpr int kLPI = G / EPL;                        // lanes per (token, group)
        constexpr int kIPW = 32 / kLPI;                      // (token, group) items per warp pass
        constexpr int kV = EPL / 8;                          // 16-byte loads per lane
        const int li = lane % kLPI, sub = lane / kLPI;
#pragma unroll 1
        for (int base0 = rw * kIPW; base0 < items; base0 += nrw * kIPW) {
            const int it = base0 + sub;
            const bool on = it < items;                      // whole items are on or off: the shuffles below stay inside one
            int m = 0, gi = 0;
            if (on) {
                if (ngq == 1) { m = it; }
                else if (ngq == 2) { m = it >> 1; gi = it & 1; }
                else { m = it / ngq; gi = it - m * ngq; }
            }
            const int g = gq0 + gi;
            uint4 vld[kV];
#pragma unroll
            for (int v = 0; v < kV; ++v)
                vld[v] = on ? ldg_v4(X + static_cast<size_t>(m) * p.ldx + g * G + li * EPL + v * 8) : make_uint4(0u, 0u, 0u, 0u);
            if (!waited) {                                   // warp-uniform; after the loads are in flight
                cluster_wait();                              // every CTA of the cluster is running (its barriers exist)
                waited = true;
            }
            float x[EPL];
#pragma unroll
            for (int v = 0; v < kV; ++v) {
                const uint32_t w[4] = {vld[v].x, vld[v].y, vld[v].z, vld[v].w};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    x[v * 8 + 2 * i] = __uint_as_float(w[i] << 16);              // BF16 -> FP32, exact (0 when off)
                    x[v * 8 + 2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
                }
            }
            if (on && p.tinv != nullptr) {
#pragma unroll
                for (int v = 0; v < EPL / 4; ++v) {
                    const float4 t = __ldg(reinterpret_cast<const float4*>(p.tinv + g * G + li * EPL) + v);
                    x[4 * v] = __fmul_rn(x[4 * v], t.x); x[4 * v + 1] = __fmul_rn(x[4 * v + 1], t.y);
                    x[4 * v + 2] = __fmul_rn(x[4 * v + 2], t.z); x[4 * v + 3] = __fmul_rn(x[4 * v + 3], t.w);
                }
            }
            float amax = 0.0f;
#pragma unroll
            for (int i = 0; i < EPL; ++i) amax = fmaxf(amax, fabsf(x[i]));
#pragma unroll
            for (int d = kLPI / 2; d >= 1; d >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, d));
            const float sc = __fdiv_rn(fmaxf(amax, 0x1p-30f), 7.0f);
            const float inv = __fdiv_rn(1.0f, sc);
            uint32_t pk[kV];
#pragma unroll
            for (int v = 0; v < kV; ++v) {
                pk[v] = 0u;
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    int q = __float2int_rn(__fmul_rn(x[v * 8 + i], inv));        // round-half-to-even
                    q = max(-7, min(7, q));
                    pk[v] |= (static_cast<uint32_t>(q) & 0xFu) << (4 * i);       // low nibble = even k
                }
            }
            if (on) {
                uint32_t* qd = reinterpret_cast<uint32_t*>(sXq + (g * kMp + m) * (G / 2) + li * (EPL / 2));
#pragma unroll
                for (int v = 0; v < kV; ++v) {
                    if (xq_bulk) {
                        qd[v] = pk[v];
                    } else {
                        const uint32_t qa = smem_u32(qd + v);
                        for (int pr = 0; pr < cs; ++pr) st_dsmem_u32(mapa_u32(qa, pr), pk[v]);
                    }
                    if (p.xq_out != nullptr)
                        *reinterpret_cast<uint32_t*>(p.xq_out + static_cast<size_t>(m) * (p.K >> 1) + g * (G / 2) + li * (EPL / 2) + v * 4) = pk[v];
                }
                if (li == 0) {
                    const float s8 = sc * 0x1p-8f;                   // MMA operands are 16*code
                    if (xq_bulk) {
                        sSx[g * kMp + m] = s8;
                    } else {
                        const uint32_t sa = smem_u32(sSx + g * kMp + m);
                        for (int pr = 0; pr < cs; ++pr) st_dsmem_u32(mapa_u32(sa, pr), __float_as_uint(s8));
                    }
                    if (p.sx_out != nullptr) p.sx_out[static_cast<size_t>(m) * ng + g] = sc;
                }
            }
        }
    };
    if (items > nrw * (32 / (G / 8))) pass(std::integral_constant<int, 16>{});
    else pass(std::integral_constant<int, 8>{});
    if (!waited) cluster_wait();                         // warps without an item
    TWQ_DCLK(5);
    TWQ_DSTAMP(22);
    if (xq_bulk) fence_proxy_async_smem();               // the bulk copies below read what this thread stored
    TWQ_DSTAMP(24);
    named_bar_sync(2, nrw * 32);                         // this CTA's share is stored (in bulk mode: in its own shared memory)
    TWQ_DSTAMP(23);
    if constexpr (kL4) asm volatile("bar.arrive 4, %0;" ::"r"((nrw + lrw) * 32) : "memory");   // q4lr stage 1 may read it
    if (xq_bulk) {
        // All-gather: this rank's K-groups (contiguous in [g][token][G/2] and [g][token]) go to every peer as two bulk
        // copies through distributed shared memory, completing on the peer's barrier.  Per-lane remote stores were 450
        // remote operations per pass and 1.8 us at M = 16 (in-kernel timeline, r02).
        if (rw == 0 && lane < cs && lane != rank && ngq > 0) {
            const uint32_t cs_a = smem_u32(sXq + gq0 * kMp * (G / 2)), ss_a = smem_u32(sSx + gq0 * kMp);
            const uint32_t rb = mapa_u32(DBAR(D_XQ), static_cast<uint32_t>(lane));
            bulk_copy_to_peer(mapa_u32(cs_a, lane), cs_a, static_cast<uint32_t>(ngq) * kMp * (G / 2), rb);
            bulk_copy_to_peer(mapa_u32(ss_a, lane), ss_a, static_cast<uint32_t>(ngq) * kMp * 4, rb);
        }
        mbar_wait_a(DBAR(D_XQ), 0);                      // every peer's share has arrived here
    } else if (cs > 1) {
        if (rw == 0 && lane < cs) mbar_arrive_remote(mapa_u32(DBAR(D_XQ), static_cast<uint32_t>(lane)));
        mbar_wait_cluster_a(DBAR(D_XQ), 0);              // every rank's share has arrived here
    }
#undef DBAR
}

// kMode >= 1 (kQ): the activation quantizer (steps a1-a2) runs inside this kernel: every cluster rank quantizes 1/cs of the
// K-groups of all tokens and the cluster all-gathers codes and scales through distributed shared memory (twq_dual_linear_x).
// kMode == 2 (kL4): in addition the low-rank branch is the paper's own 4-bit pipeline (R18-R22):
//   stage 1   H partial = sum over this rank's K-groups of sx*su*(qx . qu): the SAME quantized activation tile the residual
//             uses (L179), int8 warp MMAs on 16*code like the residual, against the U section of the q4lr blob;
//   exchange  FP32 sum in rank order, FP32 H to every peer;
//   re-quantization on the fly (L181): per token and group of gr rank indices, s_H = max(amax, 2^-30)/7 and packed 4-bit
//             Q_H in shared memory, in the activation quantizer's FP32 operation order;
//   stage 2   Ylr = sum_h s_H*sv*(Q_H . qv): a second int8 MMA against the V section, folded into the same epilogue.
template <int G, int MT, bool kDbg, int kMode, bool kWide>
__global__ void __launch_bounds__(dec_threads(kWide), 1)
decode_dual_linear_kernel(const __grid_constant__ CUtensorMap tmXq, const __grid_constant__ DecodeParams p) {
    constexpr bool kQ = kMode >= 1, kL4 = kMode == 2;
    constexpr int kDecWarps = dec_warps(kWide);
    extern __shared__ uint8_t dsm_raw[];
    // 1024-byte aligned base; the same offset in every CTA of the cluster (DSMEM addresses are formed from local ones)
    uint8_t* dsm = dsm_raw + ((1024u - (smem_u32(dsm_raw) & 1023u)) & 1023u);
    constexpr int kW = G / 32;            // 32-bit words per thread per row per group (4 or 2)
    constexpr int kBlk = 4 * G;           // bytes of one (8-channel tile, K-group) block of R4
    constexpr int kMp = 16 * MT;          // padded tokens

    float* sHpart = reinterpret_cast<float*>(dsm + p.off_hpart);   // [kMp][r] FP32 partial of H (this CTA's K slice)
    __half* sH = reinterpret_cast<__half*>(dsm + p.off_h);         // [kMp][r + 8] FP16 H (whole K)
    float* sYlr = reinterpret_cast<float*>(dsm + p.off_ylr);       // [kMp][tmax * 8]
    float* sSx = reinterpret_cast<float*>(dsm + p.off_sx);         // [ng][kMp] activation scales * 2^-8
    float* sRes = reinterpret_cast<float*>(dsm + p.off_res);       // [tile * P + part][kMp][8]
    __half* sXs = reinterpret_cast<__half*>(dsm + p.off_xs);       // [kMp][xs_stride] FP16 copy of the X slice

    // the warp index through a shuffle: the compiler then knows it is warp-uniform, and with it every role branch and loop bound
    // derived from it (otherwise each mma.sync in those loops is preceded by a WARPSYNC)
    const int warp = __shfl_sync(0xffffffffu, static_cast<int>(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
    const int gid = lane >> 2, tid4 = lane & 3;
    const int r = p.r, ng = p.ng, cs = p.cs, lrw = p.lrw;
    const int nrw = kDecWarps - lrw;
    constexpr int kTPW = MT == 1 ? 6 : (MT == 2 ? 3 : 2);   // 8-channel tiles one residual warp can own (its accumulators)
    // Warp roles by id: [0, nrw) residual, [nrw, 18) low-rank chain, 18 spare, 19 producer.  The scheduler of an SM
    // sub-partition favours HIGHER warp ids: the dependent low-rank chain and the producer must not queue behind the
    // residual warps (with the chain in warps 0-3 every step of it waited for an issue slot; in-kernel timeline, r02).
    const bool is_lr = warp >= nrw && warp < kDecWarps;
    const int lw = warp - nrw;                  // index among the low-rank warps
    const int rank = cs > 1 ? static_cast<int>(cluster_ctarank()) : 0;
    // 8-channel tiles of this CTA: an even split of the n_tiles over the grid
    // (32-bit arithmetic: n_tiles * grid < 2^31 for every shape the planner accepts; a 64-bit division is ~100 instructions)
    const int tile0 = static_cast<int>(blockIdx.x * static_cast<unsigned>(p.n_tiles) / gridDim.x);
    const int ntile = static_cast<int>((blockIdx.x + 1u) * static_cast<unsigned>(p.n_tiles) / gridDim.x) - tile0;
    // stage-1 K slice of this cluster rank, in 32-wide slabs
    const int units = kL4 ? ng : (p.K >> 5);                // q4lr: the unit of the stage-1 slice is one K-group of U
    const int u0 = static_cast<int>(static_cast<unsigned>(units) * static_cast<unsigned>(rank) / static_cast<unsigned>(cs));
    const int nu = r > 0 ? static_cast<int>(static_cast<unsigned>(units) * static_cast<unsigned>(rank + 1) / static_cast<unsigned>(cs)) - u0 : 0;
    const int nl1 = (nu + p.sc - 1) / p.sc;                 // stage-1 ring chunks
    const int slab_bytes = kL4 ? r * (G / 2) + r * 2 : r * 64;
    // Residual warps form a (tile group x K part) grid: TG groups of at most kTPW tiles, P = nrw / TG warps per group,
    // warp `part` of a group taking the K-groups g = part (mod P).  A warp thus expands the activation fragments of a
    // K-group once for all its tiles, and its tiles are independent MMA chains.
    const int TG = ntile > 0 ? (ntile + kTPW - 1) / kTPW : 1;
    const int tpg = (ntile + TG - 1) / TG;      // tiles per group
    int P = nrw / TG;
    P = max(1, min(P, ng));
    const int nloc = p.tmax * 8;
    const int hstride = r + 8;

    // The in-kernel quantizer's all-gather: per-lane remote stores for a handful of tokens (lowest latency), bulk copies through
    // distributed shared memory above that (one remote transaction per warp and peer does not scale with M).
    // (only where the low-rank chain waits for the quantized tile too: in the FP16 mode the all-gather is off the critical
    // path at these M and the local mode measured 0.3 us slower)
    const bool xq_local = kL4 && cs > 1 && p.M <= 2;
    const bool xq_bulk = kQ && cs > 1 && (p.M > 4 || xq_local);
    TWQ_DSTAMP(0);
    const uint32_t bar0 = smem_u32(dsm + p.off_bar);
#define DBAR(i) (bar0 + 8u * static_cast<uint32_t>(i))
    // Barrier initialisation: one thread per barrier without the in-kernel quantizer, serial with it.  Measured, not
    // reasoned: at the 96-register limit of the former 20-warp CTA the parallel form made the quantizer instantiations spill
    // (-0.5 us at M = 1) and the serial form the other one; with 16-warp CTAs at 128 registers nothing spills any more, and
    // the parallel form is still 0.15 us slower in the quantizer instantiations (A/B of both libraries in one run, r02).
    if (!kQ && threadIdx.x < D_COUNT) {
        const int i = threadIdx.x;
        int count = 1;                                                        // D_FULL, D_L1FULL: the producer's expect_tx
        if (i >= D_EMPTY && i < D_EMPTY + kMaxSlots) count = nrw;
        else if (i >= D_L1EMPTY && i < D_L1EMPTY + kMaxL1Slots) count = lrw > 0 ? lrw : 1;
        else if (i == D_X1 || i == D_X2 || i == D_XQ) count = cs;
        mbar_init(reinterpret_cast<uint64_t*>(dsm + p.off_bar) + i, count);
        fence_mbar_init();
    }
    if (kQ && threadIdx.x == 0) {
        uint64_t* bars = reinterpret_cast<uint64_t*>(dsm + p.off_bar);
        for (int i = 0; i < kMaxSlots; ++i) { mbar_init(&bars[D_FULL + i], 1); mbar_init(&bars[D_EMPTY + i], nrw); }
        for (int i = 0; i < kMaxL1Slots; ++i) { mbar_init(&bars[D_L1FULL + i], 1); mbar_init(&bars[D_L1EMPTY + i], lrw > 0 ? lrw : 1); }
        mbar_init(&bars[D_X1], cs);
        mbar_init(&bars[D_X2], cs);
        mbar_init(&bars[D_XQ], xq_bulk ? 1 : cs);
        fence_mbar_init();
        if (xq_bulk) {
            // the in-kernel quantizer's all-gather arrives as bulk copies from the cs - 1 peers: every K-group this rank does
            // not quantize itself, all kMp token rows of codes and scales
            const int own = static_cast<int>(static_cast<unsigned>(ng) * (rank + 1) / cs) - static_cast<int>(static_cast<unsigned>(ng) * rank / cs);
            mbar_arrive_expect_tx_a(DBAR(D_XQ), xq_local ? 0u : static_cast<uint32_t>(ng - own) * (kMp * (G / 2) + kMp * 4));
        }
    }
    __syncthreads();
    // split cluster barrier: "my mbarriers exist".  The low-rank warps wait for it before their first remote arrive,
    // everyone else before exit; it costs nothing on the way in.
    if (cs > 1) cluster_arrive_relaxed();
    pdl_launch_dependents();
    TWQ_DSTAMP(1);

    if (warp == kDecWarps + 1) {
        // ================================================================ producer warp
        // One bulk copy occupies its issuing thread for as long as the copy engine needs for the copies queued before
        // it (~60 GB/s per SM with the whole grid streaming; in-kernel timeline, r02), so (a) the copies of a lap are
        // dealt to the 32 lanes, and (b) the order of issue is the order of need: the stage-1 slice of L1 (the dependent
        // chain X*L1 -> exchange -> H*L2 is the critical path) before the residual stream.
        const uint32_t l1ring = smem_u32(dsm + p.off_l1);
        const uint8_t* l1src = static_cast<const uint8_t*>(p.L1D) + static_cast<size_t>(u0) * slab_bytes;
        const uint64_t pol_keep = policy_evict_last();           // every cluster reads all of L1: keep it in L2
        const uint64_t pol = policy_evict_first();               // the residual is streamed once
        auto copy_l1 = [&](int i, int slot) {
            const int cnt = min(p.sc, nu - i * p.sc);
            mbar_arrive_expect_tx_a(DBAR(D_L1FULL + slot), static_cast<uint32_t>(cnt) * slab_bytes);
            bulk_load_1d_a(l1ring + slot * (p.sc * slab_bytes), l1src + static_cast<size_t>(i) * p.sc * slab_bytes,
                           static_cast<uint32_t>(cnt) * slab_bytes, DBAR(D_L1FULL + slot), pol_keep);
        };
        const int l1_first = r > 0 ? min(p.l1_slots, nl1) : 0;
        if (lane < l1_first) copy_l1(lane, lane);                // first lap of the stage-1 ring: one lane per chunk
        __syncwarp();
        const uint32_t ring = smem_u32(dsm + p.off_ring);
        const uint8_t* src0 = p.R4 + static_cast<size_t>(tile0) * ng * kBlk;
        const uint32_t xq_bytes = kQ ? 0u : static_cast<uint32_t>(p.gc) * kMp * (G / 2);   // a full box, zero-filled beyond M / ng
        const uint32_t sw_bytes = static_cast<uint32_t>(ntile) * ng * 16;        // this CTA's FP16 group scales
        const int first = ntile > 0 ? min(p.nslots, p.nchunks) : 0;
        auto arm = [&](int c, int slot) {
            const int gcnt = min(p.gc, ng - c * p.gc);
            mbar_arrive_expect_tx_a(DBAR(D_FULL + slot),
                                    static_cast<uint32_t>(ntile) * gcnt * kBlk + xq_bytes + (c == 0 ? sw_bytes : 0u));
        };
        auto copy_w = [&](int c, int slot, int t) {
            const int g0 = c * p.gc, gcnt = min(p.gc, ng - g0);
            bulk_load_1d_a(ring + slot * p.slot_bytes + t * (p.gc * kBlk), src0 + (static_cast<size_t>(t) * ng + g0) * kBlk,
                           static_cast<uint32_t>(gcnt) * kBlk, DBAR(D_FULL + slot), pol);
        };
        if (lane == 0)
            for (int c = 0; c < first; ++c) arm(c, c);
        __syncwarp();
        asm volatile("bar.arrive 3, 64;" ::: "memory");          // the barriers are armed: the activation-side warp may issue
        // weights do not depend on the previous kernel: the whole first lap goes out before griddepcontrol.wait
        for (int i = lane; i < first * ntile; i += 32) copy_w(i / ntile, i / ntile, i % ntile);
        if (lane == 31 && ntile > 0) {
            // the scales ride on the first chunk's barrier (every residual warp waits for it first); stage 2 reads this
            // CTA's rows of L2T straight from L2
            bulk_load_1d_a(smem_u32(dsm + p.off_sw), p.sw16 + static_cast<size_t>(tile0) * ng * 8, sw_bytes, DBAR(D_FULL), pol);
            if (r > 0) {
                const uint32_t trow = kL4 ? static_cast<uint32_t>(p.nh) * 8 * (p.grs / 2) : 8u * r * 2;   // bytes of a tile's stage-2 operand
                bulk_prefetch_l2(static_cast<const uint8_t*>(p.L2T) + static_cast<size_t>(tile0) * trow, static_cast<uint32_t>(ntile) * trow);
            }
        }
        TWQ_DSTAMP(2);
        pdl_wait();                                              // later laps carry Xq boxes (twq_quantize_act's output)
        TWQ_DSTAMP(3);
        // later laps of both rings (long K / many tiles only): lane 0 refills stage-1 chunks, the warp refills residual chunks
        {
            int s1 = 0, lap1 = 1, i1n = l1_first;                // stage-1 ring
            int slot = 0, lap = 1, c = first;                    // residual ring
            while (i1n < nl1 || (ntile > 0 && c < p.nchunks)) {
                // stage-1 refills never wait for residual consumers and vice versa: poll both, act on what is free
                if (i1n < nl1) {
                    bool ok = false;
                    if (lane == 0) ok = mbar_try_wait_a(DBAR(D_L1EMPTY + s1), (lap1 - 1) & 1);
                    ok = __shfl_sync(0xffffffffu, ok ? 1 : 0, 0) != 0;
                    if (ok) {
                        if (lane == 0) copy_l1(i1n, s1);
                        ++i1n;
                        if (++s1 == p.l1_slots) { s1 = 0; ++lap1; }
                    }
                }
                if (ntile > 0 && c < p.nchunks) {
                    bool ok = false;
                    if (lane == 0) ok = mbar_try_wait_a(DBAR(D_EMPTY + slot), (lap - 1) & 1);
                    ok = __shfl_sync(0xffffffffu, ok ? 1 : 0, 0) != 0;
                    if (ok) {
                        if (lane == 0) arm(c, slot);
                        __syncwarp();
                        for (int t = lane; t < ntile; t += 32) copy_w(c, slot, t);
                        if (!kQ && lane == 31) tma_load_3d_a(ring + slot * p.slot_bytes + p.xq_off, &tmXq, DBAR(D_FULL + slot), 0, c * p.gc, 0);
                        ++c;
                        if (++slot == p.nslots) { slot = 0; ++lap; }
                    }
                }
            }
        }
    } else if (warp == kDecWarps) {
        // ================================================================ activation-side producer
        // The Xq boxes of the first lap.  They must wait for the previous kernel (twq_quantize_act), the weights need not:
        // issued from the producer warp behind the weight copies they were the LAST bytes of every chunk to land (the
        // copy engine works in order) and no chunk was complete before 2.4 us; from their own warp they go out as soon
        // as the previous kernel is done and land first.
        named_bar_sync(3, 64);                                   // the chunk barriers are armed
        pdl_wait();
        const int first = (!kQ && ntile > 0) ? min(p.nslots, p.nchunks) : 0;
        if (lane < first)
            tma_load_3d_a(smem_u32(dsm + p.off_ring) + lane * p.slot_bytes + p.xq_off, &tmXq, DBAR(D_FULL + lane), 0,
                          lane * p.gc, 0);
        TWQ_DSTAMP(4);
    } else if (is_lr) {
        // ================================================================ low-rank chain
        const int lrt = threadIdx.x - nrw * 32, nlr = lrw * 32;
        pdl_wait();                                              // X comes from the previous kernel of the stream
        TWQ_DSTAMP(2);
        uint8_t* sQH = dsm + p.off_qh;                           // q4lr: packed Q_H [nh][kMp][grs/2]
        float* sSH = reinterpret_cast<float*>(dsm + p.off_sh);   // q4lr: s_H * 2^-8 [nh][kMp]
        float* sH32 = reinterpret_cast<float*>(dsm + p.off_h);   // q4lr: FP32 H [kMp][r]
        if constexpr (kL4) {
            // Q_H rows beyond M and the padding beyond gr codes are zero codes; nothing else to stage: stage 1 multiplies the
            // quantized activation tile, and this rank's K-groups of it are the ones this CTA quantized itself
            for (int i = lrt; i < p.nh * kMp * (p.grs / 8); i += nlr) reinterpret_cast<uint32_t*>(sQH)[i] = 0u;
            for (int i = lrt; i < p.nh * kMp; i += nlr) sSH[i] = 0.0f;
            asm volatile("bar.sync 4, %0;" ::"r"((nrw + lrw) * 32) : "memory");   // this CTA's share of Xq / sx is in shared memory
        } else {
            // X slice (tokens x 32*nu k, BF16 -> FP16) into shared memory, four 16-byte loads in flight per thread
            const uint16_t* X = static_cast<const uint16_t*>(p.X);
            const int chunks = nu * 4;                           // 16-byte chunks per token row
            const int total = p.xrows * chunks;
            // element i = (token i / chunks, chunk i % chunks): one division per thread, then (token, chunk) advance by
            // the constant (nlr / chunks, nlr % chunks) with a carry
            int m = chunks > 0 ? lrt / chunks : 0, cq = lrt - m * chunks;
            const int dm = chunks > 0 ? nlr / chunks : 0, dc = nlr - dm * chunks;
            for (int i0 = lrt; i0 < total; i0 += 4 * nlr) {
                uint4 v[4];
                int mm[4], cc[4];
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    mm[q] = m; cc[q] = cq;
                    v[q] = make_uint4(0, 0, 0, 0);
                    if (i0 + q * nlr < total && m < p.M)
                        v[q] = ldg_v4(X + static_cast<size_t>(m) * p.ldx + u0 * 32 + cq * 8);
                    m += dm; cq += dc;
                    if (cq >= chunks) { cq -= chunks; ++m; }
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    if (i0 + q * nlr < total) {
                        uint4 w = v[q];
                        w.x = bf2_to_h2(w.x); w.y = bf2_to_h2(w.y); w.z = bf2_to_h2(w.z); w.w = bf2_to_h2(w.w);
                        *reinterpret_cast<uint4*>(sXs + mm[q] * p.xs_stride + cc[q] * 8) = w;
                    }
                }
            }
        }
        named_bar_sync(1, nlr);
        TWQ_DSTAMP(3);
        // ---- stage 1: partial H of this CTA's K slice; low-rank warp lw owns the j tiles lw, lw + lrw, ...
        // The chain is latency-bound and runs one warp per scheduler, so the loop must be tight: the body is instantiated
        // for NQ = 1 / 2 / 4 / 8 j tiles per warp with no guard inside (a missing j tile repeats the last one and is
        // dropped at the write-out), fragment addresses are hoisted and advance by constants, all fragments of a slab
        // are loaded before its MMAs, and the MMAs are interleaved over the j tiles (with per-load address arithmetic
        // and guards the same loop took 1200 cycles per slab; in-kernel timeline, r02).
        const int njt = r >> 3;
        const int nq_need = njt > lw ? (njt - lw + lrw - 1) / lrw : 0;          // j tiles of this warp
        auto stage1 = [&](auto nq_c) {
            constexpr int NQ = decltype(nq_c)::value;
            float d[NQ][MT][4];
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int t = 0; t < MT; ++t)
#pragma unroll
                    for (int e = 0; e < 4; ++e) d[q][t][e] = 0.0f;
            const uint32_t l1lane = smem_u32(dsm + p.off_l1) + gid * 64 + tid4 * 16;
            uint32_t loff[NQ];
#pragma unroll
            for (int q = 0; q < NQ; ++q) loff[q] = static_cast<uint32_t>(min(lw + q * lrw, max(njt - 1, 0))) * 512u;
            uint32_t xs_a = smem_u32(sXs) + (gid * p.xs_stride + tid4 * 8) * 2;   // advances 64 bytes per slab
            // with at most 8 tokens only rows 0..7 are staged: the gid + 8 fragment re-reads row gid (its output rows are dropped)
            const uint32_t xrow8 = p.xrows > 8 ? 8u * p.xs_stride * 2u : 0u;
            const uint32_t chunk_bytes = static_cast<uint32_t>(p.sc) * slab_bytes;
            int slot = 0, lap = 0;
            uint32_t slot_a = 0;
            TWQ_DCLK(0);
#pragma unroll 1
            for (int i = 0; i < nl1; ++i) {
                mbar_wait_a(DBAR(D_L1FULL + slot), lap & 1);
                const int cnt = min(p.sc, nu - i * p.sc);
                uint32_t la = l1lane + slot_a;
#pragma unroll 2
                for (int sl = 0; sl < cnt; ++sl, la += slab_bytes, xs_a += 64) {
                    uint4 a[MT][2];
                    uint4 l[NQ];
#pragma unroll
                    for (int t = 0; t < MT; ++t) {
                        a[t][0] = lds_v4(xs_a + t * 2 * xrow8);
                        a[t][1] = lds_v4(xs_a + t * 2 * xrow8 + xrow8);
                    }
#pragma unroll
                    for (int q = 0; q < NQ; ++q) l[q] = lds_v4(la + loff[q]);
#pragma unroll
                    for (int q = 0; q < NQ; ++q)
#pragma unroll
                        for (int t = 0; t < MT; ++t) hmma_16816(d[q][t], a[t][0].x, a[t][1].x, a[t][0].y, a[t][1].y, l[q].x, l[q].y);
#pragma unroll
                    for (int q = 0; q < NQ; ++q)
#pragma unroll
                        for (int t = 0; t < MT; ++t) hmma_16816(d[q][t], a[t][0].z, a[t][1].z, a[t][0].w, a[t][1].w, l[q].z, l[q].w);
                }
                __syncwarp();
                if (lane == 0) mbar_arrive_a(DBAR(D_L1EMPTY + slot));
                slot_a += chunk_bytes;
                if (++slot == p.l1_slots) { slot = 0; slot_a = 0; ++lap; }
            }
            TWQ_DSTAMP(4);
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                const int jt = lw + q * lrw;
                if (jt < njt) {
                    const int j = jt * 8 + tid4 * 2;
#pragma unroll
                    for (int t = 0; t < MT; ++t) {
                        *reinterpret_cast<float2*>(sHpart + (t * 16 + gid) * r + j) = make_float2(d[q][t][0], d[q][t][1]);
                        *reinterpret_cast<float2*>(sHpart + (t * 16 + gid + 8) * r + j) = make_float2(d[q][t][2], d[q][t][3]);
                    }
                }
            }
        };
        // ---- q4lr stage 1: the same loop shape on int8 MMAs.  A j tile of one K-group of U is 8 rows x G/2 bytes, exactly a
        // block of R4, and the activation fragments are the residual's: codes from the resident tile [g][token][G/2], scales
        // (with 2^-8 for the two 16*code operands) from sSx.  j tiles go in batches of at most four (registers).
        auto stage1q = [&](auto nq_c) {
            constexpr int NQ = decltype(nq_c)::value;
            constexpr int QB = NQ < 4 ? NQ : 4;
            float d[NQ][MT][4];
#pragma unroll
            for (int q = 0; q < NQ; ++q)
#pragma unroll
                for (int t = 0; t < MT; ++t)
#pragma unroll
                    for (int e = 0; e < 4; ++e) d[q][t][e] = 0.0f;
            const uint32_t ulane = smem_u32(dsm + p.off_l1) + gid * (G / 2) + tid4 * (kW * 4);
            const uint32_t sulane = smem_u32(dsm + p.off_l1) + r * (G / 2) + tid4 * 4;
            uint32_t uoff[NQ], soff[NQ];
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                const uint32_t jt = static_cast<uint32_t>(min(lw + q * lrw, max(njt - 1, 0)));
                uoff[q] = jt * kBlk;
                soff[q] = jt * 16u;
            }
            uint32_t xa = smem_u32(dsm + p.off_xq) + gid * (G / 2) + tid4 * (kW * 4) + u0 * (kMp * (G / 2));
            uint32_t sxp = smem_u32(sSx) + gid * 4 + u0 * (kMp * 4);
            constexpr uint32_t x8 = 8u * (G / 2);
            const uint32_t chunk_bytes = static_cast<uint32_t>(p.sc) * slab_bytes;
            int slot = 0, lap = 0;
            uint32_t slot_a = 0;
            TWQ_DCLK(0);
#pragma unroll 1
            for (int i = 0; i < nl1; ++i) {
                mbar_wait_a(DBAR(D_L1FULL + slot), lap & 1);
                if (i == 0) TWQ_DCLK(1);
                const int cnt = min(p.sc, nu - i * p.sc);
                uint32_t la = slot_a;
#pragma unroll 1
                for (int sl = 0; sl < cnt; ++sl, la += slab_bytes, xa += kMp * (G / 2), sxp += kMp * 4) {
#pragma unroll
                    for (int qb = 0; qb < NQ; qb += QB) {
                        uint32_t wt[QB][kW], suh[QB];
#pragma unroll
                        for (int b = 0; b < QB; ++b) {
                            lds_words<kW>(wt[b], ulane + la + uoff[qb + b]);
                            suh[b] = lds_u32(sulane + la + soff[qb + b]);
                        }
#pragma unroll
                        for (int mt = 0; mt < MT; ++mt) {
                            uint32_t x0[kW], x1[kW];
                            lds_words<kW>(x0, xa + mt * 2 * x8);
                            lds_words<kW>(x1, xa + mt * 2 * x8 + x8);
                            const float sx0 = __uint_as_float(lds_u32(sxp + mt * 64));
                            const float sx1 = __uint_as_float(lds_u32(sxp + mt * 64 + 32));
                            int dd[QB][4];
#pragma unroll
                            for (int b = 0; b < QB; ++b)
#pragma unroll
                                for (int e = 0; e < 4; ++e) dd[b][e] = 0;
#pragma unroll
                            for (int w = 0; w < kW; ++w) {
                                const uint32_t a0 = d_lo16(x0[w]), a1 = d_lo16(x1[w]), a2 = d_hi16(x0[w]), a3 = d_hi16(x1[w]);
#pragma unroll
                                for (int b = 0; b < QB; ++b) imma_16832(dd[b], a0, a1, a2, a3, d_lo16(wt[b][w]), d_hi16(wt[b][w]));
                            }
#pragma unroll
                            for (int b = 0; b < QB; ++b) {
                                const float2 su2 = __half22float2(*reinterpret_cast<const __half2*>(&suh[b]));
                                float (&a)[4] = d[qb + b][mt];
                                a[0] = fmaf(static_cast<float>(dd[b][0]) * su2.x, sx0, a[0]);
                                a[1] = fmaf(static_cast<float>(dd[b][1]) * su2.y, sx0, a[1]);
                                a[2] = fmaf(static_cast<float>(dd[b][2]) * su2.x, sx1, a[2]);
                                a[3] = fmaf(static_cast<float>(dd[b][3]) * su2.y, sx1, a[3]);
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive_a(DBAR(D_L1EMPTY + slot));
                slot_a += chunk_bytes;
                if (++slot == p.l1_slots) { slot = 0; slot_a = 0; ++lap; }
            }
            TWQ_DCLK(2);
            TWQ_DSTAMP(4);
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                const int jt = lw + q * lrw;
                if (jt < njt) {
                    const int j = jt * 8 + tid4 * 2;
#pragma unroll
                    for (int t = 0; t < MT; ++t) {
                        *reinterpret_cast<float2*>(sHpart + (t * 16 + gid) * r + j) = make_float2(d[q][t][0], d[q][t][1]);
                        *reinterpret_cast<float2*>(sHpart + (t * 16 + gid + 8) * r + j) = make_float2(d[q][t][2], d[q][t][3]);
                    }
                }
            }
        };
        if constexpr (kL4) {
            if (nq_need <= 1) stage1q(std::integral_constant<int, 1>{});
            else if (nq_need == 2) stage1q(std::integral_constant<int, 2>{});
            else if (nq_need <= 4 || MT == 4) stage1q(std::integral_constant<int, 4>{});
            else stage1q(std::integral_constant<int, MT == 4 ? 4 : kJT>{});
        } else {
            if (nq_need <= 1) stage1(std::integral_constant<int, 1>{});
            else if (nq_need == 2) stage1(std::integral_constant<int, 2>{});
            else if (nq_need <= 4 || MT == 4) stage1(std::integral_constant<int, 4>{});   // MT == 4 runs 8 low-rank warps: r / 64 <= 4
            else stage1(std::integral_constant<int, MT == 4 ? 4 : kJT>{});
        }
        // stage-2 operand of this warp's first tile (L2T rows, L2-resident by now), ahead of the exchange
        constexpr int kL2 = 8;                                   // 32-wide j steps (r <= 256)
        uint4 l2v[kL2];
        auto load_l2 = [&](int t) {
            const uint8_t* lrow = static_cast<const uint8_t*>(p.L2T) +
                                  (static_cast<size_t>((tile0 + t) * 8 + gid) * r + tid4 * 8) * 2;
#pragma unroll
            for (int js = 0; js < kL2; ++js)
                l2v[js] = (js * 32 + tid4 * 8 < r) ? ldg_nc(lrow + js * 64) : make_uint4(0, 0, 0, 0);
        };
        // q4lr: this thread's words of the V rows of a tile (row gid, grs/8 bytes from tid4 * grs/8) and the tile's scales
        const int kWr = p.grs >> 5, vrow = p.grs >> 1;
        uint32_t vv[2][4], svh[2];
        auto load_v = [&](int t) {
            const uint8_t* vb = static_cast<const uint8_t*>(p.L2T) + static_cast<size_t>(tile0 + t) * p.nh * 8 * vrow + gid * vrow + tid4 * (kWr * 4);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
#pragma unroll
                for (int w = 0; w < 4; ++w)
                    vv[h][w] = (h < p.nh && w < kWr) ? __ldg(reinterpret_cast<const uint32_t*>(vb + h * 8 * vrow) + w) : 0u;
                svh[h] = h < p.nh ? __ldg(reinterpret_cast<const uint32_t*>(p.sv16 + (static_cast<size_t>(tile0 + t) * p.nh + h) * 8) + tid4) : 0u;
            }
        };
        if (lw < ntile) {
            if constexpr (kL4) load_v(lw);
            else load_l2(lw);
        }
        named_bar_sync(1, nlr);                                  // this CTA's partial is complete in shared memory
        TWQ_DSTAMP(5);
        // ---- H = sum of the cluster's partials (fixed order), FP16, in every CTA's shared memory
        if (cs > 1) {
            cluster_wait();                                      // every peer's mbarriers are initialised
            TWQ_DSTAMP(6);
            if (lw == 0 && lane < cs) mbar_arrive_remote(mapa_u32(DBAR(D_X1), static_cast<uint32_t>(lane)));
            mbar_wait_cluster_a(DBAR(D_X1), 0);                  // every CTA's FP32 partial is visible
            TWQ_DSTAMP(7);
            // A thread owns one (token, column) element of this CTA's r/cs columns: the cs remote loads of its partials
            // go out together (a warp's 32 lanes read 32 consecutive floats of ONE peer per instruction -- one remote
            // transaction; one lane per peer was 16x the transactions and 6 us), are summed in rank order, and the FP16
            // result is stored into every peer.
            const int jc = r / cs;
            TWQ_DCLK(10);
            for (int e = lrt; e < p.M * jc; e += nlr) {
                const int m = e / jc, j = rank * jc + (e - m * jc);
                const uint32_t src = smem_u32(sHpart + m * r + j);
                float v[16];
#pragma unroll
                for (int q = 0; q < 16; ++q) v[q] = q < cs ? ld_dsmem_f(mapa_u32(src, q)) : 0.0f;
                float sum = 0.0f;
#pragma unroll
                for (int q = 0; q < 16; ++q) sum += v[q];
                if constexpr (kL4) {
                    const uint32_t dsta = smem_u32(sH32 + m * r + j);
                    for (int pr = 0; pr < cs; ++pr) st_dsmem_u32(mapa_u32(dsta, pr), __float_as_uint(sum));
                } else {
                    sum = fminf(fmaxf(sum, -65504.0f), 65504.0f);
                    const __half hv = __float2half_rn(sum);
                    const uint32_t dsta = smem_u32(sH + m * hstride + j);
                    for (int pr = 0; pr < cs; ++pr) st_dsmem_u16(mapa_u32(dsta, pr), *reinterpret_cast<const uint16_t*>(&hv));
                }
            }
            TWQ_DCLK(11);
            TWQ_DSTAMP(8);
            named_bar_sync(1, nlr);
            if (lw == 0 && lane < cs) mbar_arrive_remote(mapa_u32(DBAR(D_X2), static_cast<uint32_t>(lane)));
            mbar_wait_cluster_a(DBAR(D_X2), 0);                  // every CTA's columns of H have arrived (and nobody reads
                                                                 // this CTA's partial any more)
        } else {
            for (int i = lrt; i < p.M * r; i += nlr) {
                const int m = i / r, j = i - m * r;
                if constexpr (kL4) {
                    sH32[i] = sHpart[i];
                } else {
                    const float s = fminf(fmaxf(sHpart[i], -65504.0f), 65504.0f);
                    sH[m * hstride + j] = __float2half_rn(s);
                }
            }
            named_bar_sync(1, nlr);
        }
        if constexpr (kL4) {
            // ---- re-quantization of H on the fly (Eq. 1 L43-47 on the FP32 H, R18 / R19).  Every CTA
            // does this for all of H (a few K elements).  An item = one (token, r-group): lpi lanes, gr / lpi consecutive elements
            // each.  The chain max -> shuffles -> two divisions -> round is ~100 dependent instructions, so for the common group
            // sizes (gr = 128 / 64: four elements per lane) a warp works on kIB items at once (one item at a time took 650 ns per
            // pass on the critical path; in-kernel timeline, r02).
            const int lpi = p.gr == 128 ? 32 : (p.gr == 64 ? 16 : 8), ipw = 32 / lpi;
            const int e = p.gr / lpi, items = p.M * p.nh;
            const int li = lane & (lpi - 1), sub = lane / lpi;
            const bool dbg_out = kDbg && blockIdx.x == 0;
            if (e == 4) {
                constexpr int kIB = 4;
                for (int base = lw * ipw * kIB; base < items; base += lrw * ipw * kIB) {
                    float4 v[kIB];
                    float amax[kIB];
                    int mm[kIB], hh[kIB];
                    bool on[kIB];
#pragma unroll
                    for (int b = 0; b < kIB; ++b) {
                        const int it = base + b * ipw + sub;
                        on[b] = it < items;
                        mm[b] = on[b] ? (p.nh == 2 ? it >> 1 : it) : 0;
                        hh[b] = on[b] && p.nh == 2 ? (it & 1) : 0;
                        v[b] = on[b] ? *reinterpret_cast<const float4*>(sH32 + mm[b] * r + hh[b] * p.gr + li * 4)
                                     : make_float4(0.f, 0.f, 0.f, 0.f);
                        amax[b] = fmaxf(fmaxf(fabsf(v[b].x), fabsf(v[b].y)), fmaxf(fabsf(v[b].z), fabsf(v[b].w)));
                    }
                    for (int d = lpi >> 1; d >= 1; d >>= 1)
#pragma unroll
                        for (int b = 0; b < kIB; ++b) amax[b] = fmaxf(amax[b], __shfl_xor_sync(0xffffffffu, amax[b], d));
#pragma unroll
                    for (int b = 0; b < kIB; ++b) {
                        const float sc = __fdiv_rn(fmaxf(amax[b], 0x1p-30f), 7.0f);
                        const float inv = __fdiv_rn(1.0f, sc);
                        int q[4] = {__float2int_rn(__fmul_rn(v[b].x, inv)), __float2int_rn(__fmul_rn(v[b].y, inv)),
                                    __float2int_rn(__fmul_rn(v[b].z, inv)), __float2int_rn(__fmul_rn(v[b].w, inv))};
                        uint32_t pk = 0u;
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            q[i] = max(-7, min(7, q[i]));
                            pk |= (static_cast<uint32_t>(q[i]) & 0xFu) << (4 * i);               // low nibble = even index
                        }
                        if (on[b]) {
                            *reinterpret_cast<uint16_t*>(sQH + (hh[b] * kMp + mm[b]) * vrow + li * 2) = static_cast<uint16_t>(pk);
                            if (li == 0) sSH[hh[b] * kMp + mm[b]] = sc * 0x1p-8f;                 // both MMA operands are 16*code
                            if (dbg_out) {
                                const size_t o = static_cast<size_t>(mm[b]) * r + hh[b] * p.gr + li * 4;
                                const float hv[4] = {v[b].x, v[b].y, v[b].z, v[b].w};
                                for (int i = 0; i < 4; ++i) {
                                    if (p.dbgQH != nullptr) p.dbgQH[o + i] = static_cast<int8_t>(q[i]);
                                    if (p.dbgH != nullptr) p.dbgH[o + i] = hv[i];
                                }
                                if (li == 0 && p.dbgSH != nullptr) p.dbgSH[static_cast<size_t>(mm[b]) * p.nh + hh[b]] = sc;
                            }
                        }
                    }
                }
            } else {
                for (int base = lw * ipw; base < items; base += lrw * ipw) {
                    const int it = base + sub;
                    const bool on = it < items;
                    const int m = on ? it / p.nh : 0, h = on ? it - m * p.nh : 0;
                    const float* hp = sH32 + m * r + h * p.gr + li * e;
                    float amax = 0.0f;
                    if (on)
                        for (int i = 0; i < e; ++i) amax = fmaxf(amax, fabsf(hp[i]));
                    for (int d = lpi >> 1; d >= 1; d >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, d));
                    const float sc = __fdiv_rn(fmaxf(amax, 0x1p-30f), 7.0f);
                    const float inv = __fdiv_rn(1.0f, sc);
                    if (on) {
                        uint8_t* qp = sQH + (h * kMp + m) * vrow + li * (e >> 1);
                        for (int i = 0; i < e; i += 2) {
                            int q0 = __float2int_rn(__fmul_rn(hp[i], inv)), q1 = __float2int_rn(__fmul_rn(hp[i + 1], inv));
                            q0 = max(-7, min(7, q0));
                            q1 = max(-7, min(7, q1));
                            qp[i >> 1] = static_cast<uint8_t>((q0 & 0xF) | ((q1 & 0xF) << 4));   // low nibble = even index
                            if (dbg_out) {
                                const size_t o = static_cast<size_t>(m) * r + h * p.gr + li * e + i;
                                if (p.dbgQH != nullptr) { p.dbgQH[o] = static_cast<int8_t>(q0); p.dbgQH[o + 1] = static_cast<int8_t>(q1); }
                                if (p.dbgH != nullptr) { p.dbgH[o] = hp[i]; p.dbgH[o + 1] = hp[i + 1]; }
                            }
                        }
                        if (li == 0) {
                            sSH[h * kMp + m] = sc * 0x1p-8f;             // both MMA operands are 16*code
                            if (dbg_out && p.dbgSH != nullptr) p.dbgSH[static_cast<size_t>(m) * p.nh + h] = sc;
                        }
                    }
                }
            }
            named_bar_sync(1, nlr);
        }
        TWQ_DSTAMP(9);
        // ---- stage 2: Ylr[m, n] = sum_j H[m,j] * L2T[n,j] for this CTA's tiles
        for (int t = lw; t < ntile; t += lrw) {
            if (t != lw) {
                if constexpr (kL4) load_v(t);
                else load_l2(t);
            }
            float d2[MT][4];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int e = 0; e < 4; ++e) d2[mt][e] = 0.0f;
            if constexpr (kL4) {
                // ---- q4lr stage 2: Ylr = sum_h s_H * sv * (Q_H . qv), int8 MMAs on 16*code (K order: word w of a thread's
                // grs/8 bytes in K-step w, for Q_H and V alike)
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    if (h < p.nh) {                              // warp-uniform
                        const float2 sv2 = __half22float2(*reinterpret_cast<const __half2*>(&svh[h]));
#pragma unroll
                        for (int mt = 0; mt < MT; ++mt) {
                            const uint32_t arow = smem_u32(sQH) + ((h * kMp + mt * 16 + gid) * vrow) + tid4 * (kWr * 4);
                            uint32_t x0[4] = {0u, 0u, 0u, 0u}, x1[4] = {0u, 0u, 0u, 0u};
                            if (kWr == 4) {
                                lds_words<4>(x0, arow);
                                lds_words<4>(x1, arow + 8 * vrow);
                            } else {
#pragma unroll
                                for (int w = 0; w < 3; ++w)
                                    if (w < kWr) { x0[w] = lds_u32(arow + w * 4); x1[w] = lds_u32(arow + 8 * vrow + w * 4); }
                            }
                            int dd[4] = {0, 0, 0, 0};
#pragma unroll
                            for (int w = 0; w < 4; ++w)
                                if (w < kWr)
                                    imma_16832(dd, d_lo16(x0[w]), d_lo16(x1[w]), d_hi16(x0[w]), d_hi16(x1[w]), d_lo16(vv[h][w]), d_hi16(vv[h][w]));
                            const float s0 = sSH[h * kMp + mt * 16 + gid], s1 = sSH[h * kMp + mt * 16 + gid + 8];
                            d2[mt][0] = fmaf(static_cast<float>(dd[0]) * sv2.x, s0, d2[mt][0]);
                            d2[mt][1] = fmaf(static_cast<float>(dd[1]) * sv2.y, s0, d2[mt][1]);
                            d2[mt][2] = fmaf(static_cast<float>(dd[2]) * sv2.x, s1, d2[mt][2]);
                            d2[mt][3] = fmaf(static_cast<float>(dd[3]) * sv2.y, s1, d2[mt][3]);
                        }
                    }
                }
            } else {
#pragma unroll
            for (int js = 0; js < kL2; ++js) {
                if (js * 32 < r) {                               // warp-uniform
                    const bool live = js * 32 + tid4 * 8 < r;    // r is a multiple of 16: the last step may be half empty
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        uint4 a = make_uint4(0, 0, 0, 0), b = a;
                        if (live) {
                            a = *reinterpret_cast<const uint4*>(sH + (mt * 16 + gid) * hstride + js * 32 + tid4 * 8);
                            b = *reinterpret_cast<const uint4*>(sH + (mt * 16 + gid + 8) * hstride + js * 32 + tid4 * 8);
                        }
                        hmma_16816(d2[mt], a.x, b.x, a.y, b.y, l2v[js].x, l2v[js].y);
                        hmma_16816(d2[mt], a.z, b.z, a.w, b.w, l2v[js].z, l2v[js].w);
                    }
                }
            }
            }
            const int nl = t * 8 + tid4 * 2;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
                *reinterpret_cast<float2*>(sYlr + (mt * 16 + gid) * nloc + nl) = make_float2(d2[mt][0], d2[mt][1]);
                *reinterpret_cast<float2*>(sYlr + (mt * 16 + gid + 8) * nloc + nl) = make_float2(d2[mt][2], d2[mt][3]);
            }
        }
        TWQ_DSTAMP(10);
    } else {
        // ================================================================ residual warps
        const int rw = warp;
        const int tg = rw / P, part = rw - tg * P;
        const int t_lo = tg * tpg;                               // this warp's tiles: [t_lo, t_lo + ntw)
        const int ntw = tg < TG ? min(tpg, ntile - t_lo) : 0;
        pdl_wait();                                              // sx (or X) comes from the previous kernel of the stream
        TWQ_DSTAMP(2);
        if constexpr (kQ) {
            decode_quantize_share<G, MT, kL4>(p, dsm, xq_local ? 0 : rank, xq_local ? 1 : cs, rw, lane, nrw, lrw, xq_bulk);
        } else {
            for (int i = rw * 32 + lane; i < kMp * ng; i += nrw * 32) {
                const int g = i / kMp, m = i - g * kMp;
                sSx[i] = m < p.M ? ldg_f32(p.sx + static_cast<size_t>(m) * ng + g) * 0x1p-8f : 0.0f;   // MMA operands are 16*code
            }
            named_bar_sync(2, nrw * 32);
        }
        TWQ_DSTAMP(3);
        if (ntile > 0) {
            // The loop is issue-bound (ncu r02a: 38 K warp instructions per CTA, most of them address arithmetic), so
            // everything that does not change per K-group is hoisted: per-tile offsets are registers, the four running
            // addresses advance by constants.
            const uint32_t ring = smem_u32(dsm + p.off_ring);
            const uint32_t tstride = static_cast<uint32_t>(p.gc) * kBlk;          // bytes between tiles inside a slot
            const uint32_t lane_w = ring + t_lo * tstride + gid * (G / 2) + tid4 * (kW * 4);
            // activation codes: the Xq box of the ring slot ([token][gc][G/2]), or the resident tile the in-kernel quantizer fills ([g][token][G/2])
            const uint32_t lane_x = kQ ? smem_u32(dsm + p.off_xq) + gid * (G / 2) + tid4 * (kW * 4)
                                       : ring + p.xq_off + (gid * p.gc) * (G / 2) + tid4 * (kW * 4);
            const uint32_t x8 = kQ ? 8u * (G / 2) : 8u * p.gc * (G / 2);          // token gid -> gid + 8
            const uint32_t sw_a = smem_u32(dsm + p.off_sw) + tid4 * 4 + static_cast<uint32_t>(t_lo) * ng * 16;
            const uint32_t sx_a = smem_u32(sSx) + gid * 4;
            // The warp's tiles are worked in batches of kTB interleaved MMA chains; with more than kTB tiles they are split
            // evenly over two batches (4 -> 2 + 2, 5 -> 3 + 2): accumulator slot i holds tile tix(i); empty slots are skipped.
            const int nb0 = ntw > kTB ? (ntw + 1) / 2 : ntw;                      // tiles of the first batch
            auto tix = [&](int i) { return i < kTB ? i : nb0 + (i - kTB); };      // accumulator slot -> tile of the warp
            auto slot_on = [&](int i) { return i < kTB ? i < nb0 : nb0 + (i - kTB) < ntw; };
            uint32_t toff[kTPW], swoff[kTPW];
#pragma unroll
            for (int i = 0; i < kTPW; ++i) {
                const int ii = slot_on(i) ? tix(i) : 0;
                toff[i] = ii * tstride;
                swoff[i] = static_cast<uint32_t>(ii) * ng * 16;
            }
            const uint32_t step_w = P * kBlk, step_x = kQ ? P * kMp * (G / 2) : P * (G / 2), step_sx = P * kMp * 4, step_sw = P * 16;
            float acc[kTPW][MT][4];
#pragma unroll
            for (int i = 0; i < kTPW; ++i)
#pragma unroll
                for (int t = 0; t < MT; ++t)
#pragma unroll
                    for (int e = 0; e < 4; ++e) acc[i][t][e] = 0.0f;
            int slot = 0, lap = 0;
            uint32_t slot_a = 0;                      // slot * slot_bytes
            int gl = part;                            // next K-group of this warp, relative to the current chunk
            int g = part;                             // the same, absolute
#pragma unroll 1
            for (int c = 0; c < p.nchunks; ++c) {
                mbar_wait_a(DBAR(D_FULL + slot), lap & 1);
                if (c < 6) TWQ_DSTAMP(4 + 2 * c);
                const int gcnt = min(p.gc, ng - c * p.gc);
                if (ntw > 0) {
                    uint32_t wa = lane_w + slot_a + gl * kBlk;
                    uint32_t xa = kQ ? lane_x + g * (kMp * (G / 2)) : lane_x + slot_a + gl * (G / 2);
                    uint32_t sxp = sx_a + g * (kMp * 4);
                    uint32_t swp = sw_a + g * 16;
#pragma unroll 1
                    for (; gl < gcnt; gl += P, g += P, wa += step_w, xa += step_x, sxp += step_sx, swp += step_sw) {
                        if constexpr (MT >= 2) {
                            // Several 16-token tiles: the warp's tiles (kTPW <= kTB) are one batch whose weight fragments are
                            // loaded once per K-group; the token tiles are walked inside, each expanding its own activation
                            // fragments (16 registers at a time instead of 16 * MT).
                            uint32_t wt[kTPW][kW];
                            uint32_t swh[kTPW];
#pragma unroll
                            for (int b = 0; b < kTPW; ++b) {
                                if (b == 0 || slot_on(b)) {
                                    lds_words<kW>(wt[b], wa + toff[b]);
                                    swh[b] = lds_u32(swp + swoff[b]);
                                }
                            }
#pragma unroll
                            for (int mt = 0; mt < MT; ++mt) {
                                uint32_t x0[kW], x1[kW];
                                lds_words<kW>(x0, xa + mt * 2 * x8);
                                lds_words<kW>(x1, xa + mt * 2 * x8 + x8);
                                const float sx0 = __uint_as_float(lds_u32(sxp + mt * 64));
                                const float sx1 = __uint_as_float(lds_u32(sxp + mt * 64 + 32));
                                int dd[kTPW][4];
#pragma unroll
                                for (int b = 0; b < kTPW; ++b)
#pragma unroll
                                    for (int e = 0; e < 4; ++e) dd[b][e] = 0;
#pragma unroll
                                for (int w = 0; w < kW; ++w) {
                                    const uint32_t a0 = d_lo16(x0[w]), a1 = d_lo16(x1[w]), a2 = d_hi16(x0[w]), a3 = d_hi16(x1[w]);
#pragma unroll
                                    for (int b = 0; b < kTPW; ++b)
                                        if (b == 0 || slot_on(b)) imma_16832(dd[b], a0, a1, a2, a3, d_lo16(wt[b][w]), d_hi16(wt[b][w]));
                                }
#pragma unroll
                                for (int b = 0; b < kTPW; ++b) {
                                    if (slot_on(b)) {
                                        const float2 sw2 = __half22float2(*reinterpret_cast<const __half2*>(&swh[b]));
                                        const uint64_t swp2 = pack_f2(sw2.x, sw2.y);
                                        float (&a)[4] = acc[b][mt];
                                        const uint64_t t01 = fma2(pack_f2(static_cast<float>(dd[b][0]), static_cast<float>(dd[b][1])), swp2, 0ull);
                                        const uint64_t t23 = fma2(pack_f2(static_cast<float>(dd[b][2]), static_cast<float>(dd[b][3])), swp2, 0ull);
                                        const uint64_t a01 = fma2(t01, pack_f2(sx0, sx0), pack_f2(a[0], a[1]));
                                        const uint64_t a23 = fma2(t23, pack_f2(sx1, sx1), pack_f2(a[2], a[3]));
                                        unpack_f2(a01, a[0], a[1]);
                                        unpack_f2(a23, a[2], a[3]);
                                        if (kDbg) {
                                            if (p.dbgP != nullptr) {
                                                const int n = (tile0 + t_lo + tix(b)) * 8 + tid4 * 2;
                                                const int m0 = mt * 16 + gid;
                                                if (m0 < p.M) {
                                                    p.dbgP[(static_cast<size_t>(m0) * ng + g) * p.N + n] = dd[b][0] >> 8;
                                                    p.dbgP[(static_cast<size_t>(m0) * ng + g) * p.N + n + 1] = dd[b][1] >> 8;
                                                }
                                                if (m0 + 8 < p.M) {
                                                    p.dbgP[(static_cast<size_t>(m0 + 8) * ng + g) * p.N + n] = dd[b][2] >> 8;
                                                    p.dbgP[(static_cast<size_t>(m0 + 8) * ng + g) * p.N + n + 1] = dd[b][3] >> 8;
                                                }
                                            }
                                        }
                                    }
                                }
                            }
                        } else {
                        // activation fragments of the K-group, expanded once for all tiles of the warp
                        uint32_t ax[MT][kW][4];
                        float sxa[MT][2];
#pragma unroll
                        for (int mt = 0; mt < MT; ++mt) {
                            uint32_t x0[kW], x1[kW];
                            lds_words<kW>(x0, xa + mt * 2 * x8);
                            lds_words<kW>(x1, xa + mt * 2 * x8 + x8);
                            sxa[mt][0] = __uint_as_float(lds_u32(sxp + mt * 64));
                            sxa[mt][1] = __uint_as_float(lds_u32(sxp + mt * 64 + 32));
#pragma unroll
                            for (int w = 0; w < kW; ++w) {
                                ax[mt][w][0] = d_lo16(x0[w]); ax[mt][w][1] = d_lo16(x1[w]);
                                ax[mt][w][2] = d_hi16(x0[w]); ax[mt][w][3] = d_hi16(x1[w]);
                            }
                        }
#pragma unroll
                        for (int ib = 0; ib < kTPW; ib += kTB) {
                            if (slot_on(ib)) {                   // warp-uniform
                                // up to kTB tiles at a time: loads first, then their MMA chains interleaved
                                uint32_t wt[kTB][kW];
                                uint32_t swh[kTB];
                                int dd[kTB][MT][4];
#pragma unroll
                                for (int b = 0; b < kTB; ++b) {
                                    if (b == 0 || slot_on(ib + b)) {
                                        lds_words<kW>(wt[b], wa + toff[ib + b]);
                                        swh[b] = lds_u32(swp + swoff[ib + b]);
                                    }
                                }
#pragma unroll
                                for (int w = 0; w < kW; ++w) {   // one K-step of 32 codes per packed word
#pragma unroll
                                    for (int b = 0; b < kTB; ++b) {
                                        if (b == 0 || slot_on(ib + b)) {
                                            const uint32_t b0 = d_lo16(wt[b][w]), b1 = d_hi16(wt[b][w]);
#pragma unroll
                                            for (int mt = 0; mt < MT; ++mt)
                                                if (w == 0) imma_16832_z(dd[b][mt], ax[mt][w][0], ax[mt][w][1], ax[mt][w][2], ax[mt][w][3], b0, b1);
                                                else imma_16832(dd[b][mt], ax[mt][w][0], ax[mt][w][1], ax[mt][w][2], ax[mt][w][3], b0, b1);
                                        }
                                    }
                                }
                                // dd = 256 * P (exact); fold both scales in FP32 (sx already carries 2^-8): two packed
                                // f32x2 operations per token row instead of four scalar ones
#pragma unroll
                                for (int b = 0; b < kTB; ++b) {
                                    if (slot_on(ib + b)) {       // warp-uniform
                                        const float2 sw2 = __half22float2(*reinterpret_cast<const __half2*>(&swh[b]));
                                        const uint64_t swp2 = pack_f2(sw2.x, sw2.y);
#pragma unroll
                                        for (int mt = 0; mt < MT; ++mt) {
                                            float (&a)[4] = acc[ib + b][mt];
                                            const uint64_t t01 = fma2(pack_f2(static_cast<float>(dd[b][mt][0]), static_cast<float>(dd[b][mt][1])), swp2, 0ull);
                                            const uint64_t t23 = fma2(pack_f2(static_cast<float>(dd[b][mt][2]), static_cast<float>(dd[b][mt][3])), swp2, 0ull);
                                            const uint64_t a01 = fma2(t01, pack_f2(sxa[mt][0], sxa[mt][0]), pack_f2(a[0], a[1]));
                                            const uint64_t a23 = fma2(t23, pack_f2(sxa[mt][1], sxa[mt][1]), pack_f2(a[2], a[3]));
                                            unpack_f2(a01, a[0], a[1]);
                                            unpack_f2(a23, a[2], a[3]);
                                            if (kDbg) {
                                                if (p.dbgP != nullptr) {
                                                    const int n = (tile0 + t_lo + tix(ib + b)) * 8 + tid4 * 2;
                                                    const int m0 = mt * 16 + gid;
                                                    if (m0 < p.M) {
                                                        p.dbgP[(static_cast<size_t>(m0) * ng + g) * p.N + n] = dd[b][mt][0] >> 8;
                                                        p.dbgP[(static_cast<size_t>(m0) * ng + g) * p.N + n + 1] = dd[b][mt][1] >> 8;
                                                    }
                                                    if (m0 + 8 < p.M) {
                                                        p.dbgP[(static_cast<size_t>(m0 + 8) * ng + g) * p.N + n] = dd[b][mt][2] >> 8;
                                                        p.dbgP[(static_cast<size_t>(m0 + 8) * ng + g) * p.N + n + 1] = dd[b][mt][3] >> 8;
                                                    }
                                                }
                                            }
                                        }
                                    }
                                }
                            }
                        }
                        }
                    }
                }
                gl -= gcnt;                           // the warp's next group, relative to the next chunk
                __syncwarp();
                if (c < 6) TWQ_DSTAMP(5 + 2 * c);
                if (lane == 0) mbar_arrive_a(DBAR(D_EMPTY + slot));
                slot_a += p.slot_bytes;
                if (++slot == p.nslots) { slot = 0; slot_a = 0; ++lap; }
            }
            // this warp's partial tiles: [tile * P + part][token][8 channels], parked in the ring, which every residual
            // warp has finished reading (all chunks have landed and been consumed)
            TWQ_DSTAMP(25);
            named_bar_sync(2, nrw * 32);
            TWQ_DSTAMP(26);
#pragma unroll
            for (int i = 0; i < kTPW; ++i) {
                if (slot_on(i)) {
                    float* dst = sRes + static_cast<size_t>((t_lo + tix(i)) * P + part) * kMp * 8 + tid4 * 2;
#pragma unroll
                    for (int mt = 0; mt < MT; ++mt) {
                        *reinterpret_cast<float2*>(dst + (mt * 16 + gid) * 8) = make_float2(acc[i][mt][0], acc[i][mt][1]);
                        *reinterpret_cast<float2*>(dst + (mt * 16 + gid + 8) * 8) = make_float2(acc[i][mt][2], acc[i][mt][3]);
                    }
                }
            }
        }
    }

    // ---------------------------------------------------------------- single epilogue: sum the K-parts, add Ylr, one store
    TWQ_DSTAMP(27);
    __syncthreads();
    TWQ_DSTAMP(28);
    if (warp < kDecWarps) {
        // a thread owns four consecutive channels of one token: the P partial tiles are read as 16-byte vectors (all
        // loads independent), summed in part order, Ylr added, one rounding, one store
        const int nq4 = ntile * 2;                               // 4-channel quads of this CTA
        for (int i = threadIdx.x; i < nq4 * p.M; i += kDecWarps * 32) {
            const int m = i / nq4, q4 = i - m * nq4;
            const int t = q4 >> 1, ch = (q4 & 1) * 4;
            const float* src = sRes + (static_cast<size_t>(t * P) * kMp + m) * 8 + ch;
            float4 y = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 4
            for (int pp = 0; pp < P; ++pp) {
                const float4 v = *reinterpret_cast<const float4*>(src + static_cast<size_t>(pp) * kMp * 8);
                y.x += v.x; y.y += v.y; y.z += v.z; y.w += v.w;
            }
            const int nl = q4 * 4;
            if (r > 0) {
                const float4 v = *reinterpret_cast<const float4*>(sYlr + m * nloc + nl);
                y.x += v.x; y.y += v.y; y.z += v.z; y.w += v.w;
            }
            const size_t o = static_cast<size_t>(m) * p.ldy + tile0 * 8 + nl;
            const float yv[4] = {y.x, y.y, y.z, y.w};
            if (p.ydt == 2) {
                if ((p.ldy & 3) == 0) *reinterpret_cast<float4*>(static_cast<float*>(p.Y) + o) = y;
                else
#pragma unroll
                    for (int e = 0; e < 4; ++e) static_cast<float*>(p.Y)[o + e] = yv[e];
            } else {
                uint2 w;
                if (p.ydt == 0) {
                    const __nv_bfloat162 a = __floats2bfloat162_rn(y.x, y.y), c = __floats2bfloat162_rn(y.z, y.w);
                    w = make_uint2(*reinterpret_cast<const uint32_t*>(&a), *reinterpret_cast<const uint32_t*>(&c));
                } else {
                    const __half2 a = __floats2half2_rn(y.x, y.y), c = __floats2half2_rn(y.z, y.w);
                    w = make_uint2(*reinterpret_cast<const uint32_t*>(&a), *reinterpret_cast<const uint32_t*>(&c));
                }
                if ((p.ldy & 3) == 0) *reinterpret_cast<uint2*>(static_cast<uint8_t*>(p.Y) + o * 2) = w;
                else {
                    uint16_t* yp = static_cast<uint16_t*>(p.Y) + o;
                    yp[0] = static_cast<uint16_t>(w.x); yp[1] = static_cast<uint16_t>(w.x >> 16);
                    yp[2] = static_cast<uint16_t>(w.y); yp[3] = static_cast<uint16_t>(w.y >> 16);
                }
            }
        }
    }
    TWQ_DSTAMP(29);
    if (cs > 1 && !is_lr && !(kQ && warp < nrw && !xq_local)) cluster_wait();   // completes this thread's half of the split barrier (long since released)
    if (xq_bulk && !xq_local) {
        // The all-gather's bulk copies read the SENDER's shared memory: no CTA may exit (and hand its shared memory to another
        // block) before every peer has received its share.  Every CTA gets here after its own share arrived in full, so one
        // more cluster barrier is enough; the kernel ends with its slowest CTA either way.
        cluster_arrive_relaxed();
        cluster_wait();
    }
#undef DBAR
}

// ------------------------------------------------------------------------------------------------ host
namespace {

constexpr int kMaxDevices = 64;

template <int G, int MT, bool kDbg, int kMode, bool kWide = false>
cudaError_t decode_launch_inst(const CUtensorMap& tmXq, const DecodeParams& p, cudaStream_t stream) {
    auto kern = decode_dual_linear_kernel<G, MT, kDbg, kMode, kWide>;
    static bool attr_done[kMaxDevices] = {};       // function attributes are per device
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices || !attr_done[dev]) {
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kDecSmemMax);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < kMaxDevices) attr_done[dev] = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(p.grid));
    cfg.blockDim = dim3(dec_threads(kWide));
    cfg.dynamicSmemBytes = static_cast<size_t>(p.smem_bytes);
    cfg.stream = stream;
    cudaLaunchAttribute attrs[2];
    int na = 0;
    if (p.cs > 1) {
        attrs[na].id = cudaLaunchAttributeClusterDimension;
        attrs[na].val.clusterDim.x = static_cast<unsigned>(p.cs);
        attrs[na].val.clusterDim.y = 1;
        attrs[na].val.clusterDim.z = 1;
        ++na;
    }
    attrs[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attrs[na].val.programmaticStreamSerializationAllowed = 1;
    ++na;
    cfg.attrs = attrs;
    cfg.numAttrs = static_cast<unsigned>(na);
    return cudaLaunchKernelEx(&cfg, kern, tmXq, p);
}

// Clusters of `cs` decode CTAs that can be resident at once (one CTA per SM); conservative table without a device.
int decode_cluster_capacity(int cs, int num_sms) {
    if (cs <= 1) return num_sms;
    static int cache[kMaxDevices][17] = {};
    int dev = 0;
    const bool have_dev = cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < kMaxDevices;
    if (!have_dev) { cudaGetLastError(); dev = kMaxDevices - 1; }
    if (cache[dev][cs] > 0) return cache[dev][cs];
    int n = 0;
    if (have_dev) {
        auto kern = decode_dual_linear_kernel<128, 4, false, 0, true>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kDecSmemMax) == cudaSuccess &&
            cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(static_cast<unsigned>(num_sms / cs * cs));
            cfg.blockDim = dim3(dec_threads(true));
            cfg.dynamicSmemBytes = 200 * 1024;
            cudaLaunchAttribute attr;
            attr.id = cudaLaunchAttributeClusterDimension;
            attr.val.clusterDim.x = static_cast<unsigned>(cs);
            attr.val.clusterDim.y = 1;
            attr.val.clusterDim.z = 1;
            cfg.attrs = &attr;
            cfg.numAttrs = 1;
            if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) n = 0;
        }
        cudaGetLastError();
    }
    if (n <= 0) n = cs == 2 ? num_sms / 2 : (cs == 4 ? (num_sms / 4) * 7 / 8 : (cs == 8 ? (num_sms / 8) * 7 / 8 : (num_sms / 16) * 7 / 8));
    if (n > num_sms / cs) n = num_sms / cs;
    if (n < 1) n = 1;
    cache[dev][cs] = n;
    return n;
}

int round_up_i(int x, int a) { return (x + a - 1) / a * a; }

}  // namespace

// Fills the decode plan; false when the shape is outside this kernel's domain (the tcgen05 kernel takes it).
// quant: 0 = codes and scales come from twq_quantize_act, 1 = in-kernel quantizer, 2 = in-kernel quantizer + 4-bit low-rank branch
bool decode_make_plan(int M, int N, int K, int r, int G, int num_sms, int quant, DecodeParams* out) {
    if (M < 1 || M > kDecodeMaxM || (G != 64 && G != 128) || K % G != 0 || N % 16 != 0 || r % 16 != 0 || r > 256) return false;
    const bool lr4 = quant == 2;
    if (lr4 && (r == 0 || (r > 128 && r != 256))) return false;   // groups of H along r: r itself up to 128, else 128
    if ((plan_flags() & kPlanNoDecode) && !lr4) return false;
    DecodeParams p = {};
    p.M = M; p.N = N; p.K = K; p.r = r; p.ng = K / G;
    p.n_tiles = N / 8;
    p.mt = M <= 16 ? 1 : (M <= 32 ? 2 : 4);
    p.mp = 16 * p.mt;
    p.lrw = r > 0 ? (p.mt == 4 ? 8 : 4) : 0;              // more token tiles: stage 1 / stage 2 over eight warps
    const int nrw = dec_warps(dec_is_wide(p.mt, r, quant)) - p.lrw;
    // cluster size: H is shared by the cluster and every cluster streams all of L1 (K*r*2 bytes) from L2, so the
    // largest cluster that still covers 70 % of the SMs wins; otherwise the size covering the most SMs
    p.cs = 1;
    p.quant = quant;
    p.gr = lr4 ? (r <= 128 ? r : 128) : 0;
    p.grs = (p.gr + 31) / 32 * 32;
    p.nh = lr4 ? r / p.gr : 0;
    int cap = num_sms;
    if (r > 0 || quant) {                                     // the in-kernel quantizer shares its work across the cluster too
        int best = 0;
        bool done = false;
        for (int c = 16; c >= 1 && !done; c >>= 1) {
            if (r % c != 0) continue;                         // (r == 0 divides everything)
            const int n = decode_cluster_capacity(c, num_sms);
            if (n * c > best) { best = n * c; p.cs = c; cap = n; }
            if (n * c * 10 >= num_sms * 7) done = true;
        }
        const int forced = static_cast<int>((plan_flags() >> kPlanDecodeCsShift) & 31u);   // tests only
        if (forced >= 1 && forced <= 16 && (forced & (forced - 1)) == 0 && r % forced == 0) {
            p.cs = forced;
            cap = decode_cluster_capacity(forced, num_sms);
        }
    }
    int nclusters = cap;
    const int need = (p.n_tiles + p.cs - 1) / p.cs;           // clusters needed at one tile per CTA
    if (nclusters > need) nclusters = need;
    if (nclusters < 1) nclusters = 1;
    p.grid = nclusters * p.cs;
    p.tmax = (p.n_tiles + p.grid - 1) / p.grid;
    const int kTPWh = p.mt == 1 ? 6 : (p.mt == 2 ? 3 : 2);    // tiles per residual warp (kernel: kTPW)
    if (p.tmax > kTPWh * nrw) return false;
    // ---- shared-memory plan
    const int kBlk = 4 * G;
    p.nu_max = r > 0 ? ((lr4 ? p.ng : (K >> 5)) + p.cs - 1) / p.cs : 0;   // stage-1 units: 32-wide slabs of L1, or K-groups of U
    // X slice rows: a pitch of 64 bytes mod 128, so that the 16-byte fragment reads of two adjacent tokens hit disjoint banks
    p.xs_stride = lr4 ? 0 : p.nu_max * 32 + ((p.nu_max & 1) ? 0 : 32);
    const int slab_bytes = lr4 ? r * (G / 2) + r * 2 : r * 64;
    int o = 0;
    p.off_bar = o; o += round_up_i(D_COUNT * 8, 128);
    p.off_sw = o; o += round_up_i(p.tmax * p.ng * 16, 128);
    p.off_sx = o; o += round_up_i(p.ng * p.mp * 4, 128);
    p.off_xq = o; o += quant ? round_up_i(p.ng * p.mp * (G / 2), 128) : 0;   // resident codes [g][token][G/2] of the in-kernel quantizer
    p.off_ylr = o; o += r > 0 ? round_up_i(p.mp * p.tmax * 8 * 4, 128) : 0;
    p.off_hpart = o; o += r > 0 ? round_up_i(p.mp * r * 4, 128) : 0;
    p.off_h = o; o += r > 0 ? round_up_i(lr4 ? p.mp * r * 4 : p.mp * (r + 8) * 2, 128) : 0;
    p.off_qh = o; o += lr4 ? round_up_i(p.nh * p.mp * (p.grs / 2), 128) : 0;
    p.off_sh = o; o += lr4 ? round_up_i(p.nh * p.mp * 4, 128) : 0;
    p.xrows = M <= 8 ? 8 : p.mp;                              // token rows of the staged X slice
    p.off_xs = o; o += (r > 0 && !lr4) ? round_up_i(p.xrows * p.xs_stride * 2, 128) : 0;
    // stage-1 ring: chunks of ~16 KB of L1 slabs
    p.sc = 1; p.l1_slots = 1;
    if (r > 0) {
        p.sc = (16 * 1024) / slab_bytes;
        if (p.sc < 1) p.sc = 1;
        if (p.sc > p.nu_max) p.sc = p.nu_max > 0 ? p.nu_max : 1;
        const int chunks = (p.nu_max + p.sc - 1) / p.sc;
        const int max_l1 = p.mt == 4 ? 2 : kMaxL1Slots;       // 64 tokens: the X slice and the H partial take the room
        p.l1_slots = chunks < max_l1 ? (chunks > 0 ? chunks : 1) : max_l1;
        p.off_l1 = o; o += p.l1_slots * p.sc * slab_bytes;
    } else {
        p.off_l1 = o;
    }
    o = round_up_i(o, 1024);
    p.off_ring = o;
    // residual ring: chunk = gc K-groups of every tile of the CTA + the same groups of Xq for all (padded) tokens.
    // About four chunks per call where everything fits (consumers start on the first quarter, the tail after the last
    // byte is a quarter of the work), at most ~40 KB per slot otherwise.
    const int per_g = p.tmax * kBlk + (quant ? 0 : p.mp * (G / 2));
    const int budget = kDecSmemMax - 1024 - o;
    p.gc = (p.ng + 3) / 4;
    while (p.gc > 1 && p.gc * per_g > 40 * 1024) p.gc = (p.gc + 1) / 2;
    while (p.gc > 1 && 2 * round_up_i(p.gc * per_g, 128) > budget) p.gc = (p.gc + 1) / 2;
    if (p.gc > 256) p.gc = 256;                               // TMA box limit
    p.slot_bytes = round_up_i(p.gc * per_g, 128);
    p.xq_off = p.tmax * p.gc * kBlk;
    p.nchunks = (p.ng + p.gc - 1) / p.gc;
    p.nslots = budget / p.slot_bytes;
    if (p.nslots > kMaxSlots) p.nslots = kMaxSlots;
    if (p.nslots > p.nchunks) p.nslots = p.nchunks;
    if (p.nslots < (p.nchunks > 1 ? 2 : 1)) return false;
    // The K-part partial sums ([tile * P + part][token][8 channels], at most min(tmax, kTPW) * nrw of them) are parked in
    // the ring once every chunk has been consumed.
    const int res_bytes = (p.tmax < kTPWh ? p.tmax : kTPWh) * nrw * p.mp * 8 * 4;
    p.off_res = p.off_ring;
    const int ring_bytes = p.nslots * p.slot_bytes;
    if (res_bytes > ring_bytes && res_bytes > budget) return false;
    o += ring_bytes > res_bytes ? ring_bytes : res_bytes;
    p.smem_bytes = o + 1024;                                  // alignment slack of the dynamic base
    if (p.smem_bytes > kDecSmemMax) return false;
    *out = p;
    return true;
}

cudaError_t launch_decode(const CUtensorMap& tmXq, const DecodeParams& p, int G, cudaStream_t stream) {
    const bool dbg = p.dbgP != nullptr || p.dbgH != nullptr || p.dbgQH != nullptr || p.dbgSH != nullptr;
    if (dec_is_wide(p.mt, p.r, p.quant)) {              // four token tiles, r > 128: the 20-warp CTA
        if (G == 128) {
            if (p.quant == 1) return dbg ? decode_launch_inst<128, 4, true, 1, true>(tmXq, p, stream) : decode_launch_inst<128, 4, false, 1, true>(tmXq, p, stream);
            return dbg ? decode_launch_inst<128, 4, true, 0, true>(tmXq, p, stream) : decode_launch_inst<128, 4, false, 0, true>(tmXq, p, stream);
        }
        if (p.quant == 1) return dbg ? decode_launch_inst<64, 4, true, 1, true>(tmXq, p, stream) : decode_launch_inst<64, 4, false, 1, true>(tmXq, p, stream);
        return dbg ? decode_launch_inst<64, 4, true, 0, true>(tmXq, p, stream) : decode_launch_inst<64, 4, false, 0, true>(tmXq, p, stream);
    }
#define TWQ_DCASE(g, m)                                                                   \
    if (G == g && p.mt == m) {                                                            \
        if (p.quant == 2) return dbg ? decode_launch_inst<g, m, true, 2>(tmXq, p, stream) : decode_launch_inst<g, m, false, 2>(tmXq, p, stream); \
        if (p.quant == 1) return dbg ? decode_launch_inst<g, m, true, 1>(tmXq, p, stream) : decode_launch_inst<g, m, false, 1>(tmXq, p, stream); \
        return dbg ? decode_launch_inst<g, m, true, 0>(tmXq, p, stream) : decode_launch_inst<g, m, false, 0>(tmXq, p, stream);        \
    }
    TWQ_DCASE(128, 1) TWQ_DCASE(128, 2) TWQ_DCASE(128, 4) TWQ_DCASE(64, 1) TWQ_DCASE(64, 2) TWQ_DCASE(64, 4)
#undef TWQ_DCASE
    return cudaErrorInvalidValue;
}

}  // namespace twq
