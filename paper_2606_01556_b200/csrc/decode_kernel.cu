// decode_kernel.cu -- the fused dual-branch layer for decode-shaped calls (M <= 16 tokens), sm_100a.
//
//   Y[m,n] = sum_g sx[m,g]*sw[n,g]*P[m,g,n]  +  sum_j H[m,j]*L2[j,n],
//   P[m,g,n] = sum_{k in g} qx[m,k]*qw[n,k] (exact int32),   H = X*L1 (FP32 accumulate)
//   PAPER.md Eq. 2 (L49-50), Eq. 3 (L62), L177-181 (section 4.3), L193 (groups of G).
//
// At M <= 16 the layer streams its weights once and is bound by HBM bandwidth and by launch /
// dependency latency, not by tensor throughput.  The tcgen05 pipeline of
// fused_kernel.cuh pays several hundred cycles per TMA -> expand -> MMA -> commit -> TMEM-load
// hand-off, which a call with eight K-groups per CTA cannot amortise.  This kernel therefore keeps
// every operand in registers: each warp issues all its 16-byte weight loads up front (the bytes in
// flight per SM are what reaches HBM bandwidth), expands INT4 -> int8 with one shift/and per word
// (each code c becomes the byte 16*c, sign for free) and feeds warp-level int8 MMAs whose int32
// result is 256*P, folded with both group scales in FP32.
//
// Work split.  The grid is `nclusters` clusters of `cs` CTAs (512 threads = 16 warps).  A CTA owns T
// consecutive 16-channel tiles of N; an item is (tile, K-part): the P = 16/T (power of two) parts of a
// tile take the K-groups round-robin, each warp runs items w, w+16, ... and leaves its FP32 partial
// tile in shared memory, where a final pass sums the parts in fixed order (deterministic).
//
// Low-rank branch.  H = X*L1 needs all of K, so the cluster computes it cooperatively: CTA q
// multiplies the q-th K-slice (FP16 MMA, X converted BF16 -> FP16 in registers), the FP32 partials
// are reduce-scattered and the FP16 result all-gathered through distributed shared memory (fixed
// order), then each CTA multiplies H by its own rows of L2^T.  H never leaves the chip (L177-179).
//
// K order inside an MMA is a free permutation as long as both operands use the same one: a thread
// takes 16 consecutive bytes of a row (32 codes, or 8 halves) and uses word s of them in K-step s,
// for the weights and for the activations alike, so every global load is a 128-bit load.
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdio.h>
#include <stdlib.h>

#include "fused_kernel.h"
#include "sm100_ptx.cuh"

namespace twq {

namespace {

constexpr int kDecThreads = 512;
constexpr int kDecWarps = 16;
constexpr int kMaxItemsPerWarp = 4;     // planner keeps items <= 16 * this

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

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

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
    asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(cluster_addr));
    return v;
}
__device__ __forceinline__ float4 ld_dsmem_f4_nc(uint32_t cluster_addr) {
    float4 v;
    asm volatile("ld.shared::cluster.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(cluster_addr));
    return v;
}
__device__ __forceinline__ void st_dsmem_u16(uint32_t cluster_addr, uint16_t v) {
    asm volatile("st.shared::cluster.u16 [%0], %1;" ::"r"(cluster_addr), "h"(v) : "memory");
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
// Arrive without a per-thread release fence: used after __syncthreads() + one fence.acq_rel.cluster by
// thread 0 (the CTA's writes are ordered before that fence by the block barrier), or where the arrive only
// says "done reading".  The per-thread release form costs every warp a full memory fence (~0.5-0.9 us here).
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void fence_cluster() { asm volatile("fence.acq_rel.cluster;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

}  // namespace

// One residual pipeline slot: the packed weight words of rows gid / gid+8 for one K-group, the packed
// activation words of tokens gid (/ gid+8), and the two weight scales.
template <int G, int MT>
struct Slot {
    static constexpr int kW = G / 32;          // 32-bit words per thread per row per group (4 or 2)
    uint32_t wa[kW], wb[kW];
    uint32_t xq[MT][kW];
    float swa, swb;
};

template <int kW>
__device__ __forceinline__ void load_words(uint32_t (&dst)[kW], const uint8_t* p, bool nc_stream) {
    if constexpr (kW == 4) {
        const uint4 v = nc_stream ? ldg_nc(p) : __ldg(reinterpret_cast<const uint4*>(p));
        dst[0] = v.x; dst[1] = v.y; dst[2] = v.z; dst[3] = v.w;
    } else {
        const uint2 v = __ldg(reinterpret_cast<const uint2*>(p));
        dst[0] = v.x; dst[1] = v.y;
    }
}

#ifdef TWQ_TRACE
__device__ unsigned long long g_twq_dtrace[4 * 32];
#define TWQ_DT(k)                                                                                     \
    do {                                                                                              \
        if ((threadIdx.x & 31) == 0 && (threadIdx.x >> 5) < 2 && (blockIdx.x == 0 || blockIdx.x == 61)) { \
            unsigned long long t_;                                                                    \
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                                    \
            g_twq_dtrace[((blockIdx.x != 0) * 2 + (threadIdx.x >> 5)) * 32 + (k)] = t_;               \
        }                                                                                             \
    } while (0)
#else
#define TWQ_DT(k) do { } while (0)
#endif

template <int G, int MT, bool kDbg>
__global__ void __launch_bounds__(kDecThreads, 1) decode_dual_linear_kernel(const __grid_constant__ DecodeParams p) {
    extern __shared__ __align__(16) uint8_t dsm[];
    float* sRes = reinterpret_cast<float*>(dsm + p.off_res);      // [items][8*MT tokens][16 rows]: the epilogue reads rows contiguously
    float* sHpart = reinterpret_cast<float*>(dsm + p.off_hpart);  // [16 tokens][r]
    __half* sH = reinterpret_cast<__half*>(dsm + p.off_h);        // [16 tokens][r + 8]
    float* sYlr = reinterpret_cast<float*>(dsm + p.off_ylr);      // [16 tokens][T*16]
    float* sSx = reinterpret_cast<float*>(dsm + p.off_sx);        // [8*MT tokens][ng]
    __half* sXs = reinterpret_cast<__half*>(dsm + p.off_xs);      // [8*MT tokens][K slice + 8] FP16 copy of X

    constexpr int kW = G / 32;
    constexpr int kTok = 8 * MT;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int gid = lane >> 2, tid4 = lane & 3;
    const int r = p.r, ng = p.ng, cs = p.cs;
    const int rank = cs > 1 ? static_cast<int>(cluster_ctarank()) : 0;
    // 16-channel tiles of this CTA: an even split of the n_tiles over the grid (at most T each)
    const int tile0 = static_cast<int>(static_cast<long long>(blockIdx.x) * p.n_tiles / gridDim.x);
    const int ntile = static_cast<int>(static_cast<long long>(blockIdx.x + 1) * p.n_tiles / gridDim.x) - tile0;
    // K-parts per tile, chosen per CTA so that its ntile * P items fill the 16 warps in ONE round where
    // possible (a second item per warp would expose another DRAM round trip): P = 16 / ntile, any integer
    int P = ntile > 0 ? kDecWarps / ntile : 1;
    P = max(1, min(P, p.P));
    const int items = ntile * P;
    const int rowbytes = p.K >> 1;
    const int hstride = r + 8;

    pdl_launch_dependents();
    TWQ_DT(0);
#ifdef TWQ_TRACE
    if (p.ydt >= 100) return;     // launch-overhead probe (trace build only)
#endif

    // ---------------------------------------------------------------- residual: first loads in flight
    constexpr int kD = 4;
    Slot<G, MT> sl[kD];
    int item = warp;                       // current item of this warp
    int tile = 0, kpart = 0, cnt = 0;      // its tile, K-part and number of groups
    const uint8_t* wrow = nullptr;         // row gid of the tile in R4
    auto setup_item = [&]() {
        tile = item / P;
        kpart = item - tile * P;
        cnt = kpart < ng ? (ng - kpart + P - 1) / P : 0;
        wrow = p.R4 + static_cast<size_t>((tile0 + tile) * 16 + gid) * rowbytes + tid4 * (kW * 4);
    };
    auto load_w = [&](Slot<G, MT>& s, int i) {   // weights + weight scales of the i-th group of the item
        const int g = kpart + i * P;
        load_words<kW>(s.wa, wrow + static_cast<size_t>(g) * (G / 2), true);
        load_words<kW>(s.wb, wrow + static_cast<size_t>(g) * (G / 2) + static_cast<size_t>(8) * rowbytes, true);
        const float* sp = p.swT + static_cast<size_t>(g) * p.N + (tile0 + tile) * 16 + gid;
        s.swa = __ldg(sp);
        s.swb = __ldg(sp + 8);
    };
    auto load_x = [&](Slot<G, MT>& s, int i) {   // packed activations of tokens gid (, gid+8)
        const int g = kpart + i * P;
#pragma unroll
        for (int t = 0; t < MT; ++t) {
            const int m = gid + 8 * t;
            if (m < p.M) {
                load_words<kW>(s.xq[t], p.Xq + static_cast<size_t>(m) * rowbytes + static_cast<size_t>(g) * (G / 2) + tid4 * (kW * 4), false);
            } else {
#pragma unroll
                for (int w = 0; w < kW; ++w) s.xq[t][w] = 0u;
            }
        }
    };
    // The low-rank chain (L1T slice -> partial H -> cluster exchange -> stage 2) is the critical path of a
    // decode call, so its loads go out first; the residual weight stream is started right after and lands
    // while the cluster exchanges H.

    // ---------------------------------------------------------------- low-rank stage 1: H partial of this CTA's K slice
    if (r > 0) {
        const int units = p.K >> 5;                                  // 32-wide K units
        // K slice of this CTA: 1/cs of K, or (stage 1 over all clusters) 1/grid of K
        const int kslice = p.ncl_k > 1 ? static_cast<int>(blockIdx.x) : rank;
        const int kslices = p.ncl_k > 1 ? static_cast<int>(gridDim.x) : cs;
        const int u0 = static_cast<int>(static_cast<long long>(units) * kslice / kslices);
        const int u1 = static_cast<int>(static_cast<long long>(units) * (kslice + 1) / kslices);
        const int nu = u1 - u0;
        constexpr int kDL = 8;                                       // L1T loads in flight per thread
        // loads in the order the dependent chain needs them: X slice, first j-tile's L1T ring, residual weights
        const int xs_stride = nu * 32 + 8;                           // halves; rows padded by 16 bytes
        const uint16_t* X = static_cast<const uint16_t*>(p.X);
        const int chunks = nu * 4;                                   // 16-byte chunks per token row
        constexpr int kXV = 2;                                       // staged X chunks per thread per pass
        uint4 xv[kXV];
#pragma unroll
        for (int q = 0; q < kXV; ++q) {
            const int i = threadIdx.x + q * kDecThreads;
            const int m = i / chunks, c = i - m * chunks;
            xv[q] = make_uint4(0, 0, 0, 0);
            if (i < kTok * chunks && m < p.M) xv[q] = __ldg(reinterpret_cast<const uint4*>(X + static_cast<size_t>(m) * p.ldx + u0 * 32 + c * 8));
        }
        int jt = warp;
        const uint8_t* lrow = reinterpret_cast<const uint8_t*>(p.L1T) + (static_cast<size_t>(jt * 8 + gid) * p.K + tid4 * 8) * 2;
        uint4 lv[kDL];
        const bool j_ok = jt < (r >> 3);
#pragma unroll
        for (int s = 0; s < kDL; ++s)
            if (j_ok && s < nu) lv[s] = ldg_nc(lrow + static_cast<size_t>(u0 + s) * 64);
        // X slice (tokens x 32*nu k, BF16 -> FP16) into shared memory
#pragma unroll
        for (int q = 0; q < kXV; ++q) {
            const int i = threadIdx.x + q * kDecThreads;
            if (i < kTok * chunks) {
                const int m = i / chunks, c = i - m * chunks;
                uint4 v = xv[q];
                v.x = bf2_to_h2(v.x); v.y = bf2_to_h2(v.y); v.z = bf2_to_h2(v.z); v.w = bf2_to_h2(v.w);
                *reinterpret_cast<uint4*>(sXs + m * xs_stride + c * 8) = v;
            }
        }
        for (int i = threadIdx.x + kXV * kDecThreads; i < kTok * chunks; i += kDecThreads) {   // long K slices
            const int m = i / chunks, c = i - m * chunks;
            uint4 v = make_uint4(0, 0, 0, 0);
            if (m < p.M) v = __ldg(reinterpret_cast<const uint4*>(X + static_cast<size_t>(m) * p.ldx + u0 * 32 + c * 8));
            v.x = bf2_to_h2(v.x); v.y = bf2_to_h2(v.y); v.z = bf2_to_h2(v.z); v.w = bf2_to_h2(v.w);
            *reinterpret_cast<uint4*>(sXs + m * xs_stride + c * 8) = v;
        }
        __syncthreads();
        TWQ_DT(1);
        for (; jt < (r >> 3); jt += kDecWarps) {
            // a warp-level MMA has a latency of several hundred cycles on this part: eight independent
            // accumulators keep the dependent chain at nu/4 instead of 2*nu
            float d8[8][4];
#pragma unroll
            for (int q = 0; q < 8; ++q)
#pragma unroll
                for (int e = 0; e < 4; ++e) d8[q][e] = 0.0f;
            if (jt != warp) {
                lrow = reinterpret_cast<const uint8_t*>(p.L1T) + (static_cast<size_t>(jt * 8 + gid) * p.K + tid4 * 8) * 2;
#pragma unroll
                for (int s = 0; s < kDL; ++s)
                    if (s < nu) lv[s] = ldg_nc(lrow + static_cast<size_t>(u0 + s) * 64);
            }
            const __half* xa = sXs + gid * xs_stride + tid4 * 8;
            const __half* xb = xa + 8 * xs_stride;
            for (int ub = 0; ub < nu; ub += kDL) {
#pragma unroll
                for (int s = 0; s < kDL; ++s) {
                    if (ub + s < nu) {
                        const uint4 a = *reinterpret_cast<const uint4*>(xa + (ub + s) * 32);
                        uint4 b = make_uint4(0, 0, 0, 0);
                        if (MT == 2) b = *reinterpret_cast<const uint4*>(xb + (ub + s) * 32);
                        hmma_16816(d8[(2 * s) & 7], a.x, b.x, a.y, b.y, lv[s].x, lv[s].y);
                        hmma_16816(d8[(2 * s + 1) & 7], a.z, b.z, a.w, b.w, lv[s].z, lv[s].w);
                        if (ub + s + kDL < nu) lv[s] = ldg_nc(lrow + static_cast<size_t>(u0 + ub + s + kDL) * 64);
                    }
                }
            }
            float d[4];
#pragma unroll
            for (int e = 0; e < 4; ++e)
                d[e] = ((d8[0][e] + d8[1][e]) + (d8[2][e] + d8[3][e])) + ((d8[4][e] + d8[5][e]) + (d8[6][e] + d8[7][e]));
            const int j = jt * 8 + tid4 * 2;
            sHpart[gid * r + j] = d[0];
            sHpart[gid * r + j + 1] = d[1];
            sHpart[(gid + 8) * r + j] = d[2];
            sHpart[(gid + 8) * r + j + 1] = d[3];
        }
        TWQ_DT(2);
        if (cs > 1) {                   // release: this CTA's partial is in its shared memory
            __syncthreads();
            if (threadIdx.x == 0) fence_cluster();
            cluster_arrive_relaxed();
        }
        TWQ_DT(3);
    }
    // residual weight stream: issued after the arrive (its release fence would otherwise wait for these loads)
    if (item < items) {
        setup_item();
#pragma unroll
        for (int s = 0; s < kD; ++s)
            if (s < cnt) load_w(sl[s], s);
        // groups beyond the register ring: pull their lines into L2 now, so that the ring's refills are L2 hits
        // instead of a second DRAM round trip (CTAs with an odd tile count have 6-7 groups per item)
        for (int i = kD; i < cnt && i < 3 * kD; ++i) {
            const uint8_t* a = wrow + static_cast<size_t>(kpart + i * P) * (G / 2);
            prefetch_l2(a);
            prefetch_l2(a + static_cast<size_t>(8) * rowbytes);
        }
    }

    // stage-2 operand of this warp's first 8-channel step (L2T rows), prefetched behind the weights
    constexpr int kL2 = 8;                             // 32-wide j steps held in registers (r <= 256)
    uint4 l2v[kL2];
    const bool l2_ok = r > 0 && warp < ntile * 2;
    if (l2_ok) {
        const uint8_t* lrow = reinterpret_cast<const uint8_t*>(p.L2T) +
                              (static_cast<size_t>(tile0 * 16 + warp * 8 + gid) * r + tid4 * 8) * 2;
#pragma unroll
        for (int js = 0; js < kL2; ++js)
            l2v[js] = (js * 32 + tid4 * 8 < r) ? ldg_nc(lrow + js * 64) : make_uint4(0, 0, 0, 0);
    }

    // ---------------------------------------------------------------- quantizer outputs from here on
    TWQ_DT(4);
    pdl_wait();
    TWQ_DT(5);
    for (int i = threadIdx.x; i < kTok * ng; i += kDecThreads) {
        const int m = i / ng, g = i - m * ng;
        sSx[i] = m < p.M ? __ldg(p.sx + static_cast<size_t>(m) * ng + g) * 0x1p-8f : 0.0f;   // MMA operands are 16*code
    }
    if (item < items) {
#pragma unroll
        for (int s = 0; s < kD; ++s)
            if (s < cnt) load_x(sl[s], s);
    }

    __syncthreads();                                   // sSx visible to every warp
    TWQ_DT(9);

    // ---------------------------------------------------------------- residual items of this warp
    while (item < items) {
        float acc[MT][4];
#pragma unroll
        for (int t = 0; t < MT; ++t)
#pragma unroll
            for (int e = 0; e < 4; ++e) acc[t][e] = 0.0f;
        const int n_a = (tile0 + tile) * 16 + gid;   // output channel of rows gid (n_a) and gid+8 (n_a + 8)
        for (int ib = 0; ib < cnt; ib += kD) {
            // the kD groups in flight form independent MMA chains (one int32 tile each); issuing them
            // interleaved hides the warp-level MMA latency
            int d[kD][MT][4];
#pragma unroll
            for (int s = 0; s < kD; ++s)
#pragma unroll
                for (int t = 0; t < MT; ++t)
#pragma unroll
                    for (int e = 0; e < 4; ++e) d[s][t][e] = 0;
#pragma unroll
            for (int w = 0; w < kW; ++w) {              // one K-step of 32 codes per packed word
#pragma unroll
                for (int s = 0; s < kD; ++s) {
                    if (ib + s < cnt) {
                        const Slot<G, MT>& c = sl[s];
                        const uint32_t a0 = d_lo16(c.wa[w]), a2 = d_hi16(c.wa[w]);
                        const uint32_t a1 = d_lo16(c.wb[w]), a3 = d_hi16(c.wb[w]);
#pragma unroll
                        for (int t = 0; t < MT; ++t)
                            imma_16832(d[s][t], a0, a1, a2, a3, d_lo16(c.xq[t][w]), d_hi16(c.xq[t][w]));
                    }
                }
            }
#pragma unroll
            for (int s = 0; s < kD; ++s) {
                const int i = ib + s;
                if (i < cnt) {
                    const int g = kpart + i * P;
                    Slot<G, MT>& c = sl[s];
                    // d = 256 * P (exact); fold both scales in FP32 (sx already carries 2^-8)
#pragma unroll
                    for (int t = 0; t < MT; ++t) {
                        const float s0 = sSx[(8 * t + tid4 * 2) * ng + g], s1 = sSx[(8 * t + tid4 * 2 + 1) * ng + g];
                        acc[t][0] = fmaf(__fmul_rn(static_cast<float>(d[s][t][0]), c.swa), s0, acc[t][0]);
                        acc[t][1] = fmaf(__fmul_rn(static_cast<float>(d[s][t][1]), c.swa), s1, acc[t][1]);
                        acc[t][2] = fmaf(__fmul_rn(static_cast<float>(d[s][t][2]), c.swb), s0, acc[t][2]);
                        acc[t][3] = fmaf(__fmul_rn(static_cast<float>(d[s][t][3]), c.swb), s1, acc[t][3]);
                        if (kDbg) {
                            if (p.dbgP != nullptr) {
                                const int m0 = 8 * t + tid4 * 2;
                                if (m0 < p.M) {
                                    p.dbgP[(static_cast<size_t>(m0) * ng + g) * p.N + n_a] = d[s][t][0] >> 8;
                                    p.dbgP[(static_cast<size_t>(m0) * ng + g) * p.N + n_a + 8] = d[s][t][2] >> 8;
                                }
                                if (m0 + 1 < p.M) {
                                    p.dbgP[(static_cast<size_t>(m0 + 1) * ng + g) * p.N + n_a] = d[s][t][1] >> 8;
                                    p.dbgP[(static_cast<size_t>(m0 + 1) * ng + g) * p.N + n_a + 8] = d[s][t][3] >> 8;
                                }
                            }
                        }
                    }
                    if (i + kD < cnt) { load_w(c, i + kD); load_x(c, i + kD); }
                }
            }
        }
        float* dst = sRes + static_cast<size_t>(item) * 16 * kTok;
#pragma unroll
        for (int t = 0; t < MT; ++t) {
            const int m0 = 8 * t + tid4 * 2;
            dst[m0 * 16 + gid] = acc[t][0];
            dst[(m0 + 1) * 16 + gid] = acc[t][1];
            dst[m0 * 16 + gid + 8] = acc[t][2];
            dst[(m0 + 1) * 16 + gid + 8] = acc[t][3];
        }
        item += kDecWarps;
        if (item < items) {
            setup_item();
#pragma unroll
            for (int s = 0; s < kD; ++s)
                if (s < cnt) { load_w(sl[s], s); load_x(sl[s], s); }
        }
    }

    // ---------------------------------------------------------------- low-rank: H exchange
    if (r > 0) {
        if (cs > 1) {
            cluster_wait();                            // every CTA's FP32 partial is visible
            TWQ_DT(6);
            if (p.ncl_k > 1) {
                // Stage 1 over all clusters.  (a) reduce-scatter inside the cluster as below, but the FP32 sums of
                // this CTA's r/cs columns go to the workspace [cluster][16][r]; (b) grid-wide barrier on the
                // workspace counter; (c) sum over the clusters in fixed order (H is identical everywhere), FP16,
                // all-gather through distributed shared memory.
                const int jc = r / cs;
                const int cl = static_cast<int>(blockIdx.x) / cs;
                for (int i = threadIdx.x; i < p.M * jc; i += kDecThreads) {
                    const int m = i / jc, j = rank * jc + (i - m * jc);
                    const uint32_t src = smem_u32(sHpart + m * r + j);
                    float s = 0.0f;
                    for (int pr = 0; pr < cs; pr += 4) {
                        float v[4];
#pragma unroll
                        for (int q = 0; q < 4; ++q) v[q] = pr + q < cs ? ld_dsmem_f(mapa_u32(src, pr + q)) : 0.0f;
#pragma unroll
                        for (int q = 0; q < 4; ++q) s += v[q];
                    }
                    p.ws_h[(static_cast<size_t>(cl) * 16 + m) * r + j] = s;
                }
                __syncthreads();
                if (threadIdx.x == 0) {
                    __threadfence();
                    atomicAdd(p.ws_ctr, 1u);
                    unsigned seen, spins = 0;
                    do {
                        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(p.ws_ctr) : "memory");
                        if (seen < gridDim.x) {
                            __nanosleep(32);
                            if (++spins > (1u << 24)) __trap();   // a CTA of the grid never arrived: fail loudly, do not hang
                        }
                    } while (seen < gridDim.x);
                    __threadfence();
                }
                __syncthreads();
                for (int i = threadIdx.x; i < p.M * jc; i += kDecThreads) {
                    const int m = i / jc, j = rank * jc + (i - m * jc);
                    float s = 0.0f;
                    const float* src = p.ws_h + static_cast<size_t>(m) * r + j;
                    for (int c0 = 0; c0 < p.ncl_k; c0 += 8) {      // eight loads in flight, summed in cluster order
                        float v[8];
#pragma unroll
                        for (int q = 0; q < 8; ++q)
                            v[q] = c0 + q < p.ncl_k ? __ldcg(src + static_cast<size_t>(c0 + q) * 16 * r) : 0.0f;
#pragma unroll
                        for (int q = 0; q < 8; ++q) s += v[q];
                    }
                    s = fminf(fmaxf(s, -65504.0f), 65504.0f);
                    const __half hv = __float2half_rn(s);
                    const uint32_t dsta = smem_u32(sH + m * hstride + j);
                    for (int pr = 0; pr < cs; ++pr) st_dsmem_u16(mapa_u32(dsta, pr), *reinterpret_cast<const uint16_t*>(&hv));
                }
                __syncthreads();
                if (threadIdx.x == 0) {
                    fence_cluster();                       // release this CTA's remote stores
                    const unsigned prev = atomicAdd(p.ws_ctr, 1u);   // second round: the last CTA leaves the counter at zero
                    if (prev == 2u * gridDim.x - 1u) atomicExch(p.ws_ctr, 0u);
                }
                cluster_arrive_relaxed();
                cluster_wait();                            // every CTA's slice of H has arrived
            } else if (p.M <= 2) {
            // all-reduce by reading: every CTA sums the cs partials of the M live rows itself (fixed order, so
            // H is identical everywhere) -- one cluster barrier instead of a reduce-scatter plus an all-gather.
            // Distributed-shared-memory reads are slow (about 8 KB per microsecond per CTA here), so only for M <= 2.
            const int r4 = r >> 2;
            for (int i = threadIdx.x; i < p.M * r4; i += kDecThreads) {
                const int m = i / r4, j = (i - m * r4) * 4;
                const uint32_t src = smem_u32(sHpart + m * r + j);
                float4 s4 = make_float4(0.f, 0.f, 0.f, 0.f);
                for (int pr = 0; pr < cs; pr += 4) {   // four remote loads in flight
                    float4 v[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        v[q] = pr + q < cs ? ld_dsmem_f4_nc(mapa_u32(src, pr + q)) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                    for (int q = 0; q < 4; ++q) { s4.x += v[q].x; s4.y += v[q].y; s4.z += v[q].z; s4.w += v[q].w; }
                }
                const __half2 h01 = __floats2half2_rn(fminf(fmaxf(s4.x, -65504.0f), 65504.0f), fminf(fmaxf(s4.y, -65504.0f), 65504.0f));
                const __half2 h23 = __floats2half2_rn(fminf(fmaxf(s4.z, -65504.0f), 65504.0f), fminf(fmaxf(s4.w, -65504.0f), 65504.0f));
                uint2 o;
                o.x = *reinterpret_cast<const uint32_t*>(&h01);
                o.y = *reinterpret_cast<const uint32_t*>(&h23);
                *reinterpret_cast<uint2*>(sH + m * hstride + j) = o;
            }
            } else {
                // reduce-scatter (this CTA sums r/cs columns of the M live rows over the cs partials, fixed
                // order) + all-gather (the FP16 result goes to every CTA's sH)
                const int jc = r / cs;
                for (int i = threadIdx.x; i < p.M * jc; i += kDecThreads) {
                    const int m = i / jc, j = rank * jc + (i - m * jc);
                    const uint32_t src = smem_u32(sHpart + m * r + j);
                    float s = 0.0f;
                    for (int pr = 0; pr < cs; pr += 4) {
                        float v[4];
#pragma unroll
                        for (int q = 0; q < 4; ++q) v[q] = pr + q < cs ? ld_dsmem_f(mapa_u32(src, pr + q)) : 0.0f;
#pragma unroll
                        for (int q = 0; q < 4; ++q) s += v[q];
                    }
                    s = fminf(fmaxf(s, -65504.0f), 65504.0f);
                    const __half hv = __float2half_rn(s);
                    const uint32_t dsta = smem_u32(sH + m * hstride + j);
                    for (int pr = 0; pr < cs; ++pr) st_dsmem_u16(mapa_u32(dsta, pr), *reinterpret_cast<const uint16_t*>(&hv));
                }
                __syncthreads();
                if (threadIdx.x == 0) fence_cluster();     // release this CTA's remote stores
                cluster_arrive_relaxed();
                cluster_wait();                            // every CTA's slice of H has arrived
            }
            TWQ_DT(7);
            cluster_arrive_relaxed();                  // this CTA no longer reads its peers (waited for before exit)
            TWQ_DT(8);
            __syncthreads();
        } else {
            __syncthreads();
            for (int i = threadIdx.x; i < 16 * r; i += kDecThreads) {
                const int m = i / r, j = i - m * r;
                const float s = fminf(fmaxf(sHpart[i], -65504.0f), 65504.0f);
                sH[m * hstride + j] = __float2half_rn(s);
            }
            __syncthreads();
        }
    }
    // ---------------------------------------------------------------- low-rank stage 2
    const int nloc = p.T * 16;                         // channels of this CTA (row stride of sYlr)
    if (r > 0) {
        TWQ_DT(10);
        // Ylr[m, n] = sum_j H[m,j] * L2T[n,j] for this CTA's channels, 8 channels per warp step
        for (int nt = warp; nt < ntile * 2; nt += kDecWarps) {
            float d[4] = {0.f, 0.f, 0.f, 0.f};
            if (nt != warp) {
                const uint8_t* lrow = reinterpret_cast<const uint8_t*>(p.L2T) +
                                      (static_cast<size_t>(tile0 * 16 + nt * 8 + gid) * r + tid4 * 8) * 2;
#pragma unroll
                for (int js = 0; js < kL2; ++js)
                    l2v[js] = (js * 32 + tid4 * 8 < r) ? ldg_nc(lrow + js * 64) : make_uint4(0, 0, 0, 0);
            }
            const __half* ha = sH + gid * hstride + tid4 * 8;
            const __half* hb = ha + 8 * hstride;
#pragma unroll
            for (int js = 0; js < kL2; ++js) {
                if (js * 32 < r) {                     // warp-uniform
                    uint4 a = make_uint4(0, 0, 0, 0), b = a;
                    if (js * 32 + tid4 * 8 < r) {      // r is a multiple of 16: the last step may be half empty
                        a = *reinterpret_cast<const uint4*>(ha + js * 32);
                        b = *reinterpret_cast<const uint4*>(hb + js * 32);
                    }
                    hmma_16816(d, a.x, b.x, a.y, b.y, l2v[js].x, l2v[js].y);
                    hmma_16816(d, a.z, b.z, a.w, b.w, l2v[js].z, l2v[js].w);
                }
            }
            const int nl = nt * 8 + tid4 * 2;
            sYlr[gid * nloc + nl] = d[0];
            sYlr[gid * nloc + nl + 1] = d[1];
            sYlr[(gid + 8) * nloc + nl] = d[2];
            sYlr[(gid + 8) * nloc + nl + 1] = d[3];
        }
    }
    __syncthreads();

    TWQ_DT(12);
    // ---------------------------------------------------------------- single epilogue: sum the K-parts, add Ylr, one store
    for (int i = threadIdx.x; i < ntile * 16 * p.M; i += kDecThreads) {
        const int m = i / (ntile * 16), nl = i - m * (ntile * 16);
        const int tl = nl >> 4, row = nl & 15;
        float y = 0.0f;
        for (int pp = 0; pp < P; ++pp) y += sRes[(static_cast<size_t>(tl * P + pp) * kTok + m) * 16 + row];
        if (r > 0) y += sYlr[m * nloc + nl];
        const size_t o = static_cast<size_t>(m) * p.ldy + tile0 * 16 + nl;
        if (p.ydt == 0) static_cast<__nv_bfloat16*>(p.Y)[o] = __float2bfloat16_rn(y);
        else if (p.ydt == 1) static_cast<__half*>(p.Y)[o] = __float2half_rn(y);
        else static_cast<float*>(p.Y)[o] = y;
    }
    TWQ_DT(13);
    if (r > 0 && cs > 1) cluster_wait();               // no CTA exits while a peer may still read its partial
}

// ------------------------------------------------------------------------------------------------ host
namespace {

template <int G, int MT, bool kDbg>
cudaError_t decode_launch_inst(const DecodeParams& p, cudaStream_t stream) {
    auto kern = decode_dual_linear_kernel<G, MT, kDbg>;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 232448 - 64);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(p.grid));
    cfg.blockDim = dim3(kDecThreads);
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
    return cudaLaunchKernelEx(&cfg, kern, p);
}

// Clusters of `cs` decode CTAs that can be resident at once (one CTA per SM); conservative table without a device.
int decode_cluster_capacity(int cs, int num_sms) {
    if (cs <= 1) return num_sms;
    static int cache[17] = {0};
    if (cache[cs] > 0) return cache[cs];
    int n = 0;
    {
        auto kern = decode_dual_linear_kernel<128, 1, false>;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 232448 - 64) == cudaSuccess &&
            cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(static_cast<unsigned>(num_sms / cs * cs));
            cfg.blockDim = dim3(kDecThreads);
            cfg.dynamicSmemBytes = 128 * 1024;
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
    cache[cs] = n;
    return n;
}

}  // namespace

// Fills the decode plan; false when the shape is outside this kernel's domain (the tcgen05 kernel takes it).
bool decode_make_plan(int M, int N, int K, int r, int G, int num_sms, DecodeParams* out) {
    if (M < 1 || M > 16 || (G != 64 && G != 128) || K % G != 0 || N % 16 != 0 || r % 16 != 0 || r > 256) return false;
    DecodeParams p = {};
    p.M = M; p.N = N; p.K = K; p.r = r; p.ng = K / G;
    p.n_tiles = N / 16;
    // cluster size: the one that keeps the most SMs busy; H is shared by the cluster, so larger is cheaper
    p.cs = 1;
    int cap = num_sms;
    if (r > 0) {
        // every cluster streams all of L1 (K*r*2 bytes) from L2, so the largest cluster that still covers
        // 70 % of the SMs wins; otherwise the size covering the most SMs
        int best = 0;
        bool done = false;
        for (int c = 16; c >= 1 && !done; c >>= 1) {
            if (r % c != 0 || (K >> 5) < c) continue;
            const int n = decode_cluster_capacity(c, num_sms);
            if (n * c > best) { best = n * c; p.cs = c; cap = n; }
            if (n * c * 10 >= num_sms * 7) done = true;
        }
    }
    if (const char* e = getenv("TWQ_DEBUG_DECODE_CS")) {   // debugging aid: force the cluster size
        const int c = atoi(e);
        if (r > 0 && c >= 1 && c <= 16 && (c & (c - 1)) == 0 && r % c == 0) { p.cs = c; cap = decode_cluster_capacity(c, num_sms); }
    }
    int nclusters = cap;
    const int need = (p.n_tiles + p.cs - 1) / p.cs;           // clusters needed at one tile per CTA
    if (nclusters > need) nclusters = need;
    if (nclusters < 1) nclusters = 1;
    p.grid = nclusters * p.cs;
    p.T = (p.n_tiles + p.grid - 1) / p.grid;
    // Stage 1 over all clusters: every cluster otherwise streams ALL of L1T from L2 (K*r*2 bytes each), which is most
    // of the traffic of a decode call on the larger layers.  With the K range split over the whole grid L1T is read
    // once; the cluster-level partials of H then meet in the caller's workspace behind one grid-wide barrier (every
    // CTA is resident: the grid is at most the occupancy-queried cluster capacity).  Worth its barrier from ~16 MB
    // of avoided re-reads.
    p.ncl_k = 1;
    if (r > 0 && p.cs > 1 && nclusters > 1 && (K >> 5) >= p.grid) {
        const long long avoided = 2LL * K * r * (nclusters - 1);
        bool on = avoided >= (16LL << 20);
        if (const char* e = getenv("TWQ_DEBUG_DECODE_GRIDK")) on = atoi(e) != 0;   // testing aid: force on / off
        if (on) p.ncl_k = nclusters;
    }
    p.P = p.ng < kDecWarps ? p.ng : kDecWarps;            // upper bound; each CTA takes 16 / (its tiles), see the kernel
    if (p.T > kDecWarps * kMaxItemsPerWarp) return false;
    const int kTok = M <= 8 ? 8 : 16;
    int o = 0;
    p.off_res = o; o += (p.T > kDecWarps ? p.T : kDecWarps) * 16 * kTok * 4;   // items <= max(16, T)
    p.off_hpart = o; o += 16 * r * 4;
    p.off_h = o; o += 16 * (r + 8) * 2;
    p.off_ylr = o; o += 16 * p.T * 16 * 4;
    p.off_sx = o; o += kTok * p.ng * 4;
    o = (o + 15) & ~15;
    p.off_xs = o; o += r > 0 ? kTok * (((K >> 5) + p.cs - 1) / p.cs * 32 + 8) * 2 : 0;
    p.smem_bytes = (o + 15) & ~15;
    if (p.smem_bytes > 200 * 1024) return false;
    *out = p;
    return true;
}

cudaError_t launch_decode(const DecodeParams& p, int G, cudaStream_t stream) {
    const bool dbg = p.dbgP != nullptr;
    static const bool trace = getenv("TWQ_DEBUG_PLAN") != nullptr;
    if (trace)
        fprintf(stderr, "twq decode plan: M=%d N=%d K=%d r=%d cs=%d grid=%d T=%d P=%d smem=%d\n", p.M, p.N, p.K, p.r,
                p.cs, p.grid, p.T, p.P, p.smem_bytes);
    const int mt = p.M <= 8 ? 1 : 2;
#define TWQ_DCASE(g, m)                                                                   \
    if (G == g && mt == m) return dbg ? decode_launch_inst<g, m, true>(p, stream) : decode_launch_inst<g, m, false>(p, stream);
    TWQ_DCASE(128, 1) TWQ_DCASE(128, 2) TWQ_DCASE(64, 1) TWQ_DCASE(64, 2)
#undef TWQ_DCASE
    return cudaErrorInvalidValue;
}

}  // namespace twq
