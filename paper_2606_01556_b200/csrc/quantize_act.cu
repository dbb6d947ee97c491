// quantize_act.cu -- online per-token group quantizer (steps a1-a2 of the hot path).
//
// PAPER.md Eq. 1 (L43-47): Q_X = round(X / s_X), s_X = max|X| / q_max, q_max = 2^(k-1)-1 = 7;
// activation-side diagonal transform X*diag(lambda)^-1 (L54-58); one scale per group of G
// contiguous elements along K (L193).  The FP32 operation order is fixed by include/twq.h
// (reading R8) and must reproduce the oracle's codes and scales bit for bit, so
// this file is compiled WITHOUT fast-math and uses the *_rn intrinsics (no FMA contraction).
//
// HBM-bound: 2 B/element in, 0.5 B/element + 4 B/group out.  Each thread owns kE = 16 or 32
// consecutive k (16-byte loads, one 8- or 16-byte store); G/kE adjacent lanes form a group and
// reduce their amax with xor-shuffles.  More elements per thread mean less per-group work (two IEEE
// divides, index arithmetic) per byte: with eight the kernel was instruction-bound, not HBM-bound.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace twq {

// kIdx: index type of the chunk counter -- unsigned (32-bit divide, ~20 instructions) whenever M*K/8 < 2^31,
// which is every realistic shape; the 64-bit divide it replaces made this kernel instruction-bound (ncu r01c).
template <int kG, bool kHasT, typename kIdx = unsigned, int kE = 16>
__global__ void __launch_bounds__(256) quantize_act_kernel(const uint16_t* __restrict__ X, int M, int K, int ldx,
                                                           const float* __restrict__ tinv,
                                                           uint8_t* __restrict__ Xq, float* __restrict__ sx) {
    // Programmatic dependent launch on both sides.  This kernel is itself launched as a programmatic
    // dependent, so its blocks are scheduled while the previous kernel of the stream drains; it waits for that
    // kernel (which may have produced X, and may still read the Xq / sx buffers) before touching memory, and
    // only then lets the next kernel (twq_dual_linear) start its prologue and weight prefetch -- that kernel
    // reads X before its own griddepcontrol.wait, so the order wait -> launch_dependents matters.
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // kE = elements per thread: 32 for large problems (fewer divides and index arithmetic per byte), 16 below
    // (more threads: the small calls are latency-bound)
    constexpr int kLanesPerGroup = kG / kE;
    const int chunks_per_row = K / kE;
    const kIdx total = static_cast<kIdx>(M) * static_cast<kIdx>(chunks_per_row);
    // K % G == 0 and G % 32 == 0 guarantee that a group never straddles rows and that the
    // kLanesPerGroup lanes of a group are either all active or all inactive.
    const kIdx total_pad = (total + 31) & ~static_cast<kIdx>(31);
    for (kIdx idx = static_cast<kIdx>(blockIdx.x) * blockDim.x + threadIdx.x; idx < total_pad;
         idx += static_cast<kIdx>(gridDim.x) * blockDim.x) {
        const bool active = idx < total;
        const int m = active ? static_cast<int>(idx / static_cast<kIdx>(chunks_per_row)) : 0;
        const int c = active ? static_cast<int>(idx - static_cast<kIdx>(m) * static_cast<kIdx>(chunks_per_row)) : 0;
        float x[kE];
        if (active) {
            const uint4* src = reinterpret_cast<const uint4*>(X + static_cast<size_t>(m) * ldx + c * kE);
            uint4 rr[kE / 8];
#pragma unroll
            for (int q = 0; q < kE / 8; ++q) rr[q] = __ldg(src + q);
#pragma unroll
            for (int q = 0; q < kE / 8; ++q) {
                const uint32_t w[4] = {rr[q].x, rr[q].y, rr[q].z, rr[q].w};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    x[8 * q + 2 * i] = __uint_as_float(w[i] << 16);              // BF16 -> FP32, exact
                    x[8 * q + 2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
                }
            }
            if (kHasT) {
                const float4* tp = reinterpret_cast<const float4*>(tinv + c * kE);
#pragma unroll
                for (int q = 0; q < kE / 4; ++q) {
                    const float4 t = __ldg(tp + q);
                    x[4 * q] = __fmul_rn(x[4 * q], t.x);
                    x[4 * q + 1] = __fmul_rn(x[4 * q + 1], t.y);
                    x[4 * q + 2] = __fmul_rn(x[4 * q + 2], t.z);
                    x[4 * q + 3] = __fmul_rn(x[4 * q + 3], t.w);
                }
            }
        } else {
#pragma unroll
            for (int i = 0; i < kE; ++i) x[i] = 0.0f;
        }
        float amax = 0.0f;
#pragma unroll
        for (int i = 0; i < kE; ++i) amax = fmaxf(amax, fabsf(x[i]));
#pragma unroll
        for (int d = kLanesPerGroup / 2; d >= 1; d >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, d));
        const float amax_c = fmaxf(amax, 0x1p-30f);
        const float s = __fdiv_rn(amax_c, 7.0f);
        const float inv = __fdiv_rn(1.0f, s);
        uint32_t packed[kE / 8];
#pragma unroll
        for (int q = 0; q < kE / 8; ++q) packed[q] = 0u;
#pragma unroll
        for (int i = 0; i < kE; ++i) {
            int q = __float2int_rn(__fmul_rn(x[i], inv));  // round-half-to-even
            q = max(-7, min(7, q));
            packed[i >> 3] |= (static_cast<uint32_t>(q) & 0xFu) << (4 * (i & 7));  // low nibble = even k
        }
        if (active) {
            uint8_t* dst = Xq + static_cast<size_t>(m) * (K >> 1) + c * (kE / 2);
            if constexpr (kE == 32) *reinterpret_cast<uint4*>(dst) = make_uint4(packed[0], packed[1], packed[2], packed[3]);
            else *reinterpret_cast<uint2*>(dst) = make_uint2(packed[0], packed[1]);
            if ((c % kLanesPerGroup) == 0) sx[static_cast<size_t>(m) * (K / kG) + c / kLanesPerGroup] = s;
        }
    }
}

cudaError_t launch_quantize_act(const void* X, int M, int K, int ldx, const float* tinv, int G, uint8_t* Xq,
                                float* sx, cudaStream_t stream) {
    const bool big = static_cast<long long>(M) * K >= (1LL << 22);   // 32 elements per thread from 4 Mi elements
    const long long total = static_cast<long long>(M) * (big ? K >> 5 : K >> 4);
    const int threads = 256;
    long long blocks = (total + threads - 1) / threads;
    if (blocks > 148LL * 64) blocks = 148LL * 64;  // grid-stride beyond 64 CTAs per SM
    if (blocks < 1) blocks = 1;
    const uint16_t* Xp = static_cast<const uint16_t*>(X);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(blocks));
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr.val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    cudaError_t e;
    const bool wide = total + 8192LL * 256 >= (1LL << 31);   // 64-bit chunk counter only for > 1.7e10 elements
#define TWQ_QLAUNCH(g, t)                                                                                              \
    (wide  ? cudaLaunchKernelEx(&cfg, quantize_act_kernel<g, t, unsigned long long, 32>, Xp, M, K, ldx, tinv, Xq, sx)   \
     : big ? cudaLaunchKernelEx(&cfg, quantize_act_kernel<g, t, unsigned, 32>, Xp, M, K, ldx, tinv, Xq, sx)             \
           : cudaLaunchKernelEx(&cfg, quantize_act_kernel<g, t, unsigned, 16>, Xp, M, K, ldx, tinv, Xq, sx))
    if (G == 128) e = tinv ? TWQ_QLAUNCH(128, true) : TWQ_QLAUNCH(128, false);
    else e = tinv ? TWQ_QLAUNCH(64, true) : TWQ_QLAUNCH(64, false);
#undef TWQ_QLAUNCH
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

}  // namespace twq
