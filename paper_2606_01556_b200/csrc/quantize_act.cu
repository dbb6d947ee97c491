// quantize_act.cu -- online per-token group quantizer (steps a1-a2 of the hot path).
//
// PAPER.md Eq. 1 (L43-47): Q_X = round(X / s_X), s_X = max|X| / q_max, q_max = 2^(k-1)-1 = 7;
// activation-side diagonal transform X*diag(lambda)^-1 (L54-58); one scale per group of G
// contiguous elements along K (L193).  The FP32 operation order is fixed by include/twq.h
// (reading R8) and must reproduce the oracle's codes and scales bit for bit, so
// this file is compiled WITHOUT fast-math and uses the *_rn intrinsics (no FMA contraction).
//
// HBM-bound: 2 B/element in, 0.5 B/element + 4 B/group out.  Each thread owns 16
// consecutive k (two 16-byte loads of one 32-byte sector, one 8-byte store); G/16 adjacent lanes
// form a group and reduce their amax with xor-shuffles, so a warp covers 512 contiguous elements of
// one row (1 KB in, 256 B out).  Sixteen elements per thread halve the per-group work (two IEEE
// divides, index arithmetic) per byte: with eight the kernel was instruction-bound, not HBM-bound.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace twq {

// kIdx: index type of the chunk counter -- unsigned (32-bit divide, ~20 instructions) whenever M*K/8 < 2^31,
// which is every realistic shape; the 64-bit divide it replaces made this kernel instruction-bound (ncu r01c).
template <int kG, bool kHasT, typename kIdx = unsigned>
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
    constexpr int kLanesPerGroup = kG / 16;
    const int chunks_per_row = K >> 4;  // 16-element chunks
    const kIdx total = static_cast<kIdx>(M) * static_cast<kIdx>(chunks_per_row);
    // K % G == 0 and G % 16 == 0 guarantee that a group never straddles rows and that the
    // kLanesPerGroup lanes of a group are either all active or all inactive.
    const kIdx total_pad = (total + 31) & ~static_cast<kIdx>(31);
    for (kIdx idx = static_cast<kIdx>(blockIdx.x) * blockDim.x + threadIdx.x; idx < total_pad;
         idx += static_cast<kIdx>(gridDim.x) * blockDim.x) {
        const bool active = idx < total;
        const int m = active ? static_cast<int>(idx / static_cast<kIdx>(chunks_per_row)) : 0;
        const int c = active ? static_cast<int>(idx - static_cast<kIdx>(m) * static_cast<kIdx>(chunks_per_row)) : 0;
        float x[16];
        if (active) {
            const uint4* src = reinterpret_cast<const uint4*>(X + static_cast<size_t>(m) * ldx + c * 16);
            const uint4 r0 = __ldg(src), r1 = __ldg(src + 1);
            const uint32_t w[8] = {r0.x, r0.y, r0.z, r0.w, r1.x, r1.y, r1.z, r1.w};
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                x[2 * i] = __uint_as_float(w[i] << 16);              // BF16 -> FP32, exact
                x[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
            }
            if (kHasT) {
                const float4* tp = reinterpret_cast<const float4*>(tinv + c * 16);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float4 t = __ldg(tp + q);
                    x[4 * q] = __fmul_rn(x[4 * q], t.x);
                    x[4 * q + 1] = __fmul_rn(x[4 * q + 1], t.y);
                    x[4 * q + 2] = __fmul_rn(x[4 * q + 2], t.z);
                    x[4 * q + 3] = __fmul_rn(x[4 * q + 3], t.w);
                }
            }
        } else {
#pragma unroll
            for (int i = 0; i < 16; ++i) x[i] = 0.0f;
        }
        float amax = 0.0f;
#pragma unroll
        for (int i = 0; i < 16; ++i) amax = fmaxf(amax, fabsf(x[i]));
#pragma unroll
        for (int d = kLanesPerGroup / 2; d >= 1; d >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, d));
        const float amax_c = fmaxf(amax, 0x1p-30f);
        const float s = __fdiv_rn(amax_c, 7.0f);
        const float inv = __fdiv_rn(1.0f, s);
        uint32_t packed[2] = {0u, 0u};
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            int q = __float2int_rn(__fmul_rn(x[i], inv));  // round-half-to-even
            q = max(-7, min(7, q));
            packed[i >> 3] |= (static_cast<uint32_t>(q) & 0xFu) << (4 * (i & 7));  // low nibble = even k
        }
        if (active) {
            *reinterpret_cast<uint2*>(Xq + static_cast<size_t>(m) * (K >> 1) + c * 8) = make_uint2(packed[0], packed[1]);
            if ((c % kLanesPerGroup) == 0) sx[static_cast<size_t>(m) * (K / kG) + c / kLanesPerGroup] = s;
        }
    }
}

cudaError_t launch_quantize_act(const void* X, int M, int K, int ldx, const float* tinv, int G, uint8_t* Xq,
                                float* sx, cudaStream_t stream) {
    const long long total = static_cast<long long>(M) * (K >> 4);
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
#define TWQ_QLAUNCH(g, t)                                                                                        \
    (wide ? cudaLaunchKernelEx(&cfg, quantize_act_kernel<g, t, unsigned long long>, Xp, M, K, ldx, tinv, Xq, sx)  \
          : cudaLaunchKernelEx(&cfg, quantize_act_kernel<g, t, unsigned>, Xp, M, K, ldx, tinv, Xq, sx))
    if (G == 128) e = tinv ? TWQ_QLAUNCH(128, true) : TWQ_QLAUNCH(128, false);
    else e = tinv ? TWQ_QLAUNCH(64, true) : TWQ_QLAUNCH(64, false);
#undef TWQ_QLAUNCH
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

}  // namespace twq
