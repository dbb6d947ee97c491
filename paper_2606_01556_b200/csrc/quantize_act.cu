// quantize_act.cu -- online per-token group quantizer (steps a1-a2 of the hot path).
//
// PAPER.md Eq. 1 (L43-47): Q_X = round(X / s_X), s_X = max|X| / q_max, q_max = 2^(k-1)-1 = 7;
// activation-side diagonal transform X*diag(lambda)^-1 (L54-58); one scale per group of G
// contiguous elements along K (L193).  The FP32 operation order is fixed by include/twq.h
// (reading R8) and must reproduce the oracle's codes and scales bit for bit, so
// this file is compiled WITHOUT fast-math and uses the *_rn intrinsics (no FMA contraction).
//
// HBM-bound: 2 B/element in, 0.5 B/element + 4 B/group out.  Each thread owns 8
// consecutive k (one 16-byte load, one 4-byte store); G/8 adjacent lanes form a group and
// reduce their amax with xor-shuffles, so a warp covers 256 contiguous elements of one row
// with fully coalesced 512-byte loads and 128-byte stores.
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace twq {

template <int kG, bool kHasT>
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
    constexpr int kLanesPerGroup = kG / 8;
    const int chunks_per_row = K >> 3;  // 8-element chunks
    const long long total = static_cast<long long>(M) * chunks_per_row;
    // K % G == 0 and G % 8 == 0 guarantee that a group never straddles rows and that the
    // kLanesPerGroup lanes of a group are either all active or all inactive.
    for (long long idx = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x;
         idx < ((total + 31) & ~31LL); idx += static_cast<long long>(gridDim.x) * blockDim.x) {
        const bool active = idx < total;
        const int m = active ? static_cast<int>(idx / chunks_per_row) : 0;
        const int c = active ? static_cast<int>(idx - static_cast<long long>(m) * chunks_per_row) : 0;
        float x[8];
        if (active) {
            const uint4 raw = __ldg(reinterpret_cast<const uint4*>(X + static_cast<size_t>(m) * ldx + c * 8));
            const uint32_t w[4] = {raw.x, raw.y, raw.z, raw.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                x[2 * i] = __uint_as_float(w[i] << 16);              // BF16 -> FP32, exact
                x[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
            }
            if (kHasT) {
                const float4 t0 = __ldg(reinterpret_cast<const float4*>(tinv + c * 8));
                const float4 t1 = __ldg(reinterpret_cast<const float4*>(tinv + c * 8 + 4));
                const float t[8] = {t0.x, t0.y, t0.z, t0.w, t1.x, t1.y, t1.z, t1.w};
#pragma unroll
                for (int i = 0; i < 8; ++i) x[i] = __fmul_rn(x[i], t[i]);
            }
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i) x[i] = 0.0f;
        }
        float amax = 0.0f;
#pragma unroll
        for (int i = 0; i < 8; ++i) amax = fmaxf(amax, fabsf(x[i]));
#pragma unroll
        for (int d = kLanesPerGroup / 2; d >= 1; d >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, d));
        const float amax_c = fmaxf(amax, 0x1p-30f);
        const float s = __fdiv_rn(amax_c, 7.0f);
        const float inv = __fdiv_rn(1.0f, s);
        uint32_t packed = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            int q = __float2int_rn(__fmul_rn(x[i], inv));  // round-half-to-even
            q = max(-7, min(7, q));
            packed |= (static_cast<uint32_t>(q) & 0xFu) << (4 * i);  // low nibble = even k
        }
        if (active) {
            *reinterpret_cast<uint32_t*>(Xq + static_cast<size_t>(m) * (K >> 1) + c * 4) = packed;
            if ((c % kLanesPerGroup) == 0) sx[static_cast<size_t>(m) * (K / kG) + c / kLanesPerGroup] = s;
        }
    }
}

cudaError_t launch_quantize_act(const void* X, int M, int K, int ldx, const float* tinv, int G, uint8_t* Xq,
                                float* sx, cudaStream_t stream) {
    const long long total = static_cast<long long>(M) * (K >> 3);
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
    if (G == 128) {
        if (tinv) e = cudaLaunchKernelEx(&cfg, quantize_act_kernel<128, true>, Xp, M, K, ldx, tinv, Xq, sx);
        else e = cudaLaunchKernelEx(&cfg, quantize_act_kernel<128, false>, Xp, M, K, ldx, tinv, Xq, sx);
    } else {
        if (tinv) e = cudaLaunchKernelEx(&cfg, quantize_act_kernel<64, true>, Xp, M, K, ldx, tinv, Xq, sx);
        else e = cudaLaunchKernelEx(&cfg, quantize_act_kernel<64, false>, Xp, M, K, ldx, tinv, Xq, sx);
    }
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

}  // namespace twq
