// peak_i8.cu -- measurement aid for bench.py, not on the product path: an MMA-only loop of
// tcgen05.mma kind::i8 (128 x 128 x 32, operands in shared memory, accumulator in TMEM) on every SM, timed with
// CUDA events.  It answers SURVEY.md 8(d): "have the bench measure an MMA-only kind::i8 loop to confirm" the
// int8 = 2 x BF16 tensor peak that the prefill roofline uses.  Exported as twq_testing_measure_i8_tops
// (include/twq_testing.h).  The operand bytes are whatever the shared memory holds: only the rate matters.
#include <cuda_runtime.h>
#include <stdint.h>

#include "sm100_ptx.cuh"

namespace twq {

namespace {

constexpr int kPeakThreads = 128;
constexpr int kPeakCols = 256;        // two 128-column accumulators, alternated

__global__ void __launch_bounds__(kPeakThreads, 1) peak_i8_kernel(int iters) {
    extern __shared__ uint8_t psm_raw[];
    uint8_t* psm = psm_raw + ((1024u - (smem_u32(psm_raw) & 1023u)) & 1023u);
    uint64_t* bar = reinterpret_cast<uint64_t*>(psm + 16384);
    uint32_t* slot = reinterpret_cast<uint32_t*>(psm + 16384 + 64);
    const int warp = threadIdx.x >> 5;
    for (int i = threadIdx.x; i < 16384 / 4; i += kPeakThreads) reinterpret_cast<uint32_t*>(psm)[i] = 0x01020304u * (i + 1);
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        fence_mbar_init();
    }
    if (warp == 0) tmem_alloc<kPeakCols>(slot);
    fence_proxy_async_smem();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *slot;
    if (warp == 1) {
        // A: 128 rows x 32 bytes, B: 128 rows x 32 bytes, both K-major with the 32-byte swizzle
        const uint64_t adesc = umma_smem_desc<32>(smem_u32(psm));
        const uint64_t bdesc = umma_smem_desc<32>(smem_u32(psm + 8192));
        const uint32_t idesc = umma_idesc(2, 1, 1, 128, 128);      // D s32, A s8, B s8
        for (int it = 0; it < iters; ++it) {
            if (elect_one()) {
#pragma unroll
                for (int k = 0; k < 8; ++k) umma_i8(tmem + (k & 1) * 128, adesc, bdesc, idesc, 1u);
            }
            __syncwarp();
        }
        if (elect_one()) tc_commit(bar);
        __syncwarp();
        mbar_wait(bar, 0);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) {
        tc_fence_after();
        tmem_dealloc<kPeakCols>(tmem);
    }
}

}  // namespace

// Returns the measured dense int8 rate in TOP/s (2 ops per MAC) over `reps` launches of `iters` x 8 MMAs per SM,
// or a negative value on failure.
float measure_i8_tops(int iters, int reps, cudaStream_t stream) {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return -1.0f;
    const size_t smem = 16384 + 1024 + 256;
    if (cudaFuncSetAttribute(peak_i8_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem)) != cudaSuccess)
        return -1.0f;
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -1.0f;
    peak_i8_kernel<<<sms, kPeakThreads, smem, stream>>>(iters);      // warm-up
    float best = 0.0f;
    for (int r = 0; r < reps; ++r) {
        cudaEventRecord(e0, stream);
        peak_i8_kernel<<<sms, kPeakThreads, smem, stream>>>(iters);
        cudaEventRecord(e1, stream);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1.0f; break; }
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double ops = 2.0 * 128 * 128 * 32 * 8.0 * iters * sms;
        const float tops = static_cast<float>(ops / (ms * 1e-3) / 1e12);
        if (tops > best) best = tops;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (cudaGetLastError() != cudaSuccess) return -1.0f;
    return best;
}

}  // namespace twq
