// cold_fill.cu -- measurement aid for bench.py, not on the product path: how long does it take to bring `bytes_per_cta` of COLD
// global memory into the shared memory of every SM at once (one CTA per SM), by bulk copies (the small-batch kernel's mechanism)
// or by plain 16-byte loads?  This is the floor under any decode-shaped call that streams its weights once: the HBM roofline
// (bytes / bandwidth) ignores the latency of the first byte and the ramp of a one-shot burst.  Exported as
// twq_testing_measure_cold_fill (include/twq_testing.h); the caller provides the buffer (the library never allocates) and
// rotates regions so that nothing is L2-resident.
#include <cuda_runtime.h>
#include <stdint.h>

#include "sm100_ptx.cuh"

namespace twq {

namespace {

constexpr int kFillThreads = 512;
constexpr int kFillSmem = 200 * 1024;

// mode 0: four bulk copies per CTA (issued by four lanes), completion on one mbarrier; mode 1: 16-byte loads, eight in flight
// per thread, stored to shared memory.  tout[cta] = nanoseconds (%globaltimer) from the first instruction to the last byte.
__global__ void __launch_bounds__(kFillThreads, 1) cold_fill_kernel(const uint8_t* src, size_t stride, int bytes, int mode,
                                                                    unsigned long long* tout) {
    extern __shared__ __align__(128) uint8_t fsm[];
    uint64_t* bar = reinterpret_cast<uint64_t*>(fsm + kFillSmem);
    if (threadIdx.x == 0) {
        mbar_init(bar, 1);
        fence_mbar_init();
    }
    __syncthreads();
    unsigned long long t0, t1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
    const uint8_t* base = src + static_cast<size_t>(blockIdx.x) * stride;
    if (mode == 0) {
        const int piece = (bytes / 4) & ~15;
        if (threadIdx.x == 0) mbar_arrive_expect_tx_a(smem_u32(bar), static_cast<uint32_t>(4 * piece));
        __syncthreads();
        if (threadIdx.x < 4)
            bulk_load_1d_a(smem_u32(fsm) + threadIdx.x * piece, base + static_cast<size_t>(threadIdx.x) * piece,
                           static_cast<uint32_t>(piece), smem_u32(bar), policy_evict_first());
        if (threadIdx.x == 32) {
            mbar_wait_a(smem_u32(bar), 0);
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
            tout[blockIdx.x] = t1 - t0;
        }
    } else {
        const uint4* b4 = reinterpret_cast<const uint4*>(base);
        const int n = bytes / 16;
        for (int i0 = threadIdx.x; i0 < n; i0 += 8 * kFillThreads) {
            uint4 v[8];
#pragma unroll
            for (int q = 0; q < 8; ++q)
                if (i0 + q * kFillThreads < n)
                    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                                 : "=r"(v[q].x), "=r"(v[q].y), "=r"(v[q].z), "=r"(v[q].w) : "l"(b4 + i0 + q * kFillThreads));
#pragma unroll
            for (int q = 0; q < 8; ++q)
                if (i0 + q * kFillThreads < n) reinterpret_cast<uint4*>(fsm)[i0 + q * kFillThreads] = v[q];
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
            tout[blockIdx.x] = t1 - t0;
        }
    }
}

}  // namespace

// One launch over `ctas` CTAs; region = src + r * ctas * stride chosen by the caller.  Returns cudaSuccess / an error.
cudaError_t launch_cold_fill(const void* src, size_t stride, int bytes, int mode, int ctas, unsigned long long* tout,
                             cudaStream_t stream) {
    static bool done = false;
    if (!done) {
        cudaError_t e = cudaFuncSetAttribute(cold_fill_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kFillSmem + 64);
        if (e != cudaSuccess) return e;
        done = true;
    }
    cold_fill_kernel<<<ctas, kFillThreads, kFillSmem + 64, stream>>>(static_cast<const uint8_t*>(src), stride, bytes, mode, tout);
    return cudaGetLastError();
}

}  // namespace twq
