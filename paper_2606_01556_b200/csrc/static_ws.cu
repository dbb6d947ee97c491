// static_ws.cu -- twq_dual_linear_noalloc: twq_dual_linear for callers that cannot allocate (code under CUDA graph
// capture, serving loops, harnesses that forbid cudaMalloc).  The only kernel of this library that needs scratch memory
// is the split-K path of the tcgen05 kernel (64 < M with few output tiles: tile counters + FP32 partial sums of Y,
// include/twq.h "ws"); here that scratch is a file-scope device array instead of a caller buffer.
//
//   * the array is TWQ_NOALLOC_MAX_WS bytes (8.5 MiB): every GPU that loads the library holds it until the process exits;
//   * in host code the array's NAME is a host-side stand-in, not a device address: its device address is looked up with
//     cudaGetSymbolAddress, once per device, with that device current, and only that pointer is handed to the kernel;
//   * this file calls no cudaMalloc / cudaFree and no allocating library routine; the existing path it forwards to
//     (twq_dual_linear) allocates nothing either;
//   * all calls share the array and it keeps the last call's contents: the counters at its front are cleared on the
//     caller's stream before every launch (a memset node, legal under capture); the partial sums are written before
//     they are read.  Two calls that overlap on the GPU (different streams, no dependency) RACE on it.
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/twq.h"
#include "fused_kernel.h"

namespace {

constexpr size_t kMaxWs = TWQ_NOALLOC_MAX_WS;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_static_ws[kMaxWs];

// Device address of g_static_ws on the CURRENT device (each device has its own instance of the array).
cudaError_t static_ws_address(void** out) {
    static std::atomic<void*> cache[kMaxDevices];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool cached = dev >= 0 && dev < kMaxDevices;
    void* p = cached ? cache[dev].load(std::memory_order_acquire) : nullptr;
    if (p == nullptr) {
        e = cudaGetSymbolAddress(&p, g_static_ws);
        if (e != cudaSuccess) return e;
        if (p == nullptr) return cudaErrorInvalidSymbol;
        if (cached) cache[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return cudaSuccess;
}

}  // namespace

extern "C" {

size_t twq_noalloc_max_workspace(void) { return kMaxWs; }

twq_status twq_dual_linear_noalloc(const void* X, int ldx, const uint8_t* Xq, const float* sx, const void* packed, int M,
                                   int N, int K, int r, int G, void* Y, twq_out_dtype ydt, int ldy, void* stream) {
    // sizes first: a shape whose scratch does not fit the array is refused before anything is touched
    const size_t need = twq_workspace_bytes(M, N, K, r, G);
    if (need > kMaxWs) return TWQ_ERR_WORKSPACE;
    void* ws = nullptr;
    if (need > 0) {
        if (static_ws_address(&ws) != cudaSuccess) { cudaGetLastError(); return TWQ_ERR_CUDA; }
        // what must start at zero: the tile counters at the front of the scratch (a failed or foreign earlier call may
        // have left anything there)
        const size_t ctr = twq::workspace_counter_bytes(M, N, K, r, G);
        if (ctr > 0 && cudaMemsetAsync(ws, 0, ctr, static_cast<cudaStream_t>(stream)) != cudaSuccess) {
            cudaGetLastError();
            return TWQ_ERR_CUDA;
        }
    }
    return twq_dual_linear(X, ldx, Xq, sx, packed, M, N, K, r, G, Y, ydt, ldy, ws, need > 0 ? kMaxWs : 0, nullptr, stream);
}

}  // extern "C"
