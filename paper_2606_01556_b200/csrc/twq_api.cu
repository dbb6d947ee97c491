// twq_api.cu -- the C ABI declared in include/twq.h: argument validation (before any CUDA
// call), launch planning, TMA descriptors (cached), launch.  No compute lives here.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include <atomic>

#include "../../include/twq.h"
#include "../../include/twq_testing.h"
#include "fused_kernel.h"
#include "packed_layout.h"

namespace twq {

namespace {
std::atomic<unsigned> g_plan_flags{0u};
std::atomic<unsigned long long*> g_trace{nullptr};
}
unsigned long long* trace_buffer() { return g_trace.load(std::memory_order_relaxed); }
void g_trace_store(unsigned long long* p) { g_trace.store(p, std::memory_order_relaxed); }
unsigned plan_flags() { return g_plan_flags.load(std::memory_order_relaxed); }
void set_plan_flags(unsigned f) { g_plan_flags.store(f, std::memory_order_relaxed); }

}  // namespace twq

namespace {

thread_local int g_last_launches = 0;
constexpr int kMaxDevices = 64;

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

bool shape_ok(int M, int N, int K, int r, int G) {
    if (M < 1) return false;
    if (G != 64 && G != 128) return false;
    if (K < G || K % G != 0) return false;
    if (N < 16 || N % 16 != 0) return false;
    if (r < 0 || r > 256 || r % 16 != 0) return false;
    return true;
}

// Per-device facts, looked up once per device (relaxed atomics: the values are idempotent).
struct DevInfo {
    std::atomic<int> sms{0};      // 0 = not asked yet
    std::atomic<int> sm100{-1};   // -1 = not asked yet
};
DevInfo g_dev[kMaxDevices];

int current_device() {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return -1; }
    return dev;
}

// SM count of the current device (148 on B200; also the planning default when no device is present,
// so twq_workspace_bytes gives the same answer on a CPU-only box).
int num_sms() {
    const int dev = current_device();
    if (dev < 0 || dev >= kMaxDevices) return 148;
    int n = g_dev[dev].sms.load(std::memory_order_relaxed);
    if (n == 0) {
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) { cudaGetLastError(); return 148; }
        g_dev[dev].sms.store(n, std::memory_order_relaxed);
    }
    return n;
}

bool device_is_sm100() {
    const int dev = current_device();
    if (dev < 0) return false;
    if (dev >= kMaxDevices) {
        int major = 0;
        return cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) == cudaSuccess && major == 10;
    }
    int v = g_dev[dev].sm100.load(std::memory_order_relaxed);
    if (v < 0) {
        int major = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) { cudaGetLastError(); return false; }
        v = major == 10 ? 1 : 0;
        g_dev[dev].sm100.store(v, std::memory_order_relaxed);
    }
    return v == 1;
}

size_t ctr_bytes(const twq::FusedPlan& pl) {
    return twq::align256(static_cast<size_t>(pl.n_tiles) * pl.m_tiles * sizeof(unsigned));
}

// ------------------------------------------------------------------ the plan of a call, made once per call and cached
struct CallPlan {
    int dev, M, N, K, r, G;
    unsigned flags;
    int quant;                 // 1: planned for twq_dual_linear_x (in-kernel quantizer), 2: for twq_dual_linear_q4lr_x; only
                               // small-batch plans exist for these
    bool valid, decode;
    twq::DecodeParams dp;      // decode == true
    twq::FusedPlan fp;         // decode == false
    size_t ws_bytes;
};

const CallPlan* get_plan(int M, int N, int K, int r, int G, int quant = 0) {
    constexpr int kSlots = 16;
    thread_local CallPlan cache[kSlots];
    thread_local unsigned next = 0;
    const int dev = current_device();
    const unsigned flags = twq::plan_flags();
    for (int i = 0; i < kSlots; ++i) {
        const CallPlan& c = cache[i];
        if (c.valid && c.dev == dev && c.M == M && c.N == N && c.K == K && c.r == r && c.G == G && c.flags == flags &&
            c.quant == quant)
            return c.decode || !quant ? &c : nullptr;
    }
    CallPlan c;
    memset(&c, 0, sizeof(c));
    c.dev = dev; c.M = M; c.N = N; c.K = K; c.r = r; c.G = G; c.flags = flags; c.quant = quant;
    const int sms = num_sms();
    if (twq::decode_make_plan(M, N, K, r, G, sms, quant, &c.dp)) {
        c.decode = true;
        c.ws_bytes = 0;
    } else if (quant) {
        c.decode = false;                                      // remembered: no one-launch plan for this shape
        c.ws_bytes = 0;
    } else {
        if (!twq::fused_make_plan(M, N, K, r, G, sms, &c.fp)) return nullptr;
        c.decode = false;
        c.ws_bytes = c.fp.splits > 1 ? ctr_bytes(c.fp) + static_cast<size_t>(c.fp.splits) * M * N * sizeof(float) : 0;
    }
    c.valid = true;
    CallPlan& slot = cache[next++ % kSlots];
    slot = c;
    return slot.decode || !quant ? &slot : nullptr;
}

// ------------------------------------------------------------------ TMA descriptors, cached by everything they encode
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
    static std::atomic<EncodeTiledFn> fn{nullptr};
    EncodeTiledFn f = fn.load(std::memory_order_relaxed);
    if (!f) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess) {
            f = reinterpret_cast<EncodeTiledFn>(p);
            fn.store(f, std::memory_order_relaxed);
        }
    }
    return f;
}

struct MapKey {
    const void* ptr;
    uint64_t dim[4];
    uint64_t stride[3];      // bytes, dims 1..rank-1
    uint32_t box[4];
    int rank, dt, sw;
};

// Row-major tensor of `rank` dims (innermost first); a hit costs one 128-byte copy instead of a driver call.
bool get_map(CUtensorMap* out, const MapKey& k) {
    constexpr int kSlots = 128;
    struct Entry { MapKey key; CUtensorMap map; bool valid; };
    thread_local Entry cache[kSlots];
    uint64_t h = reinterpret_cast<uintptr_t>(k.ptr) * 0x9E3779B97F4A7C15ull;
    h ^= (k.dim[0] + 31 * k.dim[1] + 977 * k.dim[2] + 7919 * k.dim[3] + 104729ull * k.box[1] + 1299709ull * k.box[2] + k.sw) * 0xC2B2AE3D27D4EB4Full;
    Entry& e = cache[(h >> 40) % kSlots];
    if (e.valid && memcmp(&e.key, &k, sizeof(MapKey)) == 0) { *out = e.map; return true; }
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    cuuint64_t gdim[4], gstride[3];
    cuuint32_t box[4], estr[4] = {1, 1, 1, 1};
    for (int i = 0; i < 4; ++i) { gdim[i] = k.dim[i]; box[i] = k.box[i]; }
    for (int i = 0; i < 3; ++i) gstride[i] = k.stride[i];
    CUtensorMap m;
    if (enc(&m, static_cast<CUtensorMapDataType>(k.dt), static_cast<cuuint32_t>(k.rank), const_cast<void*>(k.ptr), gdim,
            gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, static_cast<CUtensorMapSwizzle>(k.sw),
            CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    e.key = k; e.map = m; e.valid = true;
    *out = m;
    return true;
}

MapKey key2d(CUtensorMapDataType dt, const void* ptr, uint64_t inner, uint64_t rows, uint64_t pitch_bytes,
             uint32_t box_inner, uint32_t box_rows, CUtensorMapSwizzle sw) {
    MapKey k;
    memset(&k, 0, sizeof(k));
    k.ptr = ptr; k.rank = 2; k.dt = static_cast<int>(dt); k.sw = static_cast<int>(sw);
    k.dim[0] = inner; k.dim[1] = rows;
    k.stride[0] = pitch_bytes;
    k.box[0] = box_inner; k.box[1] = box_rows;
    return k;
}

}  // namespace

namespace twq {
// Bytes at the front of a twq_dual_linear workspace that must be zero when a call starts (the split-K tile counters);
// 0 for shapes that need no workspace.  Used by static_ws.cu.
size_t workspace_counter_bytes(int M, int N, int K, int r, int G) {
    if (!shape_ok(M, N, K, r, G)) return 0;
    const CallPlan* cp = get_plan(M, N, K, r, G);
    return (cp && !cp->decode && cp->fp.splits > 1) ? ctr_bytes(cp->fp) : 0;
}
}  // namespace twq

extern "C" {

const char* twq_status_string(twq_status s) {
    switch (s) {
        case TWQ_OK: return "TWQ_OK";
        case TWQ_ERR_INVALID_ARG: return "TWQ_ERR_INVALID_ARG";
        case TWQ_ERR_UNSUPPORTED: return "TWQ_ERR_UNSUPPORTED";
        case TWQ_ERR_WORKSPACE: return "TWQ_ERR_WORKSPACE";
        case TWQ_ERR_CUDA: return "TWQ_ERR_CUDA";
    }
    return "TWQ_ERR_UNKNOWN";
}

int twq_last_launch_count(void) { return g_last_launches; }

void twq_testing_set_plan_flags(unsigned flags) { twq::set_plan_flags(flags); }
unsigned twq_testing_get_plan_flags(void) { return twq::plan_flags(); }
int twq_testing_set_trace_buffer(void* dev_buf) {
    twq::g_trace_store(static_cast<unsigned long long*>(dev_buf));
#ifdef TWQ_TRACE
    return 1;
#else
    return 0;
#endif
}

float twq_testing_measure_i8_tops(int iters, int reps, void* stream) {
    if (iters < 1 || reps < 1 || !device_is_sm100()) return -1.0f;
    return twq::measure_i8_tops(iters, reps, static_cast<cudaStream_t>(stream));
}

int twq_testing_cold_fill(const void* src, size_t stride, int bytes, int mode, int ctas, unsigned long long* out_ns, void* stream) {
    if (!src || !out_ns || bytes < 64 || bytes > 200 * 1024 || bytes % 64 != 0 || stride < static_cast<size_t>(bytes) || ctas < 1 ||
        (mode != 0 && mode != 1) || !device_is_sm100())
        return -1;
    return twq::launch_cold_fill(src, stride, bytes, mode, ctas, out_ns, static_cast<cudaStream_t>(stream)) == cudaSuccess ? 0 : -2;
}

int twq_testing_describe_plan(int M, int N, int K, int r, int G, int* out, int n_out) {
    if (!shape_ok(M, N, K, r, G) || !out) return -1;
    const CallPlan* cp = get_plan(M, N, K, r, G);
    if (!cp) return -1;
    int v[TWQ_PLAN_FIELDS];
    memset(v, 0, sizeof(v));
    v[TWQ_PLAN_KERNEL] = cp->decode ? 0 : 1;
    if (cp->decode) {
        v[TWQ_PLAN_CLUSTER] = cp->dp.cs; v[TWQ_PLAN_GRID] = cp->dp.grid; v[TWQ_PLAN_TILE_TOKENS] = cp->dp.mp;
        v[TWQ_PLAN_SPLITS] = 1; v[TWQ_PLAN_PAIR] = 0; v[TWQ_PLAN_SMEM] = cp->dp.smem_bytes;
        v[TWQ_PLAN_RING] = cp->dp.nslots; v[TWQ_PLAN_CHUNKS] = cp->dp.nchunks;
        v[TWQ_PLAN_S1RING] = cp->dp.l1_slots; v[TWQ_PLAN_ALIAS] = 0;
    } else {
        v[TWQ_PLAN_CLUSTER] = cp->fp.cs; v[TWQ_PLAN_GRID] = cp->fp.nclusters * cp->fp.cs; v[TWQ_PLAN_TILE_TOKENS] = cp->fp.TN;
        v[TWQ_PLAN_SPLITS] = cp->fp.splits; v[TWQ_PLAN_PAIR] = cp->fp.pair; v[TWQ_PLAN_SMEM] = cp->fp.smem_bytes;
        v[TWQ_PLAN_RING] = cp->fp.nsp; v[TWQ_PLAN_CHUNKS] = cp->fp.units;
        v[TWQ_PLAN_S1RING] = cp->fp.ns1; v[TWQ_PLAN_ALIAS] = cp->fp.alias;
    }
    for (int i = 0; i < n_out && i < TWQ_PLAN_FIELDS; ++i) out[i] = v[i];
    return TWQ_PLAN_FIELDS;
}

size_t twq_packed_bytes(int N, int K, int r, int G) {
    if (!shape_ok(1, N, K, r, G)) return 0;
    return twq::packed_layout(N, K, r, G).total;
}

twq_status twq_pack_weights(const int8_t* Rq, const void* sw, const void* L1, const void* L2, int N, int K, int r,
                            int G, void* packed, size_t packed_bytes, void* stream) {
    g_last_launches = 0;
    if (!shape_ok(1, N, K, r, G)) return TWQ_ERR_INVALID_ARG;
    if (!Rq || !sw || !packed) return TWQ_ERR_INVALID_ARG;
    if (r > 0 && (!L1 || !L2)) return TWQ_ERR_INVALID_ARG;
    if (!aligned16(Rq) || !aligned16(packed) || (reinterpret_cast<uintptr_t>(packed) & 255u)) return TWQ_ERR_INVALID_ARG;
    if (packed_bytes < twq::packed_layout(N, K, r, G).total) return TWQ_ERR_INVALID_ARG;
    if (!device_is_sm100()) return TWQ_ERR_UNSUPPORTED;
    int n = 0;
    if (twq::launch_pack_weights(Rq, sw, L1, L2, N, K, r, G, packed, static_cast<cudaStream_t>(stream), &n) !=
        cudaSuccess)
        return TWQ_ERR_CUDA;
    g_last_launches = n;
    return TWQ_OK;
}

twq_status twq_quantize_act(const void* X, int M, int K, int ldx, const float* tinv, int G, uint8_t* Xq, float* sx,
                            void* stream) {
    g_last_launches = 0;
    if (!shape_ok(M, 16, K, 0, G)) return TWQ_ERR_INVALID_ARG;
    if (!X || !Xq || !sx) return TWQ_ERR_INVALID_ARG;
    if (ldx < K || ldx % 8 != 0) return TWQ_ERR_INVALID_ARG;
    if (!aligned16(X) || !aligned16(Xq) || !aligned16(sx) || (tinv && !aligned16(tinv))) return TWQ_ERR_INVALID_ARG;
    if (!device_is_sm100()) return TWQ_ERR_UNSUPPORTED;
    if (twq::launch_quantize_act(X, M, K, ldx, tinv, G, Xq, sx, static_cast<cudaStream_t>(stream)) != cudaSuccess)
        return TWQ_ERR_CUDA;
    g_last_launches = 1;
    return TWQ_OK;
}

size_t twq_workspace_bytes(int M, int N, int K, int r, int G) {
    if (!shape_ok(M, N, K, r, G)) return 0;
    const CallPlan* cp = get_plan(M, N, K, r, G);
    return cp ? cp->ws_bytes : 0;
}

twq_status twq_dual_linear(const void* X, int ldx, const uint8_t* Xq, const float* sx, const void* packed, int M,
                           int N, int K, int r, int G, void* Y, twq_out_dtype ydt, int ldy, void* ws, size_t ws_bytes,
                           int32_t* dbg_P, void* stream) {
    g_last_launches = 0;
    if (!shape_ok(M, N, K, r, G)) return TWQ_ERR_INVALID_ARG;
    if (!Xq || !sx || !packed || !Y) return TWQ_ERR_INVALID_ARG;
    if (r > 0 && !X) return TWQ_ERR_INVALID_ARG;
    if (ydt != TWQ_OUT_BF16 && ydt != TWQ_OUT_FP16 && ydt != TWQ_OUT_FP32) return TWQ_ERR_INVALID_ARG;
    if (ldy < N) return TWQ_ERR_INVALID_ARG;
    if (r > 0 && (ldx < K || ldx % 8 != 0)) return TWQ_ERR_INVALID_ARG;
    if (!aligned16(Xq) || !aligned16(sx) || !aligned16(Y) || (X && !aligned16(X)) ||
        (reinterpret_cast<uintptr_t>(packed) & 255u))
        return TWQ_ERR_INVALID_ARG;
    const CallPlan* cp = get_plan(M, N, K, r, G);          // one plan per call (cached per shape)
    if (!cp) return TWQ_ERR_UNSUPPORTED;
    const size_t need = cp->ws_bytes;
    if (need > 0 && (!ws || ws_bytes < need)) return TWQ_ERR_WORKSPACE;
    if (need > 0 && (reinterpret_cast<uintptr_t>(ws) & 255u)) return TWQ_ERR_INVALID_ARG;
    if (!device_is_sm100()) return TWQ_ERR_UNSUPPORTED;

    const twq::PackedLayout lay = twq::packed_layout(N, K, r, G);
    const uint8_t* base = static_cast<const uint8_t*>(packed);
    const int ng = K / G;

    if (cp->decode) {
        // small batches: the bulk-copy streaming kernel of decode_kernel.cu
        twq::DecodeParams dp = cp->dp;
        dp.ldx = ldx; dp.ldy = ldy; dp.ydt = static_cast<int>(ydt);
        dp.R4 = base + lay.off_r4;
        dp.sw16 = reinterpret_cast<const __half*>(base + lay.off_sw16);
        dp.L1D = base + lay.off_l1d;
        dp.L2T = base + lay.off_l2t;
        dp.X = X; dp.sx = sx; dp.Y = Y; dp.dbgP = dbg_P;
        dp.trace = twq::trace_buffer();
        // Xq [M][K/2] as (G/2 bytes, K/G groups, M tokens); one box = gc groups of all (padded) tokens
        MapKey k;
        memset(&k, 0, sizeof(k));
        k.ptr = Xq; k.rank = 3; k.dt = static_cast<int>(CU_TENSOR_MAP_DATA_TYPE_UINT8); k.sw = static_cast<int>(CU_TENSOR_MAP_SWIZZLE_NONE);
        k.dim[0] = G / 2; k.dim[1] = ng; k.dim[2] = M;
        k.stride[0] = G / 2; k.stride[1] = K / 2;
        k.box[0] = G / 2; k.box[1] = dp.gc; k.box[2] = dp.mp;
        CUtensorMap tmXq;
        if (!get_map(&tmXq, k)) return TWQ_ERR_CUDA;
        if (twq::launch_decode(tmXq, dp, G, static_cast<cudaStream_t>(stream)) != cudaSuccess) return TWQ_ERR_CUDA;
        g_last_launches = 1;
        return TWQ_OK;
    }

    twq::FusedParams p;
    memset(&p, 0, sizeof(p));
    p.plan = cp->fp;
    const int TN = p.plan.TN;
    const int splits = p.plan.splits;

    twq::FusedMaps maps;
    memset(&maps, 0, sizeof(maps));
    bool ok = true;
    // packed INT4 tiles: rows of G/2 bytes, swizzled so that one-row-per-thread reads are conflict-free.
    // Weights: R4 [N/8][ng][8][G/2]; one box = the (8 x G/2)-byte blocks of 16 consecutive tiles for one group
    // = 128 channel rows x G/2 bytes in shared memory.
    const CUtensorMapSwizzle psw = G == 128 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_32B;
    {
        MapKey k;
        memset(&k, 0, sizeof(k));
        k.ptr = base + lay.off_r4; k.rank = 4; k.dt = static_cast<int>(CU_TENSOR_MAP_DATA_TYPE_UINT8); k.sw = static_cast<int>(psw);
        k.dim[0] = G / 2; k.dim[1] = 8; k.dim[2] = ng; k.dim[3] = N / 8;
        k.stride[0] = G / 2; k.stride[1] = 4 * static_cast<uint64_t>(G); k.stride[2] = static_cast<uint64_t>(ng) * 4 * G;
        k.box[0] = G / 2; k.box[1] = 8; k.box[2] = 1; k.box[3] = 16;
        ok &= get_map(&maps.W, k);
    }
    ok &= get_map(&maps.Xq, key2d(CU_TENSOR_MAP_DATA_TYPE_UINT8, Xq, K / 2, M, K / 2, G / 2, p.plan.pair ? TN / 2 : TN, psw));
    if (r > 0) {
        ok &= get_map(&maps.X, key2d(CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, X, K, M, static_cast<uint64_t>(ldx) * 2, 64, TN,
                                     CU_TENSOR_MAP_SWIZZLE_128B));
        ok &= get_map(&maps.L1T, key2d(CU_TENSOR_MAP_DATA_TYPE_FLOAT16, base + lay.off_l1t, K, r,
                                       static_cast<uint64_t>(K) * 2, 64, 128, CU_TENSOR_MAP_SWIZZLE_128B));
        ok &= get_map(&maps.L2T, key2d(CU_TENSOR_MAP_DATA_TYPE_FLOAT16, base + lay.off_l2t, r, N,
                                       static_cast<uint64_t>(r) * 2, 64, 128, CU_TENSOR_MAP_SWIZZLE_128B));
    }
    if (p.plan.ystage) {
        // asynchronous tile store: 16-bit outputs with a row pitch TMA accepts (a multiple of 16 bytes)
        if (static_cast<int>(ydt) <= 1 && (ldy & 7) == 0)
            ok &= get_map(&maps.Y, key2d(CU_TENSOR_MAP_DATA_TYPE_UINT16, Y, N, M, static_cast<uint64_t>(ldy) * 2, 64, TN,
                                         CU_TENSOR_MAP_SWIZZLE_128B));
        else
            p.plan.ystage = 0;     // the kernel stores from registers (the staging bytes stay unused)
    }
    if (!ok) return TWQ_ERR_CUDA;

    p.M = M; p.N = N; p.K = K; p.r = r; p.ng = ng;
    p.ldy = ldy; p.ydt = static_cast<int>(ydt);
    p.sx = sx;
    p.sw16 = reinterpret_cast<const __half*>(base + lay.off_sw16);
    p.Y = Y;
    p.dbgP = dbg_P;
    p.trace = twq::trace_buffer();
    p.ws_ctr = splits > 1 ? static_cast<unsigned*>(ws) : nullptr;
    p.ws_part = splits > 1 ? reinterpret_cast<float*>(static_cast<uint8_t*>(ws) + ctr_bytes(p.plan)) : nullptr;
    if (twq::launch_fused(maps, p, G, static_cast<cudaStream_t>(stream)) != cudaSuccess) return TWQ_ERR_CUDA;
    g_last_launches = 1;
    return TWQ_OK;
}

// Scratch for twq_dual_linear_x: nothing where the one-launch plan exists, otherwise room for the quantizer's outputs
// (codes, scales; each 256-byte aligned) in front of what twq_dual_linear itself needs.
size_t twq_workspace_bytes_x(int M, int N, int K, int r, int G) {
    if (!shape_ok(M, N, K, r, G)) return 0;
    if (get_plan(M, N, K, r, G, 1)) return 0;
    return twq::align256(static_cast<size_t>(M) * (K / 2)) + twq::align256(static_cast<size_t>(M) * (K / G) * sizeof(float)) +
           twq_workspace_bytes(M, N, K, r, G);
}

twq_status twq_dual_linear_x(const void* X, int ldx, const float* tinv, const void* packed, int M, int N, int K, int r,
                             int G, void* Y, twq_out_dtype ydt, int ldy, void* ws, size_t ws_bytes, uint8_t* Xq_out,
                             float* sx_out, int32_t* dbg_P, void* stream) {
    g_last_launches = 0;
    if (!shape_ok(M, N, K, r, G)) return TWQ_ERR_INVALID_ARG;
    if (!X || !packed || !Y) return TWQ_ERR_INVALID_ARG;
    if (ydt != TWQ_OUT_BF16 && ydt != TWQ_OUT_FP16 && ydt != TWQ_OUT_FP32) return TWQ_ERR_INVALID_ARG;
    if (ldy < N || ldx < K || ldx % 8 != 0) return TWQ_ERR_INVALID_ARG;
    if (!aligned16(X) || !aligned16(Y) || (tinv && !aligned16(tinv)) || (Xq_out && !aligned16(Xq_out)) ||
        (sx_out && !aligned16(sx_out)) || (reinterpret_cast<uintptr_t>(packed) & 255u))
        return TWQ_ERR_INVALID_ARG;
    const size_t need = twq_workspace_bytes_x(M, N, K, r, G);
    if (need > 0 && (!ws || ws_bytes < need)) return TWQ_ERR_WORKSPACE;
    if (need > 0 && (reinterpret_cast<uintptr_t>(ws) & 255u)) return TWQ_ERR_INVALID_ARG;
    if (!device_is_sm100()) return TWQ_ERR_UNSUPPORTED;
    if (const CallPlan* cp = get_plan(M, N, K, r, G, 1)) {
        // small batches: quantizer, both branches and the epilogue in ONE launch
        const twq::PackedLayout lay = twq::packed_layout(N, K, r, G);
        const uint8_t* base = static_cast<const uint8_t*>(packed);
        twq::DecodeParams dp = cp->dp;
        dp.ldx = ldx; dp.ldy = ldy; dp.ydt = static_cast<int>(ydt);
        dp.R4 = base + lay.off_r4;
        dp.sw16 = reinterpret_cast<const __half*>(base + lay.off_sw16);
        dp.L1D = base + lay.off_l1d;
        dp.L2T = base + lay.off_l2t;
        dp.X = X; dp.sx = nullptr; dp.Y = Y; dp.dbgP = dbg_P;
        dp.tinv = tinv; dp.xq_out = Xq_out; dp.sx_out = sx_out;
        dp.trace = twq::trace_buffer();
        CUtensorMap none;
        memset(&none, 0, sizeof(none));                       // the one-launch kernel issues no tensor-map copy
        if (twq::launch_decode(none, dp, G, static_cast<cudaStream_t>(stream)) != cudaSuccess) return TWQ_ERR_CUDA;
        g_last_launches = 1;
        return TWQ_OK;
    }
    // larger batches: the stand-alone quantizer into the workspace (or the caller's buffers), then the fused layer
    uint8_t* w = static_cast<uint8_t*>(ws);
    uint8_t* xq = Xq_out ? Xq_out : w;
    w += twq::align256(static_cast<size_t>(M) * (K / 2));
    float* sx = sx_out ? sx_out : reinterpret_cast<float*>(w);
    w += twq::align256(static_cast<size_t>(M) * (K / G) * sizeof(float));
    const size_t used = static_cast<size_t>(w - static_cast<uint8_t*>(ws));
    twq_status st = twq_quantize_act(X, M, K, ldx, tinv, G, xq, sx, stream);
    if (st != TWQ_OK) return st;
    st = twq_dual_linear(X, ldx, xq, sx, packed, M, N, K, r, G, Y, ydt, ldy, w, ws_bytes - used, dbg_P, stream);
    if (st != TWQ_OK) return st;
    g_last_launches = 2;
    return TWQ_OK;
}

// ------------------------------------------------------------------ the paper's 4-bit low-rank branch
static bool q4lr_rank_ok(int r) { return r >= 0 && r % 16 == 0 && (r <= 128 || r == 256); }

size_t twq_packed_bytes_q4lr(int N, int K, int r, int G) {
    if (!shape_ok(1, N, K, r, G) || !q4lr_rank_ok(r)) return 0;
    return twq::packed_layout_q4lr(N, K, r, G).total;
}

twq_status twq_pack_weights_q4lr(const int8_t* Rq, const void* sw, const int8_t* Uq, const void* su, const int8_t* Vq,
                                 const void* sv, int N, int K, int r, int G, void* packed, size_t packed_bytes,
                                 void* stream) {
    g_last_launches = 0;
    if (!shape_ok(1, N, K, r, G) || !q4lr_rank_ok(r) || r == 0) return TWQ_ERR_INVALID_ARG;
    if (!Rq || !sw || !Uq || !su || !Vq || !sv || !packed) return TWQ_ERR_INVALID_ARG;
    if (!aligned16(Rq) || (reinterpret_cast<uintptr_t>(packed) & 255u)) return TWQ_ERR_INVALID_ARG;
    if (packed_bytes < twq::packed_layout_q4lr(N, K, r, G).total) return TWQ_ERR_INVALID_ARG;
    if (!device_is_sm100()) return TWQ_ERR_UNSUPPORTED;
    int n = 0;
    if (twq::launch_pack_weights_q4lr(Rq, sw, Uq, su, Vq, sv, N, K, r, G, packed, static_cast<cudaStream_t>(stream), &n) !=
        cudaSuccess)
        return TWQ_ERR_CUDA;
    g_last_launches = n;
    return TWQ_OK;
}

twq_status twq_dual_linear_q4lr_x(const void* X, int ldx, const float* tinv, const void* packed, int M, int N, int K,
                                  int r, int G, void* Y, twq_out_dtype ydt, int ldy, uint8_t* Xq_out, float* sx_out,
                                  int32_t* dbg_P, float* dbg_H, int8_t* dbg_QH, float* dbg_sH, void* stream) {
    g_last_launches = 0;
    if (!shape_ok(M, N, K, r, G) || !q4lr_rank_ok(r) || r == 0) return TWQ_ERR_INVALID_ARG;
    if (!X || !packed || !Y) return TWQ_ERR_INVALID_ARG;
    if (ydt != TWQ_OUT_BF16 && ydt != TWQ_OUT_FP16 && ydt != TWQ_OUT_FP32) return TWQ_ERR_INVALID_ARG;
    if (ldy < N || ldx < K || ldx % 8 != 0) return TWQ_ERR_INVALID_ARG;
    if (!aligned16(X) || !aligned16(Y) || (tinv && !aligned16(tinv)) || (Xq_out && !aligned16(Xq_out)) ||
        (sx_out && !aligned16(sx_out)) || (reinterpret_cast<uintptr_t>(packed) & 255u))
        return TWQ_ERR_INVALID_ARG;
    // row slabs of at most 64 tokens (a slab start keeps every pointer 16-byte aligned: 64 rows of >= 16 bytes each)
    // (64 where the resident activation tile of 64 tokens fits in shared memory, else 32, else 16)
    int slab = 0;
    for (int s = twq::kDecodeMaxM; s >= 16 && slab == 0; s >>= 1)
        if (get_plan(M < s ? M : s, N, K, r, G, 2)) slab = s;
    if (slab == 0) return TWQ_ERR_UNSUPPORTED;
    for (int m0 = 0; m0 < M; m0 += slab)
        if (!get_plan(M - m0 < slab ? M - m0 : slab, N, K, r, G, 2)) return TWQ_ERR_UNSUPPORTED;
    if (!device_is_sm100()) return TWQ_ERR_UNSUPPORTED;
    const twq::PackedLayoutQ4 lay = twq::packed_layout_q4lr(N, K, r, G);
    const uint8_t* base = static_cast<const uint8_t*>(packed);
    const int ng = K / G;
    const size_t ybytes = ydt == TWQ_OUT_FP32 ? 4 : 2;
    CUtensorMap none;
    memset(&none, 0, sizeof(none));                           // the one-launch kernel issues no tensor-map copy
    int launches = 0;
    for (int m0 = 0; m0 < M; m0 += slab) {
        const int ms = M - m0 < slab ? M - m0 : slab;
        const CallPlan* cp = get_plan(ms, N, K, r, G, 2);
        if (!cp) return TWQ_ERR_UNSUPPORTED;
        twq::DecodeParams dp = cp->dp;
        dp.ldx = ldx; dp.ldy = ldy; dp.ydt = static_cast<int>(ydt);
        dp.R4 = base + lay.off_r4;
        dp.sw16 = reinterpret_cast<const __half*>(base + lay.off_sw16);
        dp.L1D = base + lay.off_u;
        dp.L2T = base + lay.off_v;
        dp.sv16 = reinterpret_cast<const __half*>(base + lay.off_sv16);
        dp.X = static_cast<const uint8_t*>(X) + static_cast<size_t>(m0) * ldx * 2;
        dp.sx = nullptr;
        dp.Y = static_cast<uint8_t*>(Y) + static_cast<size_t>(m0) * ldy * ybytes;
        dp.dbgP = dbg_P ? dbg_P + static_cast<size_t>(m0) * ng * N : nullptr;
        dp.dbgH = dbg_H ? dbg_H + static_cast<size_t>(m0) * r : nullptr;
        dp.dbgQH = dbg_QH ? dbg_QH + static_cast<size_t>(m0) * r : nullptr;
        dp.dbgSH = dbg_sH ? dbg_sH + static_cast<size_t>(m0) * lay.nh : nullptr;
        dp.tinv = tinv;
        dp.xq_out = Xq_out ? Xq_out + static_cast<size_t>(m0) * (K / 2) : nullptr;
        dp.sx_out = sx_out ? sx_out + static_cast<size_t>(m0) * ng : nullptr;
        dp.trace = twq::trace_buffer();
        if (twq::launch_decode(none, dp, G, static_cast<cudaStream_t>(stream)) != cudaSuccess) return TWQ_ERR_CUDA;
        ++launches;
    }
    g_last_launches = launches;
    return TWQ_OK;
}

}  // extern "C"
