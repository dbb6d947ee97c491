// twq_api.cu -- the C ABI declared in include/twq.h: argument validation (before any CUDA
// call), TMA descriptor construction, launch configuration.  No compute lives here.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include "../../include/twq.h"
#include "fused_kernel.h"
#include "packed_layout.h"

namespace {

thread_local int g_last_launches = 0;

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

bool shape_ok(int M, int N, int K, int r, int G) {
    if (M < 1) return false;
    if (G != 64 && G != 128) return false;
    if (K < G || K % G != 0) return false;
    if (N < 16 || N % 16 != 0) return false;
    if (r < 0 || r > 256 || r % 16 != 0) return false;
    return true;
}

// SM count of the current device (148 on B200; also the planning default when no device is present,
// so twq_workspace_bytes gives the same answer on a CPU-only box).
int num_sms() {
    static thread_local int cached = 0;
    if (cached == 0) {
        int dev = 0, n = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0)
            cached = n;
        else
            return 148;
    }
    return cached;
}

size_t ctr_bytes(const twq::FusedPlan& pl) {
    return twq::align256(static_cast<size_t>(pl.n_tiles) * pl.m_tiles * sizeof(unsigned));
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// 2D row-major tensor [rows][inner] with a row pitch in bytes; box = [box_rows][box_inner].
bool make_map(CUtensorMap* m, CUtensorMapDataType dt, int elem_bytes, const void* ptr, uint64_t inner, uint64_t rows,
              uint64_t pitch_bytes, uint32_t box_inner, uint32_t box_rows, CUtensorMapSwizzle sw) {
    EncodeTiledFn enc = get_encode();
    if (!enc) return false;
    cuuint64_t gdim[2] = {inner, rows};
    cuuint64_t gstride[1] = {pitch_bytes};
    cuuint32_t box[2] = {box_inner, box_rows};
    cuuint32_t estr[2] = {1, 1};
    (void)elem_bytes;
    return enc(m, dt, 2, const_cast<void*>(ptr), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, sw,
               CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool device_is_sm100() {
    static thread_local int cached = -1;
    if (cached < 0) {
        int dev = 0, major = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) return false;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return false;
        cached = major == 10 ? 1 : 0;
    }
    return cached == 1;
}

}  // namespace

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
    twq::DecodeParams dp;
    if (twq::decode_make_plan(M, N, K, r, G, num_sms(), &dp)) return twq::decode_workspace_bytes(dp);   // 0 for most
    twq::FusedPlan pl;
    if (!twq::fused_make_plan(M, N, K, r, G, num_sms(), &pl)) return 0;
    if (pl.splits <= 1) return 0;
    return ctr_bytes(pl) + static_cast<size_t>(pl.splits) * M * N * sizeof(float);
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
    const size_t need = twq_workspace_bytes(M, N, K, r, G);
    if (need > 0 && (!ws || ws_bytes < need)) return TWQ_ERR_WORKSPACE;
    if (need > 0 && (reinterpret_cast<uintptr_t>(ws) & 255u)) return TWQ_ERR_INVALID_ARG;
    if (!device_is_sm100()) return TWQ_ERR_UNSUPPORTED;

    const twq::PackedLayout lay = twq::packed_layout(N, K, r, G);
    const uint8_t* base = static_cast<const uint8_t*>(packed);

    // decode-shaped calls (M <= 16): the register-resident kernel of decode_kernel.cu
    twq::DecodeParams dp;
    if (twq::decode_make_plan(M, N, K, r, G, num_sms(), &dp)) {
        dp.ldx = ldx; dp.ldy = ldy; dp.ydt = static_cast<int>(ydt);
        dp.R4 = base + lay.off_r4;
        dp.swT = reinterpret_cast<const float*>(base + lay.off_swT);
        dp.L1T = base + lay.off_l1t;
        dp.L2T = base + lay.off_l2t;
        dp.X = X; dp.Xq = Xq; dp.sx = sx; dp.Y = Y; dp.dbgP = dbg_P;
        dp.ws_ctr = static_cast<unsigned*>(ws);
        dp.ws_h = dp.ncl_k > 1 ? reinterpret_cast<float*>(static_cast<uint8_t*>(ws) + 256) : nullptr;
        if (twq::launch_decode(dp, G, static_cast<cudaStream_t>(stream)) != cudaSuccess) return TWQ_ERR_CUDA;
        g_last_launches = 1;
        return TWQ_OK;
    }

    twq::FusedParams p;
    memset(&p, 0, sizeof(p));
    if (!twq::fused_make_plan(M, N, K, r, G, num_sms(), &p.plan)) return TWQ_ERR_UNSUPPORTED;
    const int TN = p.plan.TN;
    const int splits = p.plan.splits;

    twq::FusedMaps maps;
    memset(&maps, 0, sizeof(maps));
    bool ok = true;
    // packed INT4 tiles: rows of G/2 bytes, swizzled so that one-row-per-thread reads are conflict-free
    const CUtensorMapSwizzle psw = G == 128 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_32B;
    ok &= make_map(&maps.W, CU_TENSOR_MAP_DATA_TYPE_UINT8, 1, base + lay.off_r4, K / 2, N, K / 2, G / 2, 128, psw);
    ok &= make_map(&maps.Xq, CU_TENSOR_MAP_DATA_TYPE_UINT8, 1, Xq, K / 2, M, K / 2, G / 2, p.plan.pair ? TN / 2 : TN, psw);
    if (r > 0) {
        ok &= make_map(&maps.X, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, X, K, M, static_cast<uint64_t>(ldx) * 2, 64, TN,
                       CU_TENSOR_MAP_SWIZZLE_128B);
        ok &= make_map(&maps.L1T, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, base + lay.off_l1t, K, r,
                       static_cast<uint64_t>(K) * 2, 64, 128, CU_TENSOR_MAP_SWIZZLE_128B);
        ok &= make_map(&maps.L2T, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, base + lay.off_l2t, r, N,
                       static_cast<uint64_t>(r) * 2, 64, 128, CU_TENSOR_MAP_SWIZZLE_128B);
    }
    if (p.plan.ystage) {
        // asynchronous tile store: 16-bit outputs with a row pitch TMA accepts (a multiple of 16 bytes)
        if (static_cast<int>(ydt) <= 1 && (ldy & 7) == 0)
            ok &= make_map(&maps.Y, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, Y, N, M, static_cast<uint64_t>(ldy) * 2, 64, TN,
                           CU_TENSOR_MAP_SWIZZLE_128B);
        else
            p.plan.ystage = 0;     // the kernel stores from registers (the staging bytes stay unused)
    }
    if (!ok) return TWQ_ERR_CUDA;

    p.M = M; p.N = N; p.K = K; p.r = r; p.ng = K / G;
    p.ldy = ldy; p.ydt = static_cast<int>(ydt);
    p.sx = sx;
    p.swT = reinterpret_cast<const float*>(base + lay.off_swT);
    p.Y = Y;
    p.dbgP = dbg_P;
    p.ws_ctr = splits > 1 ? static_cast<unsigned*>(ws) : nullptr;
    p.ws_part = splits > 1 ? reinterpret_cast<float*>(static_cast<uint8_t*>(ws) + ctr_bytes(p.plan)) : nullptr;
    if (twq::launch_fused(maps, p, G, static_cast<cudaStream_t>(stream)) != cudaSuccess) return TWQ_ERR_CUDA;
    g_last_launches = 1;
    return TWQ_OK;
}

}  // extern "C"
