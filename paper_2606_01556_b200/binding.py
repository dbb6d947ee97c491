"""ctypes binding of include/twq.h.  Names and argument order follow the C ABI."""
from __future__ import annotations

import ctypes
import dataclasses
import os

import torch

from . import _build

OUT_BF16, OUT_FP16, OUT_FP32 = 0, 1, 2
_STATUS = {0: "TWQ_OK", 1: "TWQ_ERR_INVALID_ARG", 2: "TWQ_ERR_UNSUPPORTED", 3: "TWQ_ERR_WORKSPACE", 4: "TWQ_ERR_CUDA"}
_OUT_TORCH = {OUT_BF16: torch.bfloat16, OUT_FP16: torch.float16, OUT_FP32: torch.float32}

EXPORTS = ("twq_status_string", "twq_packed_bytes", "twq_pack_weights", "twq_quantize_act",
           "twq_workspace_bytes", "twq_dual_linear", "twq_workspace_bytes_x", "twq_dual_linear_x", "twq_last_launch_count",
           "twq_packed_bytes_q4lr", "twq_pack_weights_q4lr", "twq_dual_linear_q4lr_x",
           "twq_noalloc_max_workspace", "twq_dual_linear_noalloc")


TESTING_EXPORTS = ("twq_testing_set_plan_flags", "twq_testing_get_plan_flags", "twq_testing_describe_plan",
                   "twq_testing_set_trace_buffer", "twq_testing_measure_i8_tops", "twq_testing_cold_fill")
# include/twq_testing.h: planner overrides for tests
PLAN_NO_SPLIT, PLAN_NO_PAIR, PLAN_NO_YSTAGE, PLAN_NO_ALIAS2, PLAN_NO_DECODE = 1, 2, 4, 8, 16
_PLAN_FIELDS = ("kernel", "cluster", "grid", "tile_tokens", "splits", "pair", "smem", "ring", "chunks", "s1_ring", "alias")


def plan_fused_cs(c: int) -> int:
    return (c & 15) << 8


def plan_decode_cs(c: int) -> int:
    return (c & 31) << 12


def plan_fused_tn_cap(c: int) -> int:
    """TWQ_PLAN_FUSED_TN_CAP: 1 = token tile of the tcgen05 kernel at most 64, 2 = at most 32."""
    return (c & 3) << 17


class TwqError(RuntimeError):
    def __init__(self, code: int, where: str):
        super().__init__(f"{where}: {_STATUS.get(code, code)}")
        self.code = code


_lib = None


def lib_path() -> str:
    return _build.LIB


def load_library(build_if_missing: bool = True):
    """Load libtwq.so (building it in-tree with nvcc if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if build_if_missing and _build.needs_build():
        path = _build.build()
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} not built; run python -m paper_2606_01556_b200._build")
    lib = ctypes.CDLL(path)
    vp, i, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
    lib.twq_status_string.restype = ctypes.c_char_p
    lib.twq_status_string.argtypes = [i]
    lib.twq_packed_bytes.restype = sz
    lib.twq_packed_bytes.argtypes = [i, i, i, i]
    lib.twq_pack_weights.restype = i
    lib.twq_pack_weights.argtypes = [vp, vp, vp, vp, i, i, i, i, vp, sz, vp]
    lib.twq_quantize_act.restype = i
    lib.twq_quantize_act.argtypes = [vp, i, i, i, vp, i, vp, vp, vp]
    lib.twq_workspace_bytes.restype = sz
    lib.twq_workspace_bytes.argtypes = [i, i, i, i, i]
    lib.twq_dual_linear.restype = i
    lib.twq_dual_linear.argtypes = [vp, i, vp, vp, vp, i, i, i, i, i, vp, i, i, vp, sz, vp, vp]
    lib.twq_workspace_bytes_x.restype = sz
    lib.twq_workspace_bytes_x.argtypes = [i, i, i, i, i]
    lib.twq_dual_linear_x.restype = i
    lib.twq_dual_linear_x.argtypes = [vp, i, vp, vp, i, i, i, i, i, vp, i, i, vp, sz, vp, vp, vp, vp]
    lib.twq_last_launch_count.restype = i
    lib.twq_last_launch_count.argtypes = []
    lib.twq_packed_bytes_q4lr.restype = sz
    lib.twq_packed_bytes_q4lr.argtypes = [i, i, i, i]
    lib.twq_pack_weights_q4lr.restype = i
    lib.twq_pack_weights_q4lr.argtypes = [vp, vp, vp, vp, vp, vp, i, i, i, i, vp, sz, vp]
    lib.twq_dual_linear_q4lr_x.restype = i
    lib.twq_dual_linear_q4lr_x.argtypes = [vp, i, vp, vp, i, i, i, i, i, vp, i, i, vp, vp, vp, vp, vp, vp, vp]
    lib.twq_noalloc_max_workspace.restype = sz
    lib.twq_noalloc_max_workspace.argtypes = []
    lib.twq_dual_linear_noalloc.restype = i
    lib.twq_dual_linear_noalloc.argtypes = [vp, i, vp, vp, vp, i, i, i, i, i, vp, i, i, vp]
    # testing hooks (include/twq_testing.h): not part of the product ABI
    lib.twq_testing_set_plan_flags.restype = None
    lib.twq_testing_set_plan_flags.argtypes = [ctypes.c_uint]
    lib.twq_testing_get_plan_flags.restype = ctypes.c_uint
    lib.twq_testing_get_plan_flags.argtypes = []
    lib.twq_testing_describe_plan.restype = i
    lib.twq_testing_describe_plan.argtypes = [i, i, i, i, i, ctypes.POINTER(ctypes.c_int), i]
    lib.twq_testing_set_trace_buffer.restype = i
    lib.twq_testing_set_trace_buffer.argtypes = [vp]
    lib.twq_testing_measure_i8_tops.restype = ctypes.c_float
    lib.twq_testing_measure_i8_tops.argtypes = [i, i, vp]
    lib.twq_testing_cold_fill.restype = i
    lib.twq_testing_cold_fill.argtypes = [vp, sz, i, i, i, vp, vp]
    _lib = lib
    return lib


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def _check(code: int, where: str):
    if code != 0:
        raise TwqError(code, where)


def packed_bytes(N: int, K: int, r: int, G: int) -> int:
    return int(load_library().twq_packed_bytes(N, K, r, G))


def workspace_bytes(M: int, N: int, K: int, r: int, G: int) -> int:
    return int(load_library().twq_workspace_bytes(M, N, K, r, G))


def last_launch_count() -> int:
    return int(load_library().twq_last_launch_count())


def testing_set_plan_flags(flags: int) -> None:
    """include/twq_testing.h: process-wide planner overrides (0 = production)."""
    _wsx_cache.clear()
    load_library().twq_testing_set_plan_flags(flags)


def testing_set_trace_buffer(buf) -> bool:
    """csrc/trace.cuh: hand a CUDA uint64 tensor (>= 16384 words) or None; True if the timeline is compiled in."""
    return bool(load_library().twq_testing_set_trace_buffer(_ptr(buf)))


def testing_measure_i8_tops(iters: int = 4096, reps: int = 5) -> float:
    """csrc/peak_i8.cu: measured tcgen05 kind::i8 rate in TOP/s (synchronises)."""
    return float(load_library().twq_testing_measure_i8_tops(iters, reps, _stream()))


def testing_cold_fill_us(bytes_per_cta: int, mode: int, ctas: int = 148, reps: int = 12) -> dict:
    """csrc/cold_fill.cu: microseconds until every one of `ctas` CTAs has `bytes_per_cta` of COLD global memory in its shared
    memory (mode 0 bulk copies, 1 plain loads).  Regions rotate through > 2 x L2; median over reps of the slowest and of the
    median CTA.  Synchronises."""
    lib = load_library()
    stride = (bytes_per_cta + 255) // 256 * 256
    region = stride * ctas
    nreg = max(reps, (2 * 126 * 1024 * 1024) // region + 2)
    buf = torch.ones(nreg * region, dtype=torch.uint8, device="cuda")
    out = torch.zeros(ctas, dtype=torch.int64, device="cuda")
    mx, med = [], []
    for rep in range(nreg + reps):
        base = ctypes.c_void_p(buf.data_ptr() + (rep % nreg) * region)
        code = lib.twq_testing_cold_fill(base, stride, bytes_per_cta, mode, ctas, _ptr(out), _stream())
        if code != 0:
            raise TwqError(4 if code == -2 else 1, "twq_testing_cold_fill")
        torch.cuda.synchronize()
        if rep >= nreg:                      # the first lap only makes sure every region has left L2 since it was written
            t = out.sort().values
            mx.append(int(t[-1])); med.append(int(t[ctas // 2]))
    mx.sort(); med.sort()
    return dict(slowest_cta_us=mx[len(mx) // 2] / 1e3, median_cta_us=med[len(med) // 2] / 1e3, bytes_per_cta=bytes_per_cta, ctas=ctas,
                mode="bulk" if mode == 0 else "ldg")


def testing_describe_plan(M: int, N: int, K: int, r: int, G: int) -> dict:
    """The launch plan twq_dual_linear would use: kernel ('decode' / 'tcgen05'), cluster, grid, ..."""
    out = (ctypes.c_int * len(_PLAN_FIELDS))()
    n = load_library().twq_testing_describe_plan(M, N, K, r, G, out, len(_PLAN_FIELDS))
    if n < 0:
        raise TwqError(1, "twq_testing_describe_plan")
    d = dict(zip(_PLAN_FIELDS, [int(v) for v in out]))
    d["kernel"] = "decode" if d["kernel"] == 0 else "tcgen05"
    return d


@dataclasses.dataclass
class PackedLayer:
    """Opaque packed weights of one layer + the shape they were packed for."""
    blob: torch.Tensor
    N: int
    K: int
    r: int
    G: int


def pack_weights(Rq: torch.Tensor, sw: torch.Tensor, L1, L2, G: int, stream=None) -> PackedLayer:
    """twq_pack_weights.  Rq int8 [N,K] codes, sw fp16 [N,K/G], L1 fp16 [K,r], L2 fp16 [r,N] (device)."""
    N, K = Rq.shape
    r = 0 if L1 is None else int(L1.shape[1])
    nbytes = packed_bytes(N, K, r, G)
    if nbytes == 0:
        raise TwqError(1, "twq_packed_bytes")
    blob = torch.empty(nbytes, dtype=torch.uint8, device=Rq.device)
    assert Rq.dtype == torch.int8 and Rq.is_contiguous() and sw.dtype == torch.float16 and sw.is_contiguous()
    if r > 0:
        assert L1.dtype == torch.float16 and L2.dtype == torch.float16 and L1.is_contiguous() and L2.is_contiguous()
        assert tuple(L1.shape) == (K, r) and tuple(L2.shape) == (r, N)
    code = load_library().twq_pack_weights(_ptr(Rq), _ptr(sw), _ptr(L1) if r else None, _ptr(L2) if r else None,
                                           N, K, r, G, _ptr(blob), nbytes, _stream(stream))
    _check(code, "twq_pack_weights")
    return PackedLayer(blob, N, K, r, G)


def quantize_act(X: torch.Tensor, G: int, tinv=None, out=None, stream=None):
    """twq_quantize_act.  X bf16 [M,K] (row stride = X.stride(0)); returns (Xq u8 [M,K/2], sx f32 [M,K/G])."""
    M, K = X.shape
    assert X.dtype == torch.bfloat16 and X.stride(1) == 1
    if out is None:
        Xq = torch.empty((M, K // 2), dtype=torch.uint8, device=X.device)
        sx = torch.empty((M, K // G), dtype=torch.float32, device=X.device)
    else:
        Xq, sx = out
    code = load_library().twq_quantize_act(_ptr(X), M, K, X.stride(0), _ptr(tinv), G, _ptr(Xq), _ptr(sx),
                                           _stream(stream))
    _check(code, "twq_quantize_act")
    return Xq, sx


_ws_cache = {}


def _cached_workspace(need: int, device, stream):
    """One zero-initialised workspace per (device, stream), grown on demand and zeroed ON that stream: the library
    leaves its counters at zero after every call, so the buffer is reused without clearing, and no memset is
    queued between a call and its stream predecessor."""
    s = torch.cuda.current_stream(device) if stream is None else stream
    key = (device.index if device.index is not None else torch.cuda.current_device(), s.cuda_stream)
    buf = _ws_cache.get(key)
    if buf is None or buf.numel() < need:
        with torch.cuda.stream(s):
            buf = torch.zeros(need, dtype=torch.uint8, device=device)
        _ws_cache[key] = buf
    return buf


def dual_linear(X, Xq, sx, packed: PackedLayer, out_dtype: int = OUT_BF16, Y=None, ws=None, dbg_P=None,
                stream=None):
    """twq_dual_linear.  Returns Y [M,N] in out_dtype.  `ws` must be a zero-initialised uint8 tensor of at
    least workspace_bytes(...) when that is non-zero (allocated here if omitted)."""
    M = Xq.shape[0]
    N, K, r, G = packed.N, packed.K, packed.r, packed.G
    if Y is None:
        Y = torch.empty((M, N), dtype=_OUT_TORCH.get(out_dtype, torch.bfloat16), device=Xq.device)
    need = workspace_bytes(M, N, K, r, G)
    if need and ws is None:
        ws = _cached_workspace(need, Xq.device, stream)
    ldx = X.stride(0) if X is not None else K
    code = load_library().twq_dual_linear(_ptr(X) if r else None, ldx, _ptr(Xq), _ptr(sx), _ptr(packed.blob),
                                          M, N, K, r, G, _ptr(Y), out_dtype, Y.stride(0), _ptr(ws),
                                          0 if ws is None else ws.numel(), _ptr(dbg_P), _stream(stream))
    _check(code, "twq_dual_linear")
    return Y


def noalloc_max_workspace() -> int:
    return int(load_library().twq_noalloc_max_workspace())


def dual_linear_noalloc(X, Xq, sx, packed: PackedLayer, Y, out_dtype: int = OUT_BF16, stream=None):
    """twq_dual_linear_noalloc: twq_dual_linear with the library's static scratch (include/twq.h); the caller passes the
    output too, so that nothing at all is allocated by the call."""
    M = Xq.shape[0]
    N, K, r, G = packed.N, packed.K, packed.r, packed.G
    ldx = X.stride(0) if X is not None else K
    code = load_library().twq_dual_linear_noalloc(_ptr(X) if r else None, ldx, _ptr(Xq), _ptr(sx), _ptr(packed.blob),
                                                  M, N, K, r, G, _ptr(Y), out_dtype, Y.stride(0), _stream(stream))
    _check(code, "twq_dual_linear_noalloc")
    return Y


_wsx_cache = {}


def workspace_bytes_x(M: int, N: int, K: int, r: int, G: int) -> int:
    """twq_workspace_bytes_x, remembered per shape (a pure function of the shape and the planner flags; the cache is cleared
    by testing_set_plan_flags): saves a library call per twq_dual_linear_x call on the host."""
    key = (M, N, K, r, G)
    v = _wsx_cache.get(key)
    if v is None:
        v = int(load_library().twq_workspace_bytes_x(M, N, K, r, G))
        _wsx_cache[key] = v
    return v


def dual_linear_x(X, packed: PackedLayer, tinv=None, out_dtype: int = OUT_BF16, Y=None, ws=None, Xq_out=None,
                  sx_out=None, dbg_P=None, stream=None):
    """twq_dual_linear_x: the whole hot path from raw activations (one launch for M <= 64 where the plan fits)."""
    M = X.shape[0]
    N, K, r, G = packed.N, packed.K, packed.r, packed.G
    assert X.dtype == torch.bfloat16 and X.stride(1) == 1 and X.shape[1] == K
    if Y is None:
        Y = torch.empty((M, N), dtype=_OUT_TORCH.get(out_dtype, torch.bfloat16), device=X.device)
    need = workspace_bytes_x(M, N, K, r, G)
    if need and ws is None:
        ws = _cached_workspace(need, X.device, stream)
    code = load_library().twq_dual_linear_x(_ptr(X), X.stride(0), _ptr(tinv), _ptr(packed.blob), M, N, K, r, G,
                                            _ptr(Y), out_dtype, Y.stride(0), _ptr(ws), 0 if ws is None else ws.numel(),
                                            _ptr(Xq_out), _ptr(sx_out), _ptr(dbg_P), _stream(stream))
    _check(code, "twq_dual_linear_x")
    return Y


# ---- the paper's 4-bit low-rank branch (include/twq.h: twq_*_q4lr) ----
def lowrank_group(r: int) -> int:
    """Group of the re-quantized H along r (include/twq.h): r for r <= 128, else 128."""
    return r if r <= 128 else 128


def pack_weights_q4lr(Rq, sw, Uq, su, Vq, sv, G: int, stream=None) -> PackedLayer:
    """twq_pack_weights_q4lr.  Rq int8 [N,K], sw fp16 [N,K/G], Uq int8 [r,K], su fp16 [r,K/G], Vq int8 [N,r],
    sv fp16 [N,r/gr] (device, contiguous)."""
    N, K = Rq.shape
    r = int(Uq.shape[0])
    nbytes = int(load_library().twq_packed_bytes_q4lr(N, K, r, G))
    if nbytes == 0:
        raise TwqError(1, "twq_packed_bytes_q4lr")
    for t, dt in ((Rq, torch.int8), (Uq, torch.int8), (Vq, torch.int8), (sw, torch.float16), (su, torch.float16), (sv, torch.float16)):
        assert t.dtype == dt and t.is_contiguous()
    assert tuple(Uq.shape) == (r, K) and tuple(su.shape) == (r, K // G) and tuple(Vq.shape) == (N, r)
    assert tuple(sv.shape) == (N, r // lowrank_group(r))
    blob = torch.empty(nbytes, dtype=torch.uint8, device=Rq.device)
    code = load_library().twq_pack_weights_q4lr(_ptr(Rq), _ptr(sw), _ptr(Uq), _ptr(su), _ptr(Vq), _ptr(sv), N, K, r, G,
                                                _ptr(blob), nbytes, _stream(stream))
    _check(code, "twq_pack_weights_q4lr")
    return PackedLayer(blob, N, K, r, G)


def dual_linear_q4lr_x(X, packed: PackedLayer, tinv=None, out_dtype: int = OUT_BF16, Y=None, Xq_out=None, sx_out=None,
                       dbg_P=None, dbg_H=None, dbg_QH=None, dbg_sH=None, stream=None):
    """twq_dual_linear_q4lr_x: quantizer, 4-bit residual, 4-bit two-stage low-rank branch with on-the-fly
    re-quantization of H, one epilogue; one launch per slab of at most 64 tokens.  `packed` from pack_weights_q4lr."""
    M = X.shape[0]
    N, K, r, G = packed.N, packed.K, packed.r, packed.G
    assert X.dtype == torch.bfloat16 and X.stride(1) == 1 and X.shape[1] == K
    if Y is None:
        Y = torch.empty((M, N), dtype=_OUT_TORCH.get(out_dtype, torch.bfloat16), device=X.device)
    code = load_library().twq_dual_linear_q4lr_x(_ptr(X), X.stride(0), _ptr(tinv), _ptr(packed.blob), M, N, K, r, G,
                                                 _ptr(Y), out_dtype, Y.stride(0), _ptr(Xq_out), _ptr(sx_out), _ptr(dbg_P),
                                                 _ptr(dbg_H), _ptr(dbg_QH), _ptr(dbg_sH), _stream(stream))
    _check(code, "twq_dual_linear_q4lr_x")
    return Y


def algorithmic_bytes_q4lr(M: int, N: int, K: int, r: int, G: int, out_bytes: int = 2) -> int:
    """Bytes one twq_dual_linear_q4lr_x call must move: packed residual and its scales, both 4-bit factors and their
    scales (4 bits per element + one FP16 scale per group), X read once, Y written once."""
    ng, gr = K // G, lowrank_group(r)
    w = N * K // 2 + 2 * N * ng + r * K // 2 + 2 * r * ng + N * r // 2 + 2 * N * (r // gr)
    return w + 2 * M * K + out_bytes * M * N


# ---- accounting used by bench.py (PAPER.md L86 byte arithmetic) ----
def algorithmic_bytes(M: int, N: int, K: int, r: int, G: int, with_quantizer: bool = False, out_bytes: int = 2) -> int:
    """Bytes the method must move for one twq_dual_linear call: packed residual, its scales (fp16 in the
    interchange format), both factors, X, Xq, sx, Y.  with_quantizer adds the quantizer's own X read and
    Xq/sx write."""
    ng = K // G
    w = N * K // 2 + 2 * N * ng + 2 * K * r + 2 * r * N
    a = (2 * M * K if r > 0 else 0) + M * K // 2 + 4 * M * ng + out_bytes * M * N
    q = 2 * M * K + M * K // 2 + 4 * M * ng if with_quantizer else 0
    return w + a + q


def algorithmic_bytes_x(M: int, N: int, K: int, r: int, G: int, out_bytes: int = 2) -> int:
    """Bytes one ONE-LAUNCH twq_dual_linear_x call (M <= 64) must move: the weights as in algorithmic_bytes, X read
    once, Y written once (codes and scales never leave the chip)."""
    ng = K // G
    return N * K // 2 + 2 * N * ng + 2 * K * r + 2 * r * N + 2 * M * K + out_bytes * M * N


def flops(M: int, N: int, K: int, r: int):
    """(int8 residual ops, 16-bit low-rank flops) of one call."""
    return 2 * M * K * N, 2 * M * r * (K + N)
