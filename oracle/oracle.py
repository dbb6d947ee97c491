"""ctypes front-end of the CPU oracle (oracle/twq_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  The product package
paper_2606_01556_b200 never imports this module and shares no code with it.

Every function is a thin marshalling layer over the C routine of the same
name; the arithmetic lives in twq_oracle.c, each routine citing PAPER.md.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "twq_oracle.c")
_LIB = os.path.join(_HERE, "libtwq_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -ffp-contract=off (no -ffast-math): the quantizer's FP32 op order is the spec."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.twq_oracle_num_threads.restype = ctypes.c_int
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct)) if a is not None else None


def num_threads() -> int:
    return int(_load().twq_oracle_num_threads())


def quantize_act(X_bf16: np.ndarray, G: int, tinv: np.ndarray | None = None):
    """Steps 1-3 (Eq. 1).  X_bf16: uint16 [M,K] BF16 bits.
    Returns (q int8 [M,K] in [-7,7], sx float32 [M,K/G])."""
    X = np.ascontiguousarray(X_bf16, dtype=np.uint16)
    M, K = X.shape
    assert K % G == 0
    q = np.empty((M, K), np.int8)
    sx = np.empty((M, K // G), np.float32)
    if tinv is not None:
        tinv = np.ascontiguousarray(tinv, dtype=np.float32)
        assert tinv.shape == (K,)
    _load().twq_oracle_quantize_act(_p(X, ctypes.c_uint16), M, K, K, _p(tinv, ctypes.c_float), G,
                                    _p(q, ctypes.c_int8), _p(sx, ctypes.c_float))
    return q, sx


def pack_nibbles(q: np.ndarray) -> np.ndarray:
    """Step 4: int8 codes [rows,K] -> uint8 [rows,K/2], low nibble = even k (reading R10)."""
    q = np.ascontiguousarray(q, dtype=np.int8)
    rows, K = q.shape
    assert K % 2 == 0
    out = np.empty((rows, K // 2), np.uint8)
    _load().twq_oracle_pack_nibbles(_p(q, ctypes.c_int8), ctypes.c_int64(rows), K, _p(out, ctypes.c_uint8))
    return out


def unpack_nibbles(p: np.ndarray) -> np.ndarray:
    p = np.ascontiguousarray(p, dtype=np.uint8)
    rows, K2 = p.shape
    q = np.empty((rows, 2 * K2), np.int8)
    _load().twq_oracle_unpack_nibbles(_p(p, ctypes.c_uint8), ctypes.c_int64(rows), 2 * K2, _p(q, ctypes.c_int8))
    return q


def residual_P(Xq: np.ndarray, R4: np.ndarray, G: int, rows=None) -> np.ndarray:
    """Step 5 (Eq. 2): P[m,g,n] exact int64, shape [nrows, K/G, N]."""
    Xq = np.ascontiguousarray(Xq, dtype=np.uint8)
    R4 = np.ascontiguousarray(R4, dtype=np.uint8)
    M, K2 = Xq.shape
    N = R4.shape[0]
    K = 2 * K2
    assert R4.shape[1] == K2 and K % G == 0
    rows_a = None if rows is None else np.ascontiguousarray(rows, dtype=np.int32)
    nrows = M if rows is None else len(rows_a)
    P = np.empty((nrows, K // G, N), np.int64)
    _load().twq_oracle_residual_P(_p(Xq, ctypes.c_uint8), _p(R4, ctypes.c_uint8), M, N, K, G,
                                  _p(rows_a, ctypes.c_int32), nrows, _p(P, ctypes.c_int64))
    return P


def forward_from_quantized(X_bf16, Xq, sx, R4, sw, L1, L2, G: int, rows=None, want_P: bool = False):
    """Steps 5-8 on given quantizer outputs.  Returns Y float64 [nrows,N] (and P int64 [nrows,ng,N])."""
    X = np.ascontiguousarray(X_bf16, dtype=np.uint16)
    Xq = np.ascontiguousarray(Xq, dtype=np.uint8)
    sx = np.ascontiguousarray(sx, dtype=np.float32)
    R4 = np.ascontiguousarray(R4, dtype=np.uint8)
    sw = np.ascontiguousarray(sw, dtype=np.float16)
    M, K = X.shape
    N = R4.shape[0]
    ng = K // G
    assert Xq.shape == (M, K // 2) and sx.shape == (M, ng) and R4.shape == (N, K // 2) and sw.shape == (N, ng)
    if L1 is None or L1.shape[1] == 0:
        r = 0
        L1 = np.zeros((K, 0), np.float16)
        L2 = np.zeros((0, N), np.float16)
    else:
        r = L1.shape[1]
    L1 = np.ascontiguousarray(L1, dtype=np.float16)
    L2 = np.ascontiguousarray(L2, dtype=np.float16)
    assert L1.shape == (K, r) and L2.shape == (r, N)
    rows_a = None if rows is None else np.ascontiguousarray(rows, dtype=np.int32)
    nrows = M if rows is None else len(rows_a)
    Y = np.empty((nrows, N), np.float64)
    P = np.empty((nrows, ng, N), np.int64) if want_P else None
    _load().twq_oracle_forward(_p(X, ctypes.c_uint16), K, _p(Xq, ctypes.c_uint8), _p(sx, ctypes.c_float),
                               _p(R4, ctypes.c_uint8), _p(sw.view(np.uint16), ctypes.c_uint16),
                               _p(L1.view(np.uint16), ctypes.c_uint16), _p(L2.view(np.uint16), ctypes.c_uint16),
                               M, N, K, r, G, _p(rows_a, ctypes.c_int32), nrows,
                               _p(Y, ctypes.c_double), _p(P, ctypes.c_int64))
    return (Y, P) if want_P else Y


def forward(X_bf16, Rq, sw, L1, L2, G: int, tinv=None, rows=None, want_P: bool = False):
    """The whole hot path, steps 1-8: quantize X (with optional diag transform), pack, run
    both branches, merge.  Rq: int8 codes [N,K] in [-8,7].
    Returns dict(q, Xq, sx, Y [, P])."""
    q, sx = quantize_act(X_bf16, G, tinv)
    Xq = pack_nibbles(q)
    R4 = pack_nibbles(Rq)
    res = forward_from_quantized(X_bf16, Xq, sx, R4, sw, L1, L2, G, rows=rows, want_P=want_P)
    out = dict(q=q, Xq=Xq, sx=sx)
    if want_P:
        out["Y"], out["P"] = res
    else:
        out["Y"] = res
    return out


def lowrank_group(r: int) -> int:
    """Group size of the re-quantized intermediate H along r (reading R18): r for r <= 128, else 128."""
    return r if r <= 128 else 128


def forward_q4lr_from_quantized(Xq, sx, R4, sw, U4, su, V4, sv, G: int, rows=None, want_H: bool = False):
    """NEXT-1, steps on given quantizer outputs: both low-rank factors 4-bit, H re-quantized on the
    fly.  U4 [r,K/2], su fp16 [r,K/G], V4 [N,r/2], sv fp16 [N,r/Gr].  Returns Y [nrows,N] (and dict(H, QH, sH))."""
    Xq = np.ascontiguousarray(Xq, dtype=np.uint8)
    sx = np.ascontiguousarray(sx, dtype=np.float32)
    R4 = np.ascontiguousarray(R4, dtype=np.uint8)
    sw = np.ascontiguousarray(sw, dtype=np.float16)
    U4 = np.ascontiguousarray(U4, dtype=np.uint8)
    su = np.ascontiguousarray(su, dtype=np.float16)
    V4 = np.ascontiguousarray(V4, dtype=np.uint8)
    sv = np.ascontiguousarray(sv, dtype=np.float16)
    M, K2 = Xq.shape
    K, N, r = 2 * K2, R4.shape[0], U4.shape[0]
    ng, Gr = K // G, lowrank_group(U4.shape[0])
    assert r % Gr == 0 and U4.shape == (r, K2) and su.shape == (r, ng) and V4.shape == (N, r // 2) and sv.shape == (N, r // Gr)
    rows_a = None if rows is None else np.ascontiguousarray(rows, dtype=np.int32)
    nrows = M if rows is None else len(rows_a)
    Y = np.empty((nrows, N), np.float64)
    H = np.empty((nrows, r), np.float64) if want_H else None
    QH = np.empty((nrows, r), np.int8) if want_H else None
    sH = np.empty((nrows, r // Gr), np.float32) if want_H else None
    _load().twq_oracle_forward_q4lr(_p(Xq, ctypes.c_uint8), _p(sx, ctypes.c_float), _p(R4, ctypes.c_uint8),
                                    _p(sw.view(np.uint16), ctypes.c_uint16), _p(U4, ctypes.c_uint8),
                                    _p(su.view(np.uint16), ctypes.c_uint16), _p(V4, ctypes.c_uint8),
                                    _p(sv.view(np.uint16), ctypes.c_uint16), M, N, K, r, G, Gr,
                                    _p(rows_a, ctypes.c_int32), nrows, _p(Y, ctypes.c_double), _p(H, ctypes.c_double),
                                    _p(QH, ctypes.c_int8), _p(sH, ctypes.c_float))
    return (Y, dict(H=H, QH=QH, sH=sH)) if want_H else Y


def forward_q4lr(X_bf16, Rq, sw, Uq, su, Vq, sv, G: int, tinv=None, rows=None, want_H: bool = False):
    """NEXT-1, the whole path: quantize X, pack every code tensor, run both 4-bit branches, merge.
    Uq int8 [r,K], Vq int8 [N,r] codes in [-8,7].  Returns dict(q, Xq, sx, Y [, H, QH, sH])."""
    q, sx = quantize_act(X_bf16, G, tinv)
    Xq = pack_nibbles(q)
    res = forward_q4lr_from_quantized(Xq, sx, pack_nibbles(Rq), sw, pack_nibbles(Uq), su, pack_nibbles(Vq), sv, G,
                                      rows=rows, want_H=want_H)
    out = dict(q=q, Xq=Xq, sx=sx)
    if want_H:
        out["Y"] = res[0]
        out.update(res[1])
    else:
        out["Y"] = res
    return out


def round_bf16(Y: np.ndarray) -> np.ndarray:
    """FP64 -> BF16 bits with one round-to-nearest-even (reading R11)."""
    Y = np.ascontiguousarray(Y, dtype=np.float64)
    out = np.empty(Y.shape, np.uint16)
    _load().twq_oracle_round_bf16(_p(Y, ctypes.c_double), ctypes.c_int64(Y.size), _p(out, ctypes.c_uint16))
    return out


# ---- byte accounting of the method -- used to pin bench.py's formulas ----
def lowrank_fp16_bytes(m: int, n: int, r: int) -> int:
    """FP16 low-rank factors U[m,r], V[r,n]: 2 bytes each."""
    return 2 * r * (m + n)


def residual_4bit_bytes(m: int, n: int) -> int:
    """4-bit residual, scales not counted (PAPER.md L86 compares against 'the 4-bit residual')."""
    return m * n // 2
