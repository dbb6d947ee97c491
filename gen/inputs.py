"""Seeded synthetic inputs for the TwinQuant dual-component linear layer.

This module serves BOTH the CPU oracle (`oracle/`) and the CUDA path
(`paper_2606_01556_b200/`).  It holds none of the method's arithmetic: it only
draws random tensors with the shapes and statistics BASELINE.json's configs
name and casts them to the storage types (BF16 / FP16 / int8 codes).  No
quantizer, no packer, no GEMM lives here.

Recipe:
  * draws come from numpy.random.Generator(PCG64(seed)) in the fixed order
    X, outlier channels, residual codes, sw, L1, L2 (, X_cal for tinv);
  * everything is drawn in float64, cast to float32, then rounded to the
    storage type with round-to-nearest-even on the host;
  * the paper measures on LLaMA3/Qwen3 checkpoints with WikiText2 calibration
    (PAPER.md L187); those are not available, the draws below stand in for
    them: outlier-rich activations, 4-bit residual codes
    with FP16 group scales (L193), FP16 low-rank factors (L86, L177).
"""
from __future__ import annotations

import dataclasses
import numpy as np


# --------------------------------------------------------------------------
# storage-type casts (format conversion only, no method arithmetic)
# --------------------------------------------------------------------------
def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> BF16 bit pattern (uint16), round-to-nearest-even."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32).astype(np.uint64)
    rounding = ((u >> 16) & 1) + 0x7FFF
    out = ((u + rounding) >> 16).astype(np.uint16)
    # NaN stays NaN (generators never make one, but keep the cast total)
    nan = np.isnan(x)
    if nan.any():
        out = np.where(nan, np.uint16(0x7FC0), out)
    return out


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """BF16 bit pattern (uint16) -> float32, exact."""
    b = np.ascontiguousarray(b, dtype=np.uint16)
    return (b.astype(np.uint32) << 16).view(np.float32)


# --------------------------------------------------------------------------
# one layer's worth of inputs
# --------------------------------------------------------------------------
@dataclasses.dataclass
class LayerInputs:
    M: int
    K: int
    N: int
    r: int
    G: int
    X: np.ndarray        # uint16 [M,K]  BF16 bit patterns, row-major
    Rq: np.ndarray       # int8   [N,K]  residual 4-bit codes in [-8,7]
    sw: np.ndarray       # float16 [N,K/G] residual group scales
    L1: np.ndarray       # float16 [K,r]
    L2: np.ndarray       # float16 [r,N]
    tinv: np.ndarray | None = None   # float32 [K] diag transform (1/lambda) or None

    @property
    def ng(self) -> int:
        return self.K // self.G


def make_layer(M: int, K: int, N: int, r: int, G: int, *, seed: int,
               x_dist: str = "student_t", outlier_frac: float = 0.01,
               outlier_scale: float = 30.0, n_outlier: int | None = None,
               lr_sigma: float = 0.02, with_tinv: bool = False) -> LayerInputs:
    """Draw one layer.

    x_dist = "normal"    : X ~ N(0,1)                       (config 1)
             "student_t" : X iid Student-t(nu=3)            (configs 2-5)
    n_outlier channels (default floor(outlier_frac*K)) are multiplied by
    outlier_scale before the BF16 cast.
    """
    assert K % G == 0
    rng = np.random.Generator(np.random.PCG64(seed))
    if x_dist == "normal":
        X = rng.standard_normal((M, K))
    elif x_dist == "student_t":
        X = rng.standard_t(3.0, size=(M, K))
    else:
        raise ValueError(x_dist)
    n_out = int(np.floor(outlier_frac * K)) if n_outlier is None else n_outlier
    out_idx = rng.choice(K, size=n_out, replace=False) if n_out > 0 else np.zeros(0, np.int64)
    X[:, out_idx] *= outlier_scale
    Xb = f32_to_bf16_bits(X.astype(np.float32))

    Rq = rng.integers(-8, 8, size=(N, K), dtype=np.int8)          # uniform on [-8,7]
    sw = rng.uniform(0.005, 0.02, size=(N, K // G)).astype(np.float32).astype(np.float16)
    L1 = (rng.standard_normal((K, r)) * lr_sigma).astype(np.float32).astype(np.float16)
    L2 = (rng.standard_normal((r, N)) * lr_sigma).astype(np.float32).astype(np.float16)

    tinv = None
    if with_tinv:
        # tinv[k] = 1/sqrt(max_m |Xcal[m,k]|) from a separate
        # 512-token draw with the same outlier channels (alpha=0.5,
        # weight term dropped); floored at 1e-5 before inversion.  A synthetic choice.
        if x_dist == "normal":
            Xc = rng.standard_normal((512, K))
        else:
            Xc = rng.standard_t(3.0, size=(512, K))
        Xc[:, out_idx] *= outlier_scale
        amax = np.maximum(np.abs(Xc).max(axis=0), 1e-5)
        tinv = (1.0 / np.sqrt(amax)).astype(np.float32)
    return LayerInputs(M, K, N, r, G, Xb, Rq, sw, L1, L2, tinv)


def make_q4_lowrank(K: int, N: int, r: int, G: int, *, seed: int):
    """4-bit low-rank factors for the paper's own branch: codes uniform on [-8,7]
    with FP16 group scales, like the residual.  U codes [r,K] with scales [r,K/G] (groups along K); V codes [N,r] with
    scales [N,r/Gr], Gr = r for r <= 128 else 128 (groups along r).  Scale ranges are chosen so that the dequantized
    factors have about the N(0, 0.02) magnitude of the FP16 factors of configs 2-5 (code std 4.6 x 0.0043).
    Draw order: U codes, su, V codes, sv.  No method arithmetic."""
    rng = np.random.Generator(np.random.PCG64(seed))
    Gr = r if r <= 128 else 128
    Uq = rng.integers(-8, 8, size=(r, K), dtype=np.int8)
    su = rng.uniform(0.003, 0.006, size=(r, K // G)).astype(np.float32).astype(np.float16)
    Vq = rng.integers(-8, 8, size=(N, r), dtype=np.int8)
    sv = rng.uniform(0.003, 0.006, size=(N, r // Gr)).astype(np.float32).astype(np.float16)
    return Uq, su, Vq, sv


# --------------------------------------------------------------------------
# BASELINE.json configs
# --------------------------------------------------------------------------
def config1_tiny(with_tinv: bool = False) -> LayerInputs:
    """configs[0]: M=8, K=256, N=512, r=16, G=64, X~N(0,1), 4 outlier channels x20,
    L ~ N(0,0.05), seed 0."""
    return make_layer(8, 256, 512, 16, 64, seed=0, x_dist="normal", n_outlier=4,
                      outlier_scale=20.0, lr_sigma=0.05, with_tinv=with_tinv)


def config2_qproj(M: int, with_tinv: bool = False, r: int = 128) -> LayerInputs:
    """configs[1]: LLaMA3-8B q_proj, K=N=4096, r=128, G=128, M in {1,16,128}."""
    return make_layer(M, 4096, 4096, r, 128, seed=1, with_tinv=with_tinv)


def config3_mlp(which: str, M: int = 2048, r: int = 128, with_tinv: bool = False) -> LayerInputs:
    """configs[2]: LLaMA3-8B MLP at prefill; which in {"gate_up","down"}."""
    K, N = (4096, 14336) if which == "gate_up" else (14336, 4096)
    return make_layer(M, K, N, r, 128, seed=2, with_tinv=with_tinv)


def config4_qwen(which: str, M: int, r: int = 256, with_tinv: bool = False) -> LayerInputs:
    """configs[3]: Qwen3-32B-shaped; which in {"attn","gate_up","down"}."""
    K, N = {"attn": (5120, 5120), "gate_up": (5120, 25600), "down": (25600, 5120)}[which]
    return make_layer(M, K, N, r, 128, seed=3, with_tinv=with_tinv)


LLAMA70B_SHAPES = {"q": (8192, 8192), "o": (8192, 8192), "k": (8192, 1024), "v": (8192, 1024),
                   "gate_up": (8192, 28672), "down": (28672, 8192)}


def config5_llama70b(which: str, M: int, r: int = 256, with_tinv: bool = False) -> LayerInputs:
    """configs[4]: LLaMA3-70B decoder-block linear set."""
    K, N = LLAMA70B_SHAPES[which]
    return make_layer(M, K, N, r, 128, seed=4, with_tinv=with_tinv)
