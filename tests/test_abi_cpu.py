"""CPU-side checks of the C-ABI library: it builds for sm_100a, loads, exports every symbol that
include/twq.h declares, and validates arguments before touching CUDA (no compute without a GPU)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    import paper_2606_01556_b200 as twq
    return twq.load_library()


def test_header_symbols_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "twq.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(twq_[a-z0-9_]+)\s*\(", hdr))
    assert {"twq_quantize_act", "twq_pack_weights", "twq_dual_linear", "twq_packed_bytes", "twq_dual_linear_x",
            "twq_workspace_bytes", "twq_workspace_bytes_x", "twq_status_string", "twq_last_launch_count",
            "twq_packed_bytes_q4lr", "twq_pack_weights_q4lr", "twq_dual_linear_q4lr_x"} <= names
    for n in names:
        assert getattr(lib, n) is not None, n
    from paper_2606_01556_b200.binding import EXPORTS
    assert set(EXPORTS) == names


def test_status_strings(lib):
    assert lib.twq_status_string(0) == b"TWQ_OK"
    assert lib.twq_status_string(1) == b"TWQ_ERR_INVALID_ARG"
    assert lib.twq_status_string(99) == b"TWQ_ERR_UNKNOWN"


def test_packed_bytes_accounts_for_every_section(lib):
    import paper_2606_01556_b200 as twq
    N, K, r, G = 4096, 4096, 128, 128
    b = twq.packed_bytes(N, K, r, G)
    sections = [N * K // 2, (K // G) * N * 2, r * K * 2, r * K * 2, N * r * 2]   # R4, FP16 scales, L1T, L1 slabs, L2T
    assert b == sum((s + 255) & ~255 for s in sections)
    # 4-bit residual dominates: PAPER.md L86 ratio (2 r (m+n)) / (m n / 2) at r = 128 is 25 %
    assert abs((r * K * 2 + N * r * 2) / (N * K // 2) - 0.25) < 1e-12
    assert twq.packed_bytes(N, K, 0, G) == sections[0] + sections[1]
    for bad in [(4096, 4096, 128, 96), (4096, 4000, 128, 128), (4090, 4096, 128, 128), (4096, 4096, 8, 128),
                (4096, 4096, 272, 128), (4096, 64, 0, 128)]:
        assert twq.packed_bytes(*bad) == 0, bad


def test_algorithmic_bytes_pinned_to_paper_L86():
    """bench.py's byte accounting (binding.algorithmic_bytes) against the two storage ratios PAPER.md L86
    prints (tests/golden/paper_L86_storage_ratios.txt): the FP16 low-rank bytes are what the function adds when r goes
    from 0 to r, and the 4-bit residual bytes are what remains of the r = 0 weights once the FP16 group scales are taken
    out.  Also the activation-side terms, one by one (differences in M / out_bytes / with_quantizer)."""
    from paper_2606_01556_b200.binding import algorithmic_bytes as ab
    G = 128
    with open(os.path.join(ROOT, "tests", "golden", "paper_L86_storage_ratios.txt")) as f:
        rows = [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 2
    for m, n, r, pct in rows:
        K, N, r, pct = int(m), int(n), int(r), float(pct)
        # weight-side bytes = the M -> 0 limit: take two M values and extrapolate linearly
        w_r = 2 * ab(1, N, K, r, G) - ab(2, N, K, r, G)
        w_0 = 2 * ab(1, N, K, 0, G) - ab(2, N, K, 0, G)
        lowrank = w_r - w_0
        residual = w_0 - 2 * N * (K // G)                       # FP16 scales, one per group and channel (L193)
        assert residual == N * K // 2
        assert abs(100.0 * lowrank / residual - pct) < 1e-9
    # per-token terms at q_proj: X (bf16, only when r > 0), Xq (4 bit), sx (fp32 per group), Y
    N = K = 4096
    per_tok = ab(2, N, K, 128, G) - ab(1, N, K, 128, G)
    assert per_tok == 2 * K + K // 2 + 4 * (K // G) + 2 * N
    assert ab(2, N, K, 0, G) - ab(1, N, K, 0, G) == K // 2 + 4 * (K // G) + 2 * N
    assert ab(1, N, K, 128, G, out_bytes=4) - ab(1, N, K, 128, G) == 2 * N
    assert ab(3, N, K, 128, G, with_quantizer=True) - ab(3, N, K, 128, G) == 3 * (2 * K + K // 2 + 4 * (K // G))


def test_testing_hooks_are_separate_from_the_product_abi(lib):
    """include/twq_testing.h: planner overrides and plan read-back; exported, but not declared in twq.h."""
    import paper_2606_01556_b200 as twq
    from paper_2606_01556_b200.binding import TESTING_EXPORTS
    hdr = open(os.path.join(ROOT, "include", "twq_testing.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    assert set(re.findall(r"\b(twq_testing_[a-z0-9_]+)\s*\(", hdr)) == set(TESTING_EXPORTS)
    for n in TESTING_EXPORTS:
        assert getattr(lib, n) is not None
    assert "twq_testing" not in open(os.path.join(ROOT, "include", "twq.h")).read()
    # no environment variable reaches the planner
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2606_01556_b200", "csrc")):
        for f in files:
            if f.endswith((".cu", ".cuh", ".h")):
                assert "getenv" not in open(os.path.join(dirpath, f)).read(), f
    try:
        base = twq.testing_describe_plan(300, 1024, 1024, 128, 128)
        assert base["kernel"] == "tcgen05" and base["splits"] > 1
        twq.testing_set_plan_flags(twq.PLAN_NO_SPLIT)
        forced = twq.testing_describe_plan(300, 1024, 1024, 128, 128)
        assert forced["splits"] == 1 and forced["pair"] == 1
        assert twq.testing_describe_plan(16, 4096, 4096, 128, 128)["kernel"] == "decode"
        twq.testing_set_plan_flags(twq.PLAN_NO_DECODE)
        assert twq.testing_describe_plan(16, 4096, 4096, 128, 128)["kernel"] == "tcgen05"
    finally:
        twq.testing_set_plan_flags(0)


def test_workspace_rule(lib):
    import paper_2606_01556_b200 as twq
    assert twq.workspace_bytes(2048, 14336, 4096, 128, 128) == 0      # prefill: tiles fill the GPU, no split
    assert twq.workspace_bytes(1, 4096, 4096, 128, 128) == 0           # decode kernel (M <= 16): no scratch
    assert twq.workspace_bytes(16, 4096, 4096, 128, 128) == 0
    assert twq.workspace_bytes(64, 4096, 4096, 128, 128) == 0          # small-batch kernel up to M = 64
    w = twq.workspace_bytes(80, 4096, 4096, 128, 128)                  # few tiles: split-K partials + counters
    assert w > 0 and (w - 256) % (80 * 4096 * 4) == 0
    assert twq.workspace_bytes(0, 4096, 4096, 128, 128) == 0           # invalid shape


def test_argument_validation_happens_before_cuda(lib):
    """Invalid arguments are rejected with TWQ_ERR_INVALID_ARG even though this box has no GPU."""
    buf = ctypes.create_string_buffer(1 << 16)
    base = (ctypes.addressof(buf) + 255) & ~255
    p = ctypes.c_void_p(base)
    p_unaligned = ctypes.c_void_p(base + 2)
    # quantizer: null pointers, bad G, bad ldx, misaligned
    assert lib.twq_quantize_act(None, 1, 256, 256, None, 128, p, p, None) == 1
    assert lib.twq_quantize_act(p, 1, 256, 256, None, 100, p, p, None) == 1
    assert lib.twq_quantize_act(p, 1, 256, 128, None, 128, p, p, None) == 1
    assert lib.twq_quantize_act(p_unaligned, 1, 256, 256, None, 128, p, p, None) == 1
    assert lib.twq_quantize_act(p, 0, 256, 256, None, 128, p, p, None) == 1
    # packer: blob too small, missing L1 with r > 0
    assert lib.twq_pack_weights(p, p, p, p, 512, 256, 16, 64, p, 16, None) == 1
    assert lib.twq_pack_weights(p, p, None, p, 512, 256, 16, 64, p, 1 << 30, None) == 1
    # fused layer: X missing with r > 0, bad out dtype, ldy < N, workspace missing for a split shape
    assert lib.twq_dual_linear(None, 256, p, p, p, 8, 512, 256, 16, 64, p, 0, 512, None, 0, None, None) == 1
    assert lib.twq_dual_linear(p, 256, p, p, p, 8, 512, 256, 16, 64, p, 7, 512, None, 0, None, None) == 1
    assert lib.twq_dual_linear(p, 256, p, p, p, 8, 512, 256, 16, 64, p, 0, 256, None, 0, None, None) == 1
    assert lib.twq_dual_linear(p, 256, p, p, p, 72, 512, 256, 16, 64, p, 0, 512, None, 0, None, None) == 3
    # valid arguments but no sm_100 device here -> UNSUPPORTED or CUDA error, never a crash, never OK
    import torch
    if not torch.cuda.is_available():
        rc = lib.twq_quantize_act(p, 1, 256, 256, None, 128, p, p, None)
        assert rc in (2, 4)


def test_product_package_does_not_import_oracle():
    """The product path shares nothing with oracle/ (tier rule): no import, no include."""
    pkg = os.path.join(ROOT, "paper_2606_01556_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                for pat in (r"^\s*(from|import)\s+oracle", r"#include\s+[<\"].*oracle", r"twq_oracle", r"oracle[/.]"):
                    assert not re.search(pat, src, flags=re.M), (f, pat)
