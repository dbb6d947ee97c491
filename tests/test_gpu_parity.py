"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Bars (BASELINE.json north_star):
  * quantizer codes Xq and scales sx: bit-exact;
  * integer group accumulators P (dbg_P, taken from the same tcgen05 path): bit-exact;
  * FP32 output: max|Y32 - Yref| / max|Yref| <= 2e-3 against the FP64 oracle (reading R13 (i));
  * BF16 output == round-to-nearest-even of the kernel's FP32 output, bit for bit (R13 (ii)).
"""
import numpy as np
import pytest

from gen import inputs as gen

pytestmark = pytest.mark.gpu

TOL = 2e-3


@pytest.fixture(scope="module")
def twq():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a GPU")
    import paper_2606_01556_b200 as t
    t.load_library()
    return t


def _dev(a, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t if dtype is None else t.view(dtype)


def _upload(twq, L):
    import torch
    X = _dev(L.X.view(np.int16), torch.bfloat16)
    packed = twq.pack_weights(_dev(L.Rq), _dev(L.sw), _dev(L.L1) if L.r else None, _dev(L.L2) if L.r else None, L.G)
    tinv = _dev(L.tinv) if L.tinv is not None else None
    return X, packed, tinv


def _bits(t):
    import torch
    return t.view(torch.int16).cpu().numpy().view(np.uint16)


def _check_layer(twq, oracle, L, rows=None, check_P=True):
    """Full pipeline on L; compare every output (or the given token rows) with the oracle."""
    import torch
    X, packed, tinv = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, L.G, tinv)
    dbg = torch.zeros((L.M, L.ng, L.N), dtype=torch.int32, device="cuda") if check_P else None
    Y32 = twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32, dbg_P=dbg)
    Y16 = twq.dual_linear(X, Xq, sx, packed, twq.OUT_BF16)
    torch.cuda.synchronize()
    ref = oracle.forward(L.X, L.Rq, L.sw, L.L1 if L.r else None, L.L2 if L.r else None, L.G, tinv=L.tinv,
                         rows=rows, want_P=check_P)
    assert (Xq.cpu().numpy() == ref["Xq"]).all(), "codes"
    assert (sx.cpu().numpy() == ref["sx"]).all(), "scales"
    sel = slice(None) if rows is None else rows
    if check_P:
        assert (dbg.cpu().numpy()[sel].astype(np.int64) == ref["P"]).all(), "integer accumulators"
    y = Y32.cpu().numpy().astype(np.float64)[sel]
    err = np.abs(y - ref["Y"]).max() / np.abs(ref["Y"]).max()
    assert err <= TOL, err
    assert (_bits(Y16) == _bits(Y32.to(torch.bfloat16))).all(), "BF16 != rne(Y32)"
    return err


# ------------------------------------------------------------------------------ quantizer
@pytest.mark.parametrize("M,K,G,with_tinv", [(1, 128, 128, False), (3, 192, 64, True), (8, 256, 64, False),
                                             (37, 1024, 128, True), (130, 4096, 128, False)])
def test_quantizer_bit_exact(twq, oracle, M, K, G, with_tinv):
    import torch
    L = gen.make_layer(M, K, 16, 0, G, seed=100 + M, with_tinv=with_tinv)
    X = _dev(L.X.view(np.int16), torch.bfloat16)
    Xq, sx = twq.quantize_act(X, G, _dev(L.tinv) if with_tinv else None)
    q, sxr = oracle.quantize_act(L.X, G, L.tinv)
    assert (Xq.cpu().numpy() == oracle.pack_nibbles(q)).all()
    assert (sx.cpu().numpy() == sxr).all()


def test_quantizer_edges_zero_group_ties_and_row_stride(twq, oracle):
    import torch
    G, K = 64, 256
    x = np.zeros((4, K), np.float32)
    x[1, :16] = np.array([7, -7, 3, -3, .5, 1.5, 2.5, -.5, -1.5, -2.5, 6.5, .25, .75, -6.5, 1, 0]) * 4  # ties -> even
    x[2] = np.linspace(-1e-3, 1e30, K)            # huge dynamic range
    x[3, 64:128] = 1e-38                           # below the 2^-30 floor
    Xb = gen.f32_to_bf16_bits(x)
    pad = np.zeros((4, K + 64), np.uint16)         # ldx > K
    pad[:, :K] = Xb
    Xd = _dev(pad.view(np.int16), torch.bfloat16)[:, :K]
    assert Xd.stride(0) == K + 64
    Xq, sx = twq.quantize_act(Xd, G)
    q, sxr = oracle.quantize_act(Xb, G)
    assert (Xq.cpu().numpy() == oracle.pack_nibbles(q)).all()
    assert (sx.cpu().numpy() == sxr).all()
    assert (Xq.cpu().numpy()[0] == 0).all() and sx.cpu().numpy()[0, 0] == np.float32(2.0 ** -30) / np.float32(7)


# ------------------------------------------------------------------------------ fused layer, small
def test_config1_tiny(twq, oracle):
    _check_layer(twq, oracle, gen.config1_tiny())
    _check_layer(twq, oracle, gen.config1_tiny(with_tinv=True))


@pytest.mark.parametrize("M,K,N,r,G", [
    (1, 128, 16, 0, 128),        # smallest legal problem, one group, N tail inside one tile
    (5, 256, 144, 16, 64),       # ragged M, N = 128 + 16
    (17, 384, 400, 48, 128),     # TN = 32 tile with ragged tail, r not a multiple of 64
    (40, 512, 256, 128, 128),
    (70, 640, 128, 144, 64),     # r spans two 128-row blocks
    (130, 512, 384, 256, 128),   # two token tiles, ragged second
    (200, 1024, 272, 256, 128),
])
def test_ragged_shapes(twq, oracle, M, K, N, r, G):
    _check_layer(twq, oracle, gen.make_layer(M, K, N, r, G, seed=1000 + M, with_tinv=(M % 2 == 0)))


@pytest.mark.parametrize("M,K,N,r,G", [
    (1, 128, 16, 16, 128),       # one tile, one group, smallest rank
    (3, 192, 48, 16, 64),        # G = 64 (two packed words per thread), three groups
    (8, 2048, 528, 48, 128),     # r not a multiple of 32: half-empty last stage-2 step; N = 33 tiles
    (9, 1024, 272, 256, 128),    # two token tiles of the MMA (M > 8), rank 256: two j-tiles per warp
    (12, 640, 16, 0, 128),       # rank 0 in the decode kernel, fewer tiles than CTAs
    (16, 7168, 1040, 128, 128),  # long K: items with more groups than pipeline slots, several ring rounds
    (16, 512, 4112, 32, 64),     # many tiles per CTA, whole K in one part
])
def test_decode_kernel_shapes(twq, oracle, M, K, N, r, G):
    """M <= 16 takes the register-resident decode kernel (decode_kernel.cu); same bar as every other shape."""
    assert twq.workspace_bytes(M, N, K, r, G) == 0
    _check_layer(twq, oracle, gen.make_layer(M, K, N, r, G, seed=2000 + M + N, with_tinv=(M % 2 == 1)))


@pytest.mark.parametrize("M,K,N,r,G", [
    (256, 512, 512, 64, 64),      # CTA pairs with 64-wide groups
    (300, 1024, 1024, 128, 128),  # ragged last token tile: the odd CTA's half of the B rows is all padding
    (129, 256, 256, 16, 128),     # one live row in the second tile; smallest rank
    (640, 2048, 2304, 128, 128),  # several tiles per cluster and a change of token tile inside a cluster's list
    (640, 1024, 2304, 256, 128),  # rank 256: the stage-1 ring / H partial overlay the L2T tile too (plan.alias == 2),
                                  # with a new token tile's stage 1 following tiles that used L2T
    (300, 512, 1280, 256, 64),    # the same overlay with G = 64 and a ragged token tile
])
def test_fused_kernel_cta_pairs(twq, oracle, monkeypatch, M, K, N, r, G):
    """128-token tiles in an even cluster run as CTA pairs (cta_group::2, fused_kernel.cuh); same bar.
    Shapes this small would split K instead; the planner's testing switch sends them down the unsplit path."""
    monkeypatch.setenv("TWQ_DEBUG_NO_SPLIT", "1")
    assert twq.workspace_bytes(M, N, K, r, G) == 0
    rows = None if M * N * K <= 2 ** 29 else sorted(set(np.linspace(0, M - 1, 96).astype(int).tolist()))
    _check_layer(twq, oracle, gen.make_layer(M, K, N, r, G, seed=3000 + M, with_tinv=(M % 2 == 0)), rows=rows)


@pytest.mark.parametrize("pad", [0, 8, 2, 1])
@pytest.mark.parametrize("split,N", [(False, 1232), (False, 1200), (True, 1232)])
def test_fused_kernel_store_paths(twq, oracle, monkeypatch, pad, split, N):
    """Every store path of the fused kernel writes the same Y (fused_kernel.cuh, 'The store of a finished tile' in
    DESIGN.md 6.2): row pitch N + pad selects staged TMA tiles / 16-byte transposed stores (pad % 8 == 0), lane pairs
    (even pad) or element stores (odd pad); unsplit 128-token tiles (CTA pairs: 10 channel tiles) or the split-K
    fix-up.  Ragged last token tile and a last channel tile of 80 / 48 channels (the second half-tile store is
    clipped / skipped); columns beyond N must stay untouched."""
    import torch
    M, K, r, G = 300, 512, 64, 128
    if not split:
        monkeypatch.setenv("TWQ_DEBUG_NO_SPLIT", "1")
    L = gen.make_layer(M, K, N, r, G, seed=4100)
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, G)
    ref = oracle.forward(L.X, L.Rq, L.sw, L.L1, L.L2, G, want_P=False)["Y"]
    Y32 = twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32)
    assert np.abs(Y32.cpu().numpy().astype(np.float64) - ref).max() / np.abs(ref).max() <= TOL
    for od, dt in ((twq.OUT_FP32, torch.float32), (twq.OUT_BF16, torch.bfloat16), (twq.OUT_FP16, torch.float16)):
        buf = torch.full((M, N + pad), -77.0, dtype=dt, device="cuda")
        Y = buf[:, :N]
        twq.dual_linear(X, Xq, sx, packed, od, Y=Y)
        torch.cuda.synchronize()
        assert (_bits(Y.contiguous()) == _bits(Y32.to(dt))).all(), (od, pad)
        if pad:
            assert (buf[:, N:] == -77.0).all(), "wrote beyond N"


def test_rank0_is_plain_w4a4_and_zero_residual_is_lowrank(twq, oracle):
    """north_star special cases, on the GPU path."""
    import torch
    L = gen.make_layer(24, 512, 256, 0, 128, seed=31)
    _check_layer(twq, oracle, L)
    L = gen.make_layer(24, 512, 256, 64, 128, seed=32)
    L.Rq[:] = 0
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, L.G)
    Y = twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32).cpu().numpy().astype(np.float64)
    Xf = gen.bf16_bits_to_f32(L.X).astype(np.float64)
    ref = (Xf @ L.L1.astype(np.float64)) @ L.L2.astype(np.float64)      # FP64 BLAS, independent of the oracle
    assert np.abs(Y - ref).max() / np.abs(ref).max() <= TOL


def test_extreme_codes_hit_the_accumulator_bound(twq, oracle):
    """|P| = 7*8*G exactly and sign extension of -8."""
    import torch
    M, K, N, G = 4, 256, 128, 128
    x = np.full((M, K), -3.0, np.float32)          # every code = -7
    L = gen.make_layer(M, K, N, 0, G, seed=3)
    L.X = gen.f32_to_bf16_bits(x)
    L.Rq[:] = -8
    L.Rq[1::2] = 7
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, G)
    dbg = torch.zeros((M, K // G, N), dtype=torch.int32, device="cuda")
    twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32, dbg_P=dbg)
    P = dbg.cpu().numpy()
    assert (P[:, :, 0::2] == 56 * G).all() and (P[:, :, 1::2] == -49 * G).all()


def test_exactly_representable_output_is_bit_exact(twq, oracle):
    """Power-of-two scales and small integers: Y is exactly representable, so BF16 output must equal the oracle's."""
    import torch
    rng = np.random.default_rng(9)
    M, K, N, G = 16, 256, 128, 64
    L = gen.make_layer(M, K, N, 0, G, seed=4)
    # activations 7*2^p per group maximum -> sx = 2^p exactly; codes are small integers
    q = rng.integers(-2, 3, (M, K)).astype(np.float32)
    q[:, ::G] = 7
    L.X = gen.f32_to_bf16_bits(q * 0.5)                      # sx = 0.5
    L.Rq = rng.integers(-2, 3, (N, K), dtype=np.int8)
    L.sw = np.full((N, K // G), 2.0 ** -4, np.float16)
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, G)
    Y16 = twq.dual_linear(X, Xq, sx, packed, twq.OUT_BF16)
    ref = oracle.forward(L.X, L.Rq, L.sw, None, None, G)
    assert (sx.cpu().numpy() == 0.5).all()
    assert (_bits(Y16) == oracle.round_bf16(ref["Y"])).all()
    assert (ref["Y"] == gen.bf16_bits_to_f32(oracle.round_bf16(ref["Y"])).astype(np.float64)).all()  # truly exact


@pytest.mark.parametrize("M,K,N,r,G", [(1, 8192, 4096, 128, 128), (16, 8192, 2048, 256, 128), (5, 4096, 4096, 64, 64)])
def test_decode_kernel_stage1_over_all_clusters(twq, oracle, monkeypatch, M, K, N, r, G):
    """decode_kernel.cu with the K range of stage 1 split over the whole grid (DecodeParams.ncl_k > 1): cluster-level
    partials of H meet in the workspace behind a grid-wide barrier.  Forced on for shapes the oracle finishes quickly;
    the same workspace serves three calls in a row (the counter must come back to zero)."""
    import torch
    monkeypatch.setenv("TWQ_DEBUG_DECODE_GRIDK", "1")
    need = twq.workspace_bytes(M, N, K, r, G)
    assert need > 0
    L = gen.make_layer(M, K, N, r, G, seed=5200 + M)
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, G)
    ws = torch.zeros(need, dtype=torch.uint8, device="cuda")
    ref = oracle.forward(L.X, L.Rq, L.sw, L.L1, L.L2, G, want_P=False)["Y"]
    ys = [twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32, ws=ws) for _ in range(3)]
    torch.cuda.synchronize()
    for y in ys:
        assert np.abs(y.cpu().numpy().astype(np.float64) - ref).max() / np.abs(ref).max() <= TOL
        assert (y == ys[0]).all(), "not deterministic across calls"
    assert int(ws[:4].view(torch.int32).item()) == 0, "barrier counter not left at zero"
    monkeypatch.setenv("TWQ_DEBUG_DECODE_GRIDK", "0")
    assert twq.workspace_bytes(M, N, K, r, G) == 0
    y0 = twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32)
    assert np.abs(y0.cpu().numpy().astype(np.float64) - ref).max() / np.abs(ref).max() <= TOL


def test_decode_kernel_strides_fp16_output_no_workspace(twq, oracle):
    """M <= 16 runs the register-resident decode kernel: no scratch, padded Y rows untouched, repeatable."""
    import torch
    L = gen.make_layer(9, 512, 256, 32, 128, seed=41)
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, L.G)
    assert twq.workspace_bytes(L.M, L.N, L.K, L.r, L.G) == 0
    Ybig = torch.full((L.M, L.N + 64), 7.0, dtype=torch.float16, device="cuda")
    Yv = Ybig[:, :L.N]
    twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP16, Y=Yv)
    a = Yv.clone()
    twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP16, Y=Yv)
    assert torch.equal(a, Yv)
    assert (Ybig[:, L.N:] == 7.0).all()
    ref = oracle.forward(L.X, L.Rq, L.sw, L.L1, L.L2, L.G)["Y"]
    y = Yv.float().cpu().numpy().astype(np.float64)
    assert np.abs(y - ref).max() / np.abs(ref).max() <= TOL + 2.0 ** -11


def test_strides_fp16_output_and_workspace_reuse(twq, oracle):
    import torch
    L = gen.make_layer(24, 512, 256, 32, 128, seed=41)
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, L.G)
    need = twq.workspace_bytes(L.M, L.N, L.K, L.r, L.G)
    assert need > 0                                         # decode-shaped: split-K path
    ws = torch.zeros(need, dtype=torch.uint8, device="cuda")
    Ybig = torch.full((L.M, L.N + 64), 7.0, dtype=torch.float16, device="cuda")
    Yv = Ybig[:, :L.N]
    twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP16, Y=Yv, ws=ws)
    a = Yv.clone()
    twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP16, Y=Yv, ws=ws)       # same ws, not re-zeroed
    assert torch.equal(a, Yv)                                            # deterministic split-K
    assert (Ybig[:, L.N:] == 7.0).all()                                  # padding untouched
    ref = oracle.forward(L.X, L.Rq, L.sw, L.L1, L.L2, L.G)["Y"]
    y = Yv.float().cpu().numpy().astype(np.float64)
    assert np.abs(y - ref).max() / np.abs(ref).max() <= TOL + 2.0 ** -11  # + FP16 rounding of the store
    counters = ws[:256].cpu().numpy()
    assert (counters == 0).all()


def test_errors_are_reported_not_thrown_by_cuda(twq):
    import torch
    L = gen.make_layer(20, 256, 128, 0, 128, seed=5)
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, L.G)
    with pytest.raises(twq.TwqError):
        twq.dual_linear(X, Xq, sx, packed, 5)
    with pytest.raises(twq.TwqError):
        twq.quantize_act(X, 96)
    with pytest.raises(twq.TwqError) as e:
        twq.dual_linear(X, Xq, sx, packed, twq.OUT_BF16, ws=torch.zeros(256, dtype=torch.uint8, device="cuda"))
    assert e.value.code == 3


# ------------------------------------------------------------------------------ BASELINE.json configs
@pytest.mark.parametrize("M", [1, 16, 128])
def test_config2_qproj(twq, oracle, M):
    _check_layer(twq, oracle, gen.config2_qproj(M, with_tinv=(M == 16)))


def _sample_rows(M, n):
    return sorted(set(np.linspace(0, M - 1, n).astype(int).tolist()))


@pytest.mark.parametrize("which,r", [("gate_up", 128), ("down", 128), ("gate_up", 256)])
def test_config3_mlp_prefill_sampled(twq, oracle, which, r):
    """Full size, the launch configuration bench.py times; 64 token rows (all N, all groups) are compared."""
    L = gen.config3_mlp(which, M=2048, r=r)
    _check_layer(twq, oracle, L, rows=_sample_rows(2048, 64))


def test_config3_every_row_of_one_ntile(twq, oracle):
    """All 2048 token rows of the n-tile [1280,1408) of gate/up: covers every token tile of the grid."""
    import torch
    L = gen.config3_mlp("gate_up", M=2048, r=128)
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, L.G)
    Y32 = twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32).cpu().numpy().astype(np.float64)
    n0, n1 = 1280, 1408
    ref = oracle.forward(L.X, L.Rq[n0:n1], L.sw[n0:n1], L.L1, np.ascontiguousarray(L.L2[:, n0:n1]), L.G)["Y"]
    assert np.abs(Y32[:, n0:n1] - ref).max() / np.abs(ref).max() <= TOL


@pytest.mark.parametrize("which,M,nrows", [("attn", 64, None), ("gate_up", 1, None), ("down", 1, None),
                                           ("attn", 4096, 24)])
def test_config4_qwen(twq, oracle, which, M, nrows):
    L = gen.config4_qwen(which, M)
    _check_layer(twq, oracle, L, rows=None if nrows is None else _sample_rows(M, nrows), check_P=(M <= 64))


@pytest.mark.parametrize("which,M", [("q", 1), ("k", 8), ("down", 16), ("gate_up", 2)])
def test_config5_llama70b(twq, oracle, which, M):
    _check_layer(twq, oracle, gen.config5_llama70b(which, M), check_P=(which != "gate_up"))


def test_config5_llama70b_largest_prefill_sampled(twq, oracle):
    """configs[4] at its largest layer and a prefill batch: gate/up K = 8192, N = 28672, r = 256, M = 2048 (the
    rank-256 buffers force the 64-token tile); 24 token rows x all N are compared, without the P dump (60 GB)."""
    L = gen.config5_llama70b("gate_up", 2048)
    _check_layer(twq, oracle, L, rows=_sample_rows(2048, 24), check_P=False)
