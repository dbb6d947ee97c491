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


@pytest.fixture
def plan_flags(twq):
    """Planner overrides of include/twq_testing.h for one test (reset to 0 afterwards)."""
    yield twq.testing_set_plan_flags
    twq.testing_set_plan_flags(0)


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
    """Full pipeline on L; compare every output (or the given token rows) with the oracle.  The integer accumulators are
    dumped for the whole call (dbg_P [M, ng, N] lives in HBM only) and the sampled rows are gathered on the device."""
    import torch
    X, packed, tinv = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, L.G, tinv)
    dbg = torch.zeros((L.M, L.ng, L.N), dtype=torch.int32, device="cuda") if check_P else None
    need = twq.workspace_bytes(L.M, L.N, L.K, L.r, L.G)
    ws = torch.zeros(need, dtype=torch.uint8, device="cuda") if need else None
    Y32 = twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32, dbg_P=dbg, ws=ws)
    Y16 = twq.dual_linear(X, Xq, sx, packed, twq.OUT_BF16, ws=ws)
    torch.cuda.synchronize()
    ref = oracle.forward(L.X, L.Rq, L.sw, L.L1 if L.r else None, L.L2 if L.r else None, L.G, tinv=L.tinv,
                         rows=rows, want_P=check_P)
    assert (Xq.cpu().numpy() == ref["Xq"]).all(), "codes"
    assert (sx.cpu().numpy() == ref["sx"]).all(), "scales"
    sel = slice(None) if rows is None else torch.tensor(rows, device="cuda")
    if check_P:
        assert (dbg[sel].cpu().numpy().astype(np.int64) == ref["P"]).all(), "integer accumulators"
        del dbg
    y = Y32[sel].cpu().numpy().astype(np.float64)
    err = np.abs(y - ref["Y"]).max() / np.abs(ref["Y"]).max()
    assert err <= TOL, err
    assert torch.equal(Y16.view(torch.int16), Y32.to(torch.bfloat16).view(torch.int16)), "BF16 != rne(Y32)"
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
    (16, 7168, 1040, 128, 128),  # long K: more ring chunks than slots, several ring rounds
    (16, 512, 4112, 32, 64),     # many tiles per CTA, whole K in one part
    (17, 384, 400, 48, 128),     # two 16-token MMA tiles, second almost empty
    (32, 1024, 528, 256, 64),    # two full token tiles, rank 256, G = 64
    (25, 2048, 2064, 128, 128),  # ragged second token tile, N = 258 tiles over the grid
    (2, 256, 8192, 16, 128),     # many tiles per CTA; smallest rank
    (4, 128, 16, 256, 128),      # one K-group, two tiles, rank 256 with most cluster ranks holding no K slab
    (33, 512, 272, 256, 64),     # four 16-token MMA tiles, the third almost empty, the fourth empty; rank 256
    (64, 2048, 1040, 128, 128),  # four full token tiles
    (50, 1024, 4112, 48, 128),   # ragged fourth token tile, many tiles per CTA
    (40, 640, 16, 0, 128),       # rank 0 with four token tiles
])
def test_decode_kernel_shapes(twq, oracle, M, K, N, r, G):
    """M <= 64 takes the bulk-copy streaming kernel (decode_kernel.cu); same bar as every other shape."""
    assert twq.testing_describe_plan(M, N, K, r, G)["kernel"] == "decode"
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
def test_fused_kernel_cta_pairs(twq, oracle, plan_flags, M, K, N, r, G):
    """128-token tiles in an even cluster run as CTA pairs (cta_group::2, fused_kernel.cuh); same bar.
    Shapes this small would split K instead; the planner's testing override sends them down the unsplit path."""
    plan_flags(twq.PLAN_NO_SPLIT)
    plan = twq.testing_describe_plan(M, N, K, r, G)
    assert plan["kernel"] == "tcgen05" and plan["pair"] == 1 and plan["splits"] == 1
    assert twq.workspace_bytes(M, N, K, r, G) == 0
    rows = None if M * N * K <= 2 ** 29 else sorted(set(np.linspace(0, M - 1, 96).astype(int).tolist()))
    _check_layer(twq, oracle, gen.make_layer(M, K, N, r, G, seed=3000 + M, with_tinv=(M % 2 == 0)), rows=rows)


@pytest.mark.parametrize("cap,tn,M,K,N,r,G", [
    (1, 64, 256, 1024, 2048, 128, 128),    # 4 token tiles of 64, several per cluster
    (2, 32, 128, 2048, 4096, 128, 128),    # the mid-M measurement of DESIGN.md 6.3: 4 x 32 tokens, no K split, no workspace
    (2, 32, 100, 512, 1040, 64, 64),       # ragged token tile and channel tile, G = 64
    (1, 64, 200, 1024, 1024, 256, 128),    # rank 256 beside a 64-token tile
])
def test_fused_kernel_small_token_tiles_unsplit(twq, oracle, plan_flags, cap, tn, M, K, N, r, G):
    """M > 64 with the token tile capped (TWQ_PLAN_FUSED_TN_CAP): the 32- / 64-token instantiations of the tcgen05 kernel
    walking several token tiles, which production shapes only reach through the rank-256 fallback; same bar."""
    plan_flags(twq.plan_fused_tn_cap(cap) | twq.PLAN_NO_SPLIT)
    plan = twq.testing_describe_plan(M, N, K, r, G)
    assert plan["kernel"] == "tcgen05" and plan["tile_tokens"] == tn and plan["splits"] == 1
    assert twq.workspace_bytes(M, N, K, r, G) == 0
    _check_layer(twq, oracle, gen.make_layer(M, K, N, r, G, seed=3300 + M, with_tinv=(M % 2 == 0)))


@pytest.mark.parametrize("pad", [0, 8, 2, 1])
@pytest.mark.parametrize("split,N", [(False, 1232), (False, 1200), (True, 1232)])
def test_fused_kernel_store_paths(twq, oracle, plan_flags, pad, split, N):
    """Every store path of the fused kernel writes the same Y (fused_kernel.cuh, 'The store of a finished tile' in
    DESIGN.md 6.2): row pitch N + pad selects staged TMA tiles / 16-byte transposed stores (pad % 8 == 0), lane pairs
    (even pad) or element stores (odd pad); unsplit 128-token tiles (CTA pairs: 10 channel tiles) or the split-K
    fix-up.  Ragged last token tile and a last channel tile of 80 / 48 channels (the second half-tile store is
    clipped / skipped); columns beyond N must stay untouched."""
    import torch
    M, K, r, G = 300, 512, 64, 128
    if not split:
        plan_flags(twq.PLAN_NO_SPLIT)
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


@pytest.mark.parametrize("M,flags,kernel,pair,split", [
    (5, 0, "decode", 0, False),           # small-batch kernel, one token tile
    (24, 0, "decode", 0, False),          # small-batch kernel, two token tiles
    (40, 0, "decode", 0, False),          # small-batch kernel, four token tiles
    (72, 0, "tcgen05", 0, True),          # tcgen05 kernel, split-K path
    (300, 1, "tcgen05", 1, False),        # tcgen05 kernel, CTA pairs (PLAN_NO_SPLIT)
    (24, 16, "tcgen05", 0, True),         # small batch forced onto the tcgen05 kernel (PLAN_NO_DECODE)
])
def test_rank0_is_plain_w4a4_and_zero_residual_is_lowrank(twq, oracle, plan_flags, M, flags, kernel, pair, split):
    """north_star special cases on every GPU path.  With R = 0 the output is the low-rank product alone, so an error
    of that branch cannot hide under max|Yref| of the (much larger) residual branch."""
    import torch
    plan_flags(flags)
    K, N = 512, 512
    plan = twq.testing_describe_plan(M, N, K, 64, 128)
    assert plan["kernel"] == kernel and plan["pair"] == pair and (plan["splits"] > 1) == split, plan
    L = gen.make_layer(M, K, N, 0, 128, seed=31)
    _check_layer(twq, oracle, L)
    L = gen.make_layer(M, K, N, 64, 128, seed=32)
    L.Rq[:] = 0
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, L.G)
    ws = None
    need = twq.workspace_bytes(M, N, K, L.r, L.G)
    if need:
        ws = torch.zeros(need, dtype=torch.uint8, device="cuda")
    Y = twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32, ws=ws).cpu().numpy().astype(np.float64)
    Xf = gen.bf16_bits_to_f32(L.X).astype(np.float64)
    ref = (Xf @ L.L1.astype(np.float64)) @ L.L2.astype(np.float64)      # FP64 BLAS, independent of the oracle
    # H is rounded once to FP16 (reading R12): 2^-11 relative per term of the r-term sum
    assert np.abs(Y - ref).max() / np.abs(ref).max() <= 1e-3


@pytest.mark.parametrize("M,flags", [(7, 0), (20, 0), (40, 0), (72, 0), (300, 1)])
def test_lowrank_fp16_rewrite_saturates_as_documented(twq, oracle, plan_flags, M, flags):
    """include/twq.h: the low-rank branch rewrites X (BF16) to FP16 on chip -- exact in [2^-14, 65504], saturating
    above.  With R = 0 the output is that branch alone: it must equal the FP64 product of the CLAMPED activations
    (values beyond +-65504 saturate; values below 2^-14 only lose bits far under the tolerance).  Every kernel path."""
    import torch
    plan_flags(flags)
    K, N, r, G = 512, 512, 32, 128
    L = gen.make_layer(M, K, N, r, G, seed=77, lr_sigma=0.002)
    L.Rq[:] = 0
    x = gen.bf16_bits_to_f32(L.X).copy()
    x[:, 5] = 3.0e5                      # beyond FP16 range
    x[:, 17] = -1.0e6
    x[:, 40] = 2.0 ** -20                # FP16 subnormal
    x[:, 41] = 2.0 ** -30                # flushes to zero
    L.X = gen.f32_to_bf16_bits(x)
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, G)
    need = twq.workspace_bytes(M, N, K, r, G)
    ws = torch.zeros(need, dtype=torch.uint8, device="cuda") if need else None
    Y = twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32, ws=ws).cpu().numpy().astype(np.float64)
    xc = np.clip(gen.bf16_bits_to_f32(L.X).astype(np.float64), -65504.0, 65504.0)
    ref = (xc @ L.L1.astype(np.float64)) @ L.L2.astype(np.float64)
    assert np.isfinite(Y).all()
    assert np.abs(Y - ref).max() / np.abs(ref).max() <= 1e-3
    unclamped = (gen.bf16_bits_to_f32(L.X).astype(np.float64) @ L.L1.astype(np.float64)) @ L.L2.astype(np.float64)
    assert np.abs(unclamped - ref).max() / np.abs(ref).max() > 0.1      # the clamp is what the kernel computes, not X itself


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


@pytest.mark.parametrize("cs", [1, 2, 4, 8, 16])
@pytest.mark.parametrize("M,K,N,r,G", [(1, 4096, 1024, 128, 128), (16, 2048, 2048, 256, 128), (20, 1024, 528, 64, 64),
                                       (56, 512, 528, 128, 128)])
def test_decode_kernel_every_cluster_size(twq, oracle, plan_flags, cs, M, K, N, r, G):
    """decode_kernel.cu shares H = X*L1 inside a thread-block cluster: every cluster size the planner can pick
    (16 on an idle B200) gives the same Y within the tolerance, repeatably, with no workspace."""
    import torch
    plan_flags(twq.plan_decode_cs(cs))
    plan = twq.testing_describe_plan(M, N, K, r, G)
    assert plan["kernel"] == "decode" and plan["cluster"] == cs, plan
    assert twq.workspace_bytes(M, N, K, r, G) == 0
    L = gen.make_layer(M, K, N, r, G, seed=5200 + M)
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, G)
    ref = oracle.forward(L.X, L.Rq, L.sw, L.L1, L.L2, G, want_P=False)["Y"]
    ys = [twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32) for _ in range(3)]
    torch.cuda.synchronize()
    for y in ys:
        assert np.abs(y.cpu().numpy().astype(np.float64) - ref).max() / np.abs(ref).max() <= TOL
        assert (y == ys[0]).all(), "not deterministic across calls"


def test_decode_kernel_strides_fp16_output_no_workspace(twq, oracle):
    """Small batches run the bulk-copy streaming kernel: no scratch, padded Y rows untouched, repeatable."""
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
    L = gen.make_layer(72, 512, 256, 32, 128, seed=41)
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, L.G)
    need = twq.workspace_bytes(L.M, L.N, L.K, L.r, L.G)
    assert need > 0                                         # few output tiles: split-K path of the tcgen05 kernel
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
    L = gen.make_layer(72, 256, 128, 0, 128, seed=5)
    X, packed, _ = _upload(twq, L)
    Xq, sx = twq.quantize_act(X, L.G)
    with pytest.raises(twq.TwqError):
        twq.dual_linear(X, Xq, sx, packed, 5)
    with pytest.raises(twq.TwqError):
        twq.quantize_act(X, 96)
    with pytest.raises(twq.TwqError) as e:
        twq.dual_linear(X, Xq, sx, packed, twq.OUT_BF16, ws=torch.zeros(256, dtype=torch.uint8, device="cuda"))
    assert e.value.code == 3


# ------------------------------------------------------------------------------ the whole hot path in one call
@pytest.mark.parametrize("M,K,N,r,G,with_tinv", [
    (1, 128, 16, 0, 128, False),      # smallest problem, rank 0 (no low-rank warps), one group
    (3, 192, 48, 16, 64, True),       # G = 64, three groups over the cluster ranks (most ranks quantize nothing)
    (8, 2048, 528, 48, 128, False),
    (16, 4096, 4096, 128, 128, True), # configs[1] at the headline M, diagonal transform
    (1, 4096, 4096, 128, 128, False),
    (25, 2048, 2064, 128, 128, True), # two token tiles, ragged
    (64, 2048, 1040, 128, 128, False),# four token tiles
    (50, 1024, 4112, 0, 128, True),   # rank 0 with many tiles
    (12, 8192, 1024, 256, 128, False),# configs[4] k / v shape
])
def test_dual_linear_x_one_launch(twq, oracle, M, K, N, r, G, with_tinv):
    """twq_dual_linear_x at M <= 64: quantizer, both branches and the epilogue in ONE launch.  The codes and scales it
    produces on chip (copied out through Xq_out / sx_out) and the integer accumulators are bit-identical to the oracle,
    and Y is bit-identical to the two-call path wherever both use the same grid (same arithmetic, same order)."""
    import torch
    L = gen.make_layer(M, K, N, r, G, seed=7000 + M + N, with_tinv=with_tinv)
    X, packed, tinv = _upload(twq, L)
    assert twq.workspace_bytes_x(M, N, K, r, G) == 0
    Xq_o = torch.full((M, K // 2), 0x55, dtype=torch.uint8, device="cuda")
    sx_o = torch.full((M, K // G), -1.0, dtype=torch.float32, device="cuda")
    dbg = torch.zeros((M, L.ng, N), dtype=torch.int32, device="cuda")
    Y32 = twq.dual_linear_x(X, packed, tinv, twq.OUT_FP32, Xq_out=Xq_o, sx_out=sx_o, dbg_P=dbg)
    assert twq.last_launch_count() == 1
    Y16 = twq.dual_linear_x(X, packed, tinv, twq.OUT_BF16)
    torch.cuda.synchronize()
    ref = oracle.forward(L.X, L.Rq, L.sw, L.L1 if r else None, L.L2 if r else None, G, tinv=L.tinv, want_P=True)
    assert (Xq_o.cpu().numpy() == ref["Xq"]).all(), "codes"
    assert (sx_o.cpu().numpy() == ref["sx"]).all(), "scales"
    assert (dbg.cpu().numpy().astype(np.int64) == ref["P"]).all(), "integer accumulators"
    err = np.abs(Y32.cpu().numpy().astype(np.float64) - ref["Y"]).max() / np.abs(ref["Y"]).max()
    assert err <= TOL, err
    assert torch.equal(Y16.view(torch.int16), Y32.to(torch.bfloat16).view(torch.int16)), "BF16 != rne(Y32)"
    Xq, sx = twq.quantize_act(X, G, tinv)
    Y2 = twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32)
    if r > 0:      # same grid, same K-parts, same order of every sum: bit-identical
        assert torch.equal(Y2, Y32), "one-launch path differs from quantize_act + dual_linear"
    else:          # rank 0: the one-launch call still runs clusters (they share the quantizer), the two-call path does not
        assert (Y2 - Y32).abs().max().item() <= 1e-5 * float(np.abs(ref["Y"]).max())


@pytest.mark.parametrize("M,K,N,r,G", [(1, 4096, 4096, 128, 128), (5, 2048, 1040, 64, 64), (16, 4096, 4096, 128, 128),
                                       (33, 2048, 2064, 128, 128), (64, 1024, 4096, 256, 128)])
def test_dual_linear_x_is_deterministic_under_repetition(twq, M, K, N, r, G):
    """The one-launch kernel hands data between CTAs of a cluster three times (quantized tile, H partials, H) through
    distributed shared memory, by per-lane stores or bulk copies, ordered by mbarriers only.  A missing fence or an early exit
    shows up as a run-to-run difference: 60 back-to-back calls on rotating outputs must be bit-identical, codes included."""
    import torch
    L = gen.make_layer(M, K, N, r, G, seed=7200 + M, with_tinv=True)
    X, packed, tinv = _upload(twq, L)
    Ys = [torch.empty((M, N), dtype=torch.float32, device="cuda") for _ in range(4)]
    Xqs = [torch.empty((M, K // 2), dtype=torch.uint8, device="cuda") for _ in range(4)]
    Y0 = twq.dual_linear_x(X, packed, tinv, twq.OUT_FP32).clone()
    Xq0, _ = twq.quantize_act(X, G, tinv)
    for i in range(60):
        twq.dual_linear_x(X, packed, tinv, twq.OUT_FP32, Y=Ys[i % 4], Xq_out=Xqs[i % 4] if i % 3 == 0 else None)
        if i % 4 == 3:
            for Y in Ys:
                assert torch.equal(Y, Y0), i
    torch.cuda.synchronize()
    for Xq in Xqs:
        assert torch.equal(Xq, Xq0)


@pytest.mark.parametrize("M,K,N,r,G", [(80, 512, 384, 32, 128), (300, 1024, 1024, 128, 128)])
def test_dual_linear_x_larger_batches_use_the_workspace(twq, oracle, M, K, N, r, G):
    """Beyond the small-batch kernel twq_dual_linear_x runs the stand-alone quantizer into the workspace, then the fused
    layer: two launches, same results; the caller's Xq_out / sx_out are used instead of the workspace when given."""
    import torch
    L = gen.make_layer(M, K, N, r, G, seed=7100 + M, with_tinv=True)
    X, packed, tinv = _upload(twq, L)
    need = twq.workspace_bytes_x(M, N, K, r, G)
    assert need >= M * K // 2 + 4 * M * (K // G)
    ws = torch.zeros(need, dtype=torch.uint8, device="cuda")
    Y = twq.dual_linear_x(X, packed, tinv, twq.OUT_FP32, ws=ws)
    assert twq.last_launch_count() == 2
    sx_o = torch.empty((M, K // G), dtype=torch.float32, device="cuda")
    Xq_o = torch.empty((M, K // 2), dtype=torch.uint8, device="cuda")
    Yb = twq.dual_linear_x(X, packed, tinv, twq.OUT_FP32, ws=ws, Xq_out=Xq_o, sx_out=sx_o)
    torch.cuda.synchronize()
    ref = oracle.forward(L.X, L.Rq, L.sw, L.L1, L.L2, G, tinv=L.tinv)
    assert (Xq_o.cpu().numpy() == ref["Xq"]).all() and (sx_o.cpu().numpy() == ref["sx"]).all()
    assert torch.equal(Y, Yb)
    assert np.abs(Y.cpu().numpy().astype(np.float64) - ref["Y"]).max() / np.abs(ref["Y"]).max() <= TOL
    with pytest.raises(twq.TwqError) as e:
        twq.dual_linear_x(X, packed, tinv, twq.OUT_FP32, ws=torch.zeros(256, dtype=torch.uint8, device="cuda"))
    assert e.value.code == 3


# ------------------------------------------------------------------------------ BASELINE.json configs
@pytest.mark.parametrize("M", [1, 16, 128])
def test_config2_qproj(twq, oracle, M):
    _check_layer(twq, oracle, gen.config2_qproj(M, with_tinv=(M == 16)))


def _sample_rows(M, n):
    return sorted(set(np.linspace(0, M - 1, n).astype(int).tolist()))


@pytest.mark.parametrize("which,r", [("gate_up", 128), ("down", 128), ("gate_up", 256), ("down", 256)])
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


@pytest.mark.parametrize("which,M,nrows", [
    ("attn", 64, None), ("gate_up", 1, None), ("down", 1, None),
    ("gate_up", 64, 32), ("down", 64, 16),                       # M = 64 on the wide and the deep layer
    ("attn", 4096, 24), ("gate_up", 4096, 24), ("down", 4096, 16),   # the largest M of configs[3], every layer
])
def test_config4_qwen(twq, oracle, which, M, nrows):
    """configs[3] (Qwen3-32B shapes, r = 256) at M in {1, 64, 4096}: full size, the launch configuration bench.py
    times; sampled token rows x all N x all groups, INCLUDING the integer accumulators."""
    L = gen.config4_qwen(which, M)
    _check_layer(twq, oracle, L, rows=None if nrows is None else _sample_rows(M, nrows))


@pytest.mark.parametrize("which,M,nrows", [
    ("q", 1, None), ("k", 8, None), ("down", 16, None), ("gate_up", 2, None), ("o", 4, None), ("v", 16, None),
    ("v", 32, None), ("k", 64, None),                            # M = 32 / 64: two / four token tiles of the small-batch kernel
    ("o", 2048, 24), ("down", 2048, 16), ("gate_up", 2048, 24),  # prefill on the square, the deep and the wide layer
    ("q", 8192, 24), ("gate_up", 8192, 16),                      # the top of the "M = 1..8192" sweep
])
def test_config5_llama70b(twq, oracle, which, M, nrows):
    """configs[4] (LLaMA3-70B decoder-block linear set, r = 256) from M = 1 to M = 8192, full size; sampled token
    rows x all N x all groups for the prefill batches, INCLUDING the integer accumulators."""
    L = gen.config5_llama70b(which, M)
    _check_layer(twq, oracle, L, rows=None if nrows is None else _sample_rows(M, nrows))
