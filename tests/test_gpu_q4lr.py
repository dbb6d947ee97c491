"""GPU parity of the paper's 4-bit low-rank branch through the C ABI:
twq_pack_weights_q4lr + twq_dual_linear_q4lr_x against oracle.forward_q4lr.

Bars (readings R18-R22):
  * activation codes / scales and the residual's integer accumulators P: bit-exact;
  * H (FP32 sum on the GPU, FP64 in the oracle): within 1e-5 of max|H|;
  * the re-quantizer takes its integer decision in FP32 on both sides, each from its own H (R22): the GPU's Q_H / s_H are
    EXACTLY the FP32 quantizer of Eq. 1 applied to the GPU's H (restated here in numpy float32), and differ from the
    oracle's only where the oracle's H * (1/s_H) lies within 1e-3 of a rounding boundary, by one step;
  * Y: within 1e-5 of the FP64 value formed from the GPU's own Q_H / s_H (every other term from the oracle), and within
    north_star's 2e-3 of the oracle's Y;  BF16 output == rne(FP32 output) bit for bit.
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
    yield twq.testing_set_plan_flags
    twq.testing_set_plan_flags(0)


def _dev(a, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t if dtype is None else t.view(dtype)


def _np_requant(H32, Gr):
    M, r = H32.shape
    h = H32.reshape(M, r // Gr, Gr)
    amax = np.maximum(np.abs(h).max(axis=2), np.float32(2.0 ** -30))
    s = (amax / np.float32(7.0)).astype(np.float32)
    inv = (np.float32(1.0) / s).astype(np.float32)
    q = np.clip(np.rint((h * inv[:, :, None]).astype(np.float32)), -7, 7).astype(np.int8)
    return q.reshape(M, r), s


def _check(twq, oracle, M, K, N, r, G, with_tinv=False, seed=0, expect_launches=None):
    import torch
    L = gen.make_layer(M, K, N, 0, G, seed=8000 + seed, with_tinv=with_tinv)
    Uq, su, Vq, sv = gen.make_q4_lowrank(K, N, r, G, seed=9000 + seed)
    Gr = twq.lowrank_group(r)
    X = _dev(L.X.view(np.int16), torch.bfloat16)
    tinv = _dev(L.tinv) if L.tinv is not None else None
    packed = twq.pack_weights_q4lr(_dev(L.Rq), _dev(L.sw), _dev(Uq), _dev(su), _dev(Vq), _dev(sv), G)
    Xq_o = torch.full((M, K // 2), 0x55, dtype=torch.uint8, device="cuda")
    sx_o = torch.full((M, K // G), -1.0, dtype=torch.float32, device="cuda")
    dP = torch.zeros((M, L.ng, N), dtype=torch.int32, device="cuda")
    dH = torch.full((M, r), float("nan"), dtype=torch.float32, device="cuda")
    dQ = torch.full((M, r), 99, dtype=torch.int8, device="cuda")
    dS = torch.full((M, r // Gr), -1.0, dtype=torch.float32, device="cuda")
    Y32 = twq.dual_linear_q4lr_x(X, packed, tinv, twq.OUT_FP32, Xq_out=Xq_o, sx_out=sx_o, dbg_P=dP, dbg_H=dH, dbg_QH=dQ,
                                 dbg_sH=dS)
    if expect_launches is not None:
        assert twq.last_launch_count() == expect_launches
    Y16 = twq.dual_linear_q4lr_x(X, packed, tinv, twq.OUT_BF16)
    torch.cuda.synchronize()
    ref = oracle.forward_q4lr(L.X, L.Rq, L.sw, Uq, su, Vq, sv, G, tinv=L.tinv, want_H=True)
    res = oracle.forward(L.X, L.Rq, L.sw, None, None, G, tinv=L.tinv, want_P=True)
    assert (Xq_o.cpu().numpy() == ref["Xq"]).all(), "codes"
    assert (sx_o.cpu().numpy() == ref["sx"]).all(), "scales"
    assert (dP.cpu().numpy().astype(np.int64) == res["P"]).all(), "residual accumulators"
    H, QH, sH = dH.cpu().numpy(), dQ.cpu().numpy(), dS.cpu().numpy()
    hmax = np.abs(ref["H"]).max()
    assert np.abs(H.astype(np.float64) - ref["H"]).max() <= 1e-5 * hmax, "H"
    q_np, s_np = _np_requant(H, Gr)                       # the decision in FP32, from the GPU's own H: exact
    assert (sH == s_np).all(), "s_H is not Eq. 1 of the kernel's H"
    assert (QH == q_np).all(), "Q_H is not Eq. 1 of the kernel's H"
    assert np.allclose(sH, ref["sH"], rtol=1e-5, atol=0), "s_H against the oracle"
    diff = QH.astype(np.int32) - ref["QH"].astype(np.int32)
    if diff.any():
        t = ref["H"] / np.repeat(ref["sH"].astype(np.float64), Gr, axis=1)
        dist = np.abs(np.abs(t - np.floor(t)) - 0.5)
        bad = diff != 0
        assert np.abs(diff).max() <= 1 and (dist[bad] < 1e-3).all(), "Q_H differs away from a rounding boundary"
        assert bad.sum() <= max(2, M * r // 500)
    # Y from the kernel's own Q_H / s_H, every other term from the oracle (FP64)
    ylr = np.zeros((M, N))
    for h in range(r // Gr):
        P2 = QH[:, h * Gr:(h + 1) * Gr].astype(np.int64) @ Vq[:, h * Gr:(h + 1) * Gr].astype(np.int64).T
        ylr += sH[:, h:h + 1].astype(np.float64) * sv[:, h].astype(np.float64)[None, :] * P2
    y = Y32.cpu().numpy().astype(np.float64)
    ymax = np.abs(ref["Y"]).max()
    assert np.abs(y - (res["Y"] + ylr)).max() <= 1e-5 * ymax, "Y against its own Q_H"
    err = np.abs(y - ref["Y"]).max() / ymax
    assert err <= TOL, err
    assert np.abs(ylr).max() > 0.005 * ymax               # the branch matters in this case
    assert torch.equal(Y16.view(torch.int16), Y32.to(torch.bfloat16).view(torch.int16)), "BF16 != rne(Y32)"
    return err


@pytest.mark.parametrize("M,K,N,r,G,with_tinv", [
    (8, 256, 512, 16, 64, False),       # configs[0] shape: gr = 16, stored rows padded to 32 codes
    (3, 192, 48, 32, 64, True),         # three K-groups over the cluster ranks: most ranks hold no slice of U
    (1, 4096, 4096, 128, 128, False),   # configs[1], M = 1
    (16, 4096, 4096, 128, 128, True),   # configs[1], headline M, diagonal transform
    (8, 2048, 528, 48, 128, False),     # gr = 48: padded rows, ragged tile count
    (40, 1024, 528, 96, 64, True),      # four token tiles (M > 32), gr = 96 (three MMA K-steps)
    (25, 2048, 2064, 128, 128, True),   # two token tiles
    (64, 2048, 1040, 128, 128, False),  # the largest slab
    (12, 8192, 1024, 256, 128, False),  # r = 256: two r-groups, eight j tiles per warp
    (16, 5120, 5120, 256, 128, False),  # configs[3] q shape
])
def test_q4lr_one_launch(twq, oracle, M, K, N, r, G, with_tinv):
    _check(twq, oracle, M, K, N, r, G, with_tinv, seed=M + N + r, expect_launches=1)


@pytest.mark.parametrize("M,K,N,r,G", [
    (16, 4096, 14336, 128, 128),     # configs[2] gate/up
    (8, 14336, 4096, 128, 128),      # configs[2] down: 112 K-groups
    (16, 4096, 14336, 256, 128),     # configs[2] at r = 256
    (16, 8192, 8192, 256, 128),      # configs[4] q / o
    (4, 5120, 25600, 256, 128),      # configs[3] gate/up
])
def test_q4lr_config_shapes_small_batches(twq, oracle, M, K, N, r, G):
    """The layer shapes of BASELINE.json's configs 3-5 at decode-sized M through the 4-bit low-rank path."""
    _check(twq, oracle, M, K, N, r, G, False, seed=M + N // 7 + r, expect_launches=1)


@pytest.mark.parametrize("M,K,N,r,G", [
    (4, 25600, 5120, 256, 128),      # configs[3] down: 200 K-groups
    (1, 8192, 28672, 256, 128),      # configs[4] gate/up: 32 channel tiles per CTA beside a 64 KB resident activation tile
])
def test_q4lr_shapes_beyond_shared_memory_are_refused_not_wrong(twq, M, K, N, r, G):
    """Where the resident quantized tile, the FP32 H and the rings do not fit in shared memory even for a 16-token slab the call
    returns TWQ_ERR_UNSUPPORTED (include/twq.h) and launches nothing."""
    import torch
    L = gen.make_layer(M, K, 64, 0, G, seed=8400)
    X = _dev(L.X.view(np.int16), torch.bfloat16)
    nbytes = int(twq.load_library().twq_packed_bytes_q4lr(N, K, r, G))
    assert nbytes > 0
    packed = twq.PackedLayer(torch.zeros(nbytes, dtype=torch.uint8, device="cuda"), N, K, r, G)
    Y = torch.full((M, N), 3.0, dtype=torch.float32, device="cuda")
    with pytest.raises(twq.TwqError) as e:
        twq.dual_linear_q4lr_x(X, packed, None, twq.OUT_FP32, Y=Y)
    assert e.value.code == 2
    torch.cuda.synchronize()
    assert (Y == 3.0).all()


def test_q4lr_long_K_takes_smaller_slabs(twq, oracle):
    """configs[3] q shape at M = 64: the quantized tile of 64 (or 32) tokens, the FP32 H and its partial do not fit beside
    the rings at r = 256, so the call runs as four slabs of 16 tokens."""
    _check(twq, oracle, 64, 5120, 5120, 256, 128, False, seed=77, expect_launches=4)


@pytest.mark.parametrize("M", [65, 130])
def test_q4lr_slabs_of_64_tokens(twq, oracle, M):
    """Larger M: consecutive slabs of at most 64 tokens, one launch each (include/twq.h)."""
    _check(twq, oracle, M, 1024, 512, 64, 128, True, seed=M, expect_launches=(M + 63) // 64)


@pytest.mark.parametrize("cs", [1, 2, 4, 8, 16])
@pytest.mark.parametrize("M,K,N,r,G", [(1, 4096, 1024, 128, 128), (20, 1024, 528, 64, 64), (16, 2048, 2048, 256, 128)])
def test_q4lr_every_cluster_size(twq, oracle, plan_flags, cs, M, K, N, r, G):
    plan_flags(twq.plan_decode_cs(cs))
    _check(twq, oracle, M, K, N, r, G, False, seed=cs + M)


@pytest.mark.parametrize("M,K,N,r,G", [(1, 4096, 4096, 128, 128), (2, 1024, 528, 32, 64), (16, 4096, 4096, 128, 128),
                                       (40, 2048, 1040, 256, 128)])
def test_q4lr_is_deterministic_under_repetition(twq, M, K, N, r, G):
    """Four hand-offs between the CTAs of a cluster (quantized tile -- local for one or two tokens --, H partials, H) ordered
    by mbarriers only: 60 back-to-back calls must be bit-identical, the re-quantized codes included."""
    import torch
    L = gen.make_layer(M, K, N, 0, G, seed=8300 + M, with_tinv=True)
    Uq, su, Vq, sv = gen.make_q4_lowrank(K, N, r, G, seed=9300 + M)
    X = _dev(L.X.view(np.int16), torch.bfloat16)
    tinv = _dev(L.tinv)
    packed = twq.pack_weights_q4lr(_dev(L.Rq), _dev(L.sw), _dev(Uq), _dev(su), _dev(Vq), _dev(sv), G)
    Y0 = twq.dual_linear_q4lr_x(X, packed, tinv, twq.OUT_FP32).clone()
    Q0 = torch.empty((M, r), dtype=torch.int8, device="cuda")
    twq.dual_linear_q4lr_x(X, packed, tinv, twq.OUT_FP32, dbg_QH=Q0)
    Ys = [torch.empty((M, N), dtype=torch.float32, device="cuda") for _ in range(4)]
    Q = torch.empty((M, r), dtype=torch.int8, device="cuda")
    for i in range(60):
        twq.dual_linear_q4lr_x(X, packed, tinv, twq.OUT_FP32, Y=Ys[i % 4], dbg_QH=Q if i % 5 == 0 else None)
        if i % 4 == 3:
            for Y in Ys:
                assert torch.equal(Y, Y0), i
            assert torch.equal(Q, Q0)


@pytest.mark.parametrize("M,out", [(7, "fp16"), (70, "bf16")])
def test_q4lr_row_strides_and_16_bit_outputs(twq, oracle, M, out):
    """ldx > K, ldy > N (a pitch that is not a multiple of 16 bytes for the second slab's start to matter), FP16 / BF16
    outputs, two slabs: outputs equal the rounding of the FP32 output, padding columns of Y untouched."""
    import torch
    K, N, r, G = 1024, 528, 64, 128
    L = gen.make_layer(M, K, N, 0, G, seed=8500 + M, with_tinv=True)
    Uq, su, Vq, sv = gen.make_q4_lowrank(K, N, r, G, seed=9500 + M)
    buf = np.zeros((M, K + 72), np.uint16)
    buf[:, :K] = L.X
    X = _dev(buf.view(np.int16), torch.bfloat16)[:, :K]
    assert X.stride(0) == K + 72
    tinv = _dev(L.tinv)
    packed = twq.pack_weights_q4lr(_dev(L.Rq), _dev(L.sw), _dev(Uq), _dev(su), _dev(Vq), _dev(sv), G)
    Y32 = twq.dual_linear_q4lr_x(X, packed, tinv, twq.OUT_FP32)
    dt, code = (torch.float16, twq.OUT_FP16) if out == "fp16" else (torch.bfloat16, twq.OUT_BF16)
    Ybuf = torch.full((M, N + 6), 5.0, dtype=dt, device="cuda")
    Y = Ybuf[:, :N]
    assert Y.stride(0) == N + 6
    twq.dual_linear_q4lr_x(X, packed, tinv, code, Y=Y)
    torch.cuda.synchronize()
    assert torch.equal(Y.contiguous().view(torch.int16), Y32.to(dt).view(torch.int16))
    assert (Ybuf[:, N:] == 5.0).all()
    ref = oracle.forward_q4lr(L.X, L.Rq, L.sw, Uq, su, Vq, sv, G, tinv=L.tinv)["Y"]
    assert np.abs(Y32.cpu().numpy().astype(np.float64) - ref).max() / np.abs(ref).max() <= TOL


def test_q4lr_zero_factor_is_the_plain_residual(twq, oracle):
    """U = 0: H = 0, s_H = 2^-30 / 7, Q_H = 0, and Y is the rank-0 layer (north_star's r = 0 reduction)."""
    import torch
    M, K, N, r, G = 5, 1024, 256, 64, 128
    L = gen.make_layer(M, K, N, 0, G, seed=8100)
    Uq, su, Vq, sv = gen.make_q4_lowrank(K, N, r, G, seed=9100)
    X = _dev(L.X.view(np.int16), torch.bfloat16)
    packed = twq.pack_weights_q4lr(_dev(L.Rq), _dev(L.sw), _dev(np.zeros_like(Uq)), _dev(su), _dev(Vq), _dev(sv), G)
    dQ = torch.full((M, r), 99, dtype=torch.int8, device="cuda")
    dS = torch.full((M, 1), -1.0, dtype=torch.float32, device="cuda")
    Y = twq.dual_linear_q4lr_x(X, packed, None, twq.OUT_FP32, dbg_QH=dQ, dbg_sH=dS)
    p0 = twq.pack_weights(_dev(L.Rq), _dev(L.sw), None, None, G)
    Y0 = twq.dual_linear_x(X, p0, None, twq.OUT_FP32)
    torch.cuda.synchronize()
    assert (dQ == 0).all() and (dS.cpu().numpy() == np.float32(2.0 ** -30) / np.float32(7.0)).all()
    ref = oracle.forward(L.X, L.Rq, L.sw, None, None, G)["Y"]
    assert np.abs(Y.cpu().numpy() - ref).max() <= 1e-5 * np.abs(ref).max()
    assert (Y - Y0).abs().max().item() <= 1e-5 * float(np.abs(ref).max())


def test_q4lr_errors(twq):
    import torch
    lib = twq.load_library()
    assert lib.twq_packed_bytes_q4lr(256, 256, 144, 128) == 0          # r > 128 must be 256
    assert lib.twq_packed_bytes_q4lr(256, 256, 0, 128) > 0
    L = gen.make_layer(4, 256, 64, 0, 64, seed=1)
    Uq, su, Vq, sv = gen.make_q4_lowrank(256, 64, 32, 64, seed=2)
    packed = twq.pack_weights_q4lr(_dev(L.Rq), _dev(L.sw), _dev(Uq), _dev(su), _dev(Vq), _dev(sv), 64)
    X = _dev(L.X.view(np.int16), torch.bfloat16)
    Y = torch.empty((4, 32), dtype=torch.float32, device="cuda")        # ldy < N
    with pytest.raises(twq.TwqError) as e:
        twq.dual_linear_q4lr_x(X, packed, None, twq.OUT_FP32, Y=Y)
    assert e.value.code == 1
