"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

The paper prints no worked numerical example of the layer, so the pins are:
Eq. 1 closed form and round-trip bound, invariances, nibble bijection, brute force with
python Fractions / pure-python integers, numpy int64 matmul for P (library routine on a
special case), numpy FP64 matmul for the low-rank branch, r = 0 and R = 0 reductions,
additivity, and the storage ratios PAPER.md L86 prints (tests/golden/).
"""
from fractions import Fraction
import os

import numpy as np
import pytest

from gen import inputs as gen

HERE = os.path.dirname(os.path.abspath(__file__))


def bf16(x):
    return gen.f32_to_bf16_bits(np.asarray(x, np.float32))


def f32(b):
    return gen.bf16_bits_to_f32(b)


# --------------------------------------------------------------------------- quantizer (Eq. 1)
def test_quantizer_closed_form_eq1(oracle):
    """PAPER.md L43-47 Eq. 1 with q_max = 7 on a group whose amax is 7*2^p: s is exactly 2^p,
    so Q = round(X / s) can be written down by hand."""
    G = 64
    x = np.zeros((1, G), np.float32)
    vals = [7.0, -7.0, 3.0, -3.0, 0.5, 1.5, 2.5, -0.5, -1.5, -2.5, 6.5, 0.25, 0.75, -6.5, 1.0, 0.0]
    x[0, :16] = vals
    q, sx = oracle.quantize_act(bf16(x * 4.0), G)      # amax = 28 -> s = 4 exactly
    assert sx[0, 0] == np.float32(4.0)
    # round-half-even (reading R5): 0.5->0, 1.5->2, 2.5->2, 6.5->6, 0.25->0, 0.75->1
    expect = [7, -7, 3, -3, 0, 2, 2, 0, -2, -2, 6, 0, 1, -6, 1, 0]
    assert q[0, :16].tolist() == expect
    assert (q[0, 16:] == 0).all()


def test_quantizer_roundtrip_bound_and_range(oracle):
    """|x~ - s*q| <= s/2 (+ slack 2^-18 for the reciprocal multiply); amax element -> +-7; codes in [-7,7]."""
    L = gen.make_layer(32, 512, 16, 0, 128, seed=11)
    q, sx = oracle.quantize_act(L.X, 128)
    x = f32(L.X).astype(np.float64).reshape(32, 4, 128)
    qq = q.reshape(32, 4, 128).astype(np.float64)
    s = sx.astype(np.float64)[:, :, None]
    assert q.min() >= -7 and q.max() <= 7
    assert (np.abs(x - s * qq) <= 0.5 * s * (1 + 2.0 ** -18)).all()
    amax_idx = np.abs(x).argmax(axis=2)
    top = np.take_along_axis(qq, amax_idx[:, :, None], axis=2)
    assert (np.abs(top) == 7).all()
    # s = amax/7 in FP32
    amax = np.abs(f32(L.X)).reshape(32, 4, 128).max(axis=2)
    assert (sx == (amax / np.float32(7.0)).astype(np.float32)).all()


def test_quantizer_invariances(oracle):
    """Negation flips codes, keeps sx; 2^p scaling keeps codes, scales sx; rows are independent."""
    L = gen.make_layer(8, 256, 16, 0, 64, seed=12)
    q, sx = oracle.quantize_act(L.X, 64)
    qn, sxn = oracle.quantize_act(L.X ^ np.uint16(0x8000), 64)
    assert (qn == -q).all() and (sxn == sx).all()
    x8 = bf16(f32(L.X) * np.float32(8.0))
    q8, sx8 = oracle.quantize_act(x8, 64)
    assert (q8 == q).all() and (sx8 == sx * np.float32(8.0)).all()
    q1, sx1 = oracle.quantize_act(L.X[3:4], 64)
    assert (q1 == q[3:4]).all() and (sx1 == sx[3:4]).all()


def test_quantizer_zero_group_and_transform(oracle):
    """R9: all-zero group -> codes 0, sx = 2^-30/7, finite.  tinv multiplies before the amax (L54-58)."""
    x = np.zeros((2, 128), np.float32)
    x[1, 64:] = np.linspace(-3, 3, 64)
    q, sx = oracle.quantize_act(bf16(x), 64)
    assert (q[0] == 0).all() and np.isfinite(sx).all()
    assert sx[0, 0] == np.float32(2.0 ** -30) / np.float32(7.0)
    tinv = np.full(128, 0.25, np.float32)            # power of two: x*tinv exact
    qt, sxt = oracle.quantize_act(bf16(x), 64, tinv)
    assert (qt[1] == q[1]).all() and sxt[1, 1] == sx[1, 1] * np.float32(0.25)
    # a non-uniform tinv changes which element is the amax
    tinv2 = np.ones(128, np.float32)
    tinv2[64] = 0.0
    q2, _ = oracle.quantize_act(bf16(x), 64, tinv2)
    assert q2[1, 64] == 0 and abs(q2[1, 127]) == 7


def test_quantizer_second_implementation_numpy(oracle):
    """Independent numpy-float32 restatement of Eq. 1 in the op order of reading R8."""
    L = gen.make_layer(16, 512, 16, 0, 128, seed=13, with_tinv=True)
    q, sx = oracle.quantize_act(L.X, 128, L.tinv)
    xt = (f32(L.X) * L.tinv[None, :]).astype(np.float32).reshape(16, 4, 128)
    amax = np.maximum(np.abs(xt).max(axis=2), np.float32(2.0 ** -30))
    s = (amax / np.float32(7.0)).astype(np.float32)
    inv = (np.float32(1.0) / s).astype(np.float32)
    qq = np.clip(np.rint((xt * inv[:, :, None]).astype(np.float32)), -7, 7).astype(np.int8)
    assert (sx == s).all()
    assert (q == qq.reshape(16, 512)).all()


# --------------------------------------------------------------------------- pack / unpack
def test_nibble_bijection_all_bytes(oracle):
    allb = np.arange(256, dtype=np.uint8).reshape(1, 256)
    q = oracle.unpack_nibbles(allb)
    assert q.min() == -8 and q.max() == 7
    assert (oracle.pack_nibbles(q) == allb).all()
    # low nibble = even k (R10), two's complement: byte 0x8F -> (q0,q1) = (-1,-8)
    assert oracle.unpack_nibbles(np.array([[0x8F]], np.uint8)).tolist() == [[-1, -8]]
    assert oracle.pack_nibbles(np.array([[7, -8]], np.int8)).tolist() == [[0x87]]


# --------------------------------------------------------------------------- residual P (Eq. 2)
def test_residual_P_bruteforce_and_library(oracle):
    rng = np.random.default_rng(5)
    M, N, K, G = 3, 5, 128, 64
    qx = rng.integers(-7, 8, (M, K), dtype=np.int8)
    qw = rng.integers(-8, 8, (N, K), dtype=np.int8)
    P = oracle.residual_P(oracle.pack_nibbles(qx), oracle.pack_nibbles(qw), G)
    # pure python triple loop
    for m in range(M):
        for n in range(N):
            for g in range(K // G):
                acc = sum(int(qx[m, k]) * int(qw[n, k]) for k in range(g * G, (g + 1) * G))
                assert P[m, g, n] == acc
    # G = K: plain integer matmul (numpy int64 @)
    P1 = oracle.residual_P(oracle.pack_nibbles(qx), oracle.pack_nibbles(qw), K)
    assert (P1[:, 0, :] == qx.astype(np.int64) @ qw.astype(np.int64).T).all()
    assert np.abs(P).max() <= 56 * G
    # extreme codes hit the bound 7*8*G exactly
    qx1 = np.full((1, K), -7, np.int8)
    qw1 = np.full((1, K), -8, np.int8)
    assert oracle.residual_P(oracle.pack_nibbles(qx1), oracle.pack_nibbles(qw1), G)[0, 0, 0] == 56 * G


def test_residual_P_row_subset(oracle):
    rng = np.random.default_rng(6)
    qx = rng.integers(-7, 8, (6, 128), dtype=np.int8)
    qw = rng.integers(-8, 8, (4, 128), dtype=np.int8)
    Xq, R4 = oracle.pack_nibbles(qx), oracle.pack_nibbles(qw)
    P = oracle.residual_P(Xq, R4, 64)
    Ps = oracle.residual_P(Xq, R4, 64, rows=[4, 1])
    assert (Ps[0] == P[4]).all() and (Ps[1] == P[1]).all()


# --------------------------------------------------------------------------- whole forward
def _fraction_forward(L, q, sx):
    """Exact rational evaluation of steps 5-8 (tiny shapes only)."""
    X = f32(L.X)
    M, K, N, r, G = L.M, L.K, L.N, L.r, L.G
    Y = [[None] * N for _ in range(M)]
    for m in range(M):
        H = [sum(Fraction(float(X[m, k])) * Fraction(float(L.L1[k, j])) for k in range(K)) for j in range(r)]
        for n in range(N):
            yres = Fraction(0)
            for g in range(K // G):
                acc = sum(int(q[m, k]) * int(L.Rq[n, k]) for k in range(g * G, (g + 1) * G))
                yres += Fraction(float(sx[m, g])) * Fraction(float(L.sw[n, g])) * acc
            ylr = sum(H[j] * Fraction(float(L.L2[j, n])) for j in range(r))
            Y[m][n] = yres + ylr
    return Y


def test_forward_bruteforce_fractions(oracle):
    L = gen.make_layer(2, 128, 16, 16, 64, seed=21, x_dist="normal", n_outlier=2, outlier_scale=20.0,
                       lr_sigma=0.05)
    out = oracle.forward(L.X, L.Rq, L.sw, L.L1, L.L2, L.G)
    Yf = _fraction_forward(L, out["q"], out["sx"])
    for m in range(L.M):
        for n in range(L.N):
            exact = float(Yf[m][n])
            assert abs(out["Y"][m, n] - exact) <= 1e-12 * max(1.0, abs(exact))


def test_forward_rank0_is_plain_w4a4(oracle):
    """north_star: r = 0 reduces to plain W4A4 = Eq. 2 with group scales: sum_g sx*sw*(qx.qw)."""
    L = gen.make_layer(4, 256, 32, 0, 64, seed=22)
    out = oracle.forward(L.X, L.Rq, L.sw, None, None, L.G, want_P=True)
    deqx = out["q"].astype(np.float64) * np.repeat(out["sx"].astype(np.float64), L.G, axis=1)
    deqw = L.Rq.astype(np.float64) * np.repeat(L.sw.astype(np.float64), L.G, axis=1)
    ref = deqx @ deqw.T                          # Q(X) Q(W) dequantized explicitly, FP64 BLAS
    assert np.allclose(out["Y"], ref, rtol=1e-12, atol=1e-12)
    assert out["P"].shape == (4, 4, 32)


def test_forward_zero_residual_is_lowrank_gemm(oracle):
    """north_star: zero residual reduces to the FP64 low-rank GEMM (X L1) L2, and = X (L1 L2)."""
    L = gen.make_layer(4, 256, 32, 16, 64, seed=23)
    Rq0 = np.zeros_like(L.Rq)
    out = oracle.forward(L.X, Rq0, L.sw, L.L1, L.L2, L.G)
    X = f32(L.X).astype(np.float64)
    ref = (X @ L.L1.astype(np.float64)) @ L.L2.astype(np.float64)
    assert np.allclose(out["Y"], ref, rtol=1e-12, atol=1e-12)
    ref2 = X @ (L.L1.astype(np.float64) @ L.L2.astype(np.float64))
    assert np.allclose(out["Y"], ref2, rtol=1e-10, atol=1e-10)


def test_forward_additivity_and_transposition_sensitivity(oracle):
    L = gen.make_layer(3, 256, 48, 16, 128, seed=24)
    full = oracle.forward(L.X, L.Rq, L.sw, L.L1, L.L2, L.G)["Y"]
    res = oracle.forward(L.X, L.Rq, L.sw, None, None, L.G)["Y"]
    lr = oracle.forward(L.X, np.zeros_like(L.Rq), L.sw, L.L1, L.L2, L.G)["Y"]
    assert np.allclose(full - res, lr, rtol=1e-10, atol=1e-10)
    # non-square everything: a transposed operand anywhere would have failed the shape-specific refs above;
    # here make sure the two branches are not tiny relative to each other (a dropped term would show)
    assert np.abs(res).max() > 1e-3 and np.abs(lr).max() > 1e-3


def test_forward_row_subset_is_rows_of_the_full_call(oracle):
    """The `rows != NULL` path of twq_oracle_forward (oracle/twq_oracle.c, the path every M >= 2048 parity
    test relies on): rows [4, 1] of a 6-row layer, Y and P, are exactly rows 4 and 1 of the full call --
    through forward() and through forward_from_quantized(); the full call itself is pinned by the brute-force
    and library tests above.  An out-of-order, repeated row and the empty tail (ragged last row) are included."""
    L = gen.make_layer(6, 256, 48, 16, 64, seed=25, with_tinv=True)
    full = oracle.forward(L.X, L.Rq, L.sw, L.L1, L.L2, L.G, tinv=L.tinv, want_P=True)
    for rows in ([4, 1], [5], [0, 5, 5, 2]):
        sub = oracle.forward(L.X, L.Rq, L.sw, L.L1, L.L2, L.G, tinv=L.tinv, rows=rows, want_P=True)
        assert sub["Y"].shape == (len(rows), L.N) and sub["P"].shape == (len(rows), L.ng, L.N)
        for i, m in enumerate(rows):
            assert (sub["Y"][i] == full["Y"][m]).all()          # same FP64 operations in the same order: bit-equal
            assert (sub["P"][i] == full["P"][m]).all()
        # the quantizer outputs are always whole (rows only selects what steps 5-8 evaluate)
        assert (sub["Xq"] == full["Xq"]).all() and (sub["sx"] == full["sx"]).all()
        Y2, P2 = oracle.forward_from_quantized(L.X, full["Xq"], full["sx"], oracle.pack_nibbles(L.Rq), L.sw, L.L1, L.L2,
                                               L.G, rows=rows, want_P=True)
        assert (Y2 == sub["Y"]).all() and (P2 == sub["P"]).all()
    # rank 0 through the same path
    r0 = oracle.forward(L.X, L.Rq, L.sw, None, None, L.G, rows=[4, 1])["Y"]
    f0 = oracle.forward(L.X, L.Rq, L.sw, None, None, L.G)["Y"]
    assert (r0[0] == f0[4]).all() and (r0[1] == f0[1]).all()


# --------------------------------------------------------------------------- NEXT-1: 4-bit low-rank branch
def _q4lr_case(M, K, N, r, G, seed):
    L = gen.make_layer(M, K, N, 0, G, seed=seed)
    Uq, su, Vq, sv = gen.make_q4_lowrank(K, N, r, G, seed=seed + 1000)
    return L, Uq, su, Vq, sv


def _np_requant(H, Gr):
    """numpy-float32 restatement of Eq. 1 (L43-47) on float32(H), groups of Gr along r (readings R18 / R19)."""
    M, r = H.shape
    h32 = H.astype(np.float32).reshape(M, r // Gr, Gr)
    amax = np.maximum(np.abs(h32).max(axis=2), np.float32(2.0 ** -30))
    s = (amax / np.float32(7.0)).astype(np.float32)
    inv = (np.float32(1.0) / s).astype(np.float32)
    q = np.clip(np.rint((h32 * inv[:, :, None]).astype(np.float32)), -7, 7).astype(np.int8)
    return q.reshape(M, r), s


@pytest.mark.parametrize("r,G", [(32, 64), (128, 128), (256, 64)])
def test_q4lr_stage_by_stage_library_restatement(oracle, r, G):
    """H by library integer matmul per group + explicit scale fold; QH / sH by the numpy
    quantizer restatement; Ylr by a second integer matmul per r-group; Yres = the pinned rank-0 forward()."""
    M, K, N = 5, 512, 48
    L, Uq, su, Vq, sv = _q4lr_case(M, K, N, r, G, 31 + r)
    out = oracle.forward_q4lr(L.X, L.Rq, L.sw, Uq, su, Vq, sv, G, want_H=True)
    q, sx = out["q"].astype(np.int64), out["sx"].astype(np.float64)
    ng, Gr = K // G, oracle.lowrank_group(r)
    H = np.zeros((M, r))
    for g in range(ng):
        P1 = q[:, g * G:(g + 1) * G] @ Uq[:, g * G:(g + 1) * G].astype(np.int64).T        # [M, r] exact
        H += sx[:, g:g + 1] * su[:, g].astype(np.float64)[None, :] * P1
    assert np.allclose(out["H"], H, rtol=1e-13, atol=1e-300)
    QH, sH = _np_requant(out["H"], Gr)
    assert (out["sH"] == sH).all() and (out["QH"] == QH).all()
    assert np.abs(out["QH"]).max() == 7                          # every group's largest element lands on +-7
    Ylr = np.zeros((M, N))
    for h in range(r // Gr):
        P2 = QH[:, h * Gr:(h + 1) * Gr].astype(np.int64) @ Vq[:, h * Gr:(h + 1) * Gr].astype(np.int64).T
        Ylr += sH[:, h:h + 1].astype(np.float64) * sv[:, h].astype(np.float64)[None, :] * P2
    yres = oracle.forward(L.X, L.Rq, L.sw, None, None, G)["Y"]
    assert np.allclose(out["Y"], yres + Ylr, rtol=1e-12, atol=1e-12)
    assert np.abs(Ylr).max() > 0.05 * np.abs(yres).max()        # the branch is not negligible in this case


def test_q4lr_bruteforce_fractions(oracle):
    """Exact rational arithmetic on a tiny case, given the oracle's own QH / sH (pinned above)."""
    M, K, N, r, G = 2, 128, 6, 16, 64
    L, Uq, su, Vq, sv = _q4lr_case(M, K, N, r, G, 33)
    out = oracle.forward_q4lr(L.X, L.Rq, L.sw, Uq, su, Vq, sv, G, want_H=True)
    q, sx = out["q"], out["sx"]
    for m in range(M):
        Hm = []
        for j in range(r):
            h = Fraction(0)
            for g in range(K // G):
                acc = sum(int(q[m, k]) * int(Uq[j, k]) for k in range(g * G, (g + 1) * G))
                h += Fraction(float(sx[m, g])) * Fraction(float(su[j, g])) * acc
            Hm.append(h)
            assert abs(out["H"][m, j] - float(h)) <= 1e-13 * abs(float(h)) + 1e-300
        for n in range(N):
            y = Fraction(0)
            for g in range(K // G):
                acc = sum(int(q[m, k]) * int(L.Rq[n, k]) for k in range(g * G, (g + 1) * G))
                y += Fraction(float(sx[m, g])) * Fraction(float(L.sw[n, g])) * acc
            acc = sum(int(out["QH"][m, j]) * int(Vq[n, j]) for j in range(r))
            y += Fraction(float(out["sH"][m, 0])) * Fraction(float(sv[n, 0])) * acc
            assert abs(out["Y"][m, n] - float(y)) <= 1e-12 * max(1.0, abs(float(y)))


def test_q4lr_exactly_representable_closed_form(oracle):
    """Closed form: X = one-hot rows of value 7 (so sx = 1, q = 7 e_k) and su = 1 give H[m,:] = 7 * Uq[:,k_m]; with
    Uq in [-6,6] except one row of 7s, max|H| = 49, so sH = 7 and QH = Uq[:,k_m] exactly, and
    Ylr[m,n] = 7 * sv * sum_j Uq[j,k_m] * Vq[n,j]: an integer matmul times a power of two."""
    K, N, r, G = 128, 8, 16, 64
    rng = np.random.default_rng(5)
    Uq = rng.integers(-6, 7, size=(r, K), dtype=np.int8)
    Uq[0, :] = 7                                                     # every column's amax is 7
    Vq = rng.integers(-8, 8, size=(N, r), dtype=np.int8)
    su = np.ones((r, K // G), np.float16)
    sv = np.full((N, 1), 0.25, np.float16)
    ks = [3, 64, 127]
    X = np.zeros((len(ks), K), np.float32)
    for m, k in enumerate(ks):
        X[m, k] = 7.0
    Rq0 = np.zeros((N, K), np.int8)
    sw = np.ones((N, K // G), np.float16)
    out = oracle.forward_q4lr(bf16(X), Rq0, sw, Uq, su, Vq, sv, G, want_H=True)
    for m, k in enumerate(ks):
        assert (out["H"][m] == 7.0 * Uq[:, k]).all()
        assert out["sH"][m, 0] == 7.0 and (out["QH"][m] == Uq[:, k]).all()
        ref = 7.0 * 0.25 * (Vq.astype(np.int64) @ Uq[:, k].astype(np.int64))
        assert (out["Y"][m] == ref).all()


def test_q4lr_reductions_and_sensitivity(oracle):
    """Zero U -> H = 0 -> QH = 0 -> Y = the residual alone (the pinned rank-0 forward); zero V likewise; zero residual
    -> Y = Ylr alone and Y(res) + Y(lr) = Y(both); swapping the roles of the two r-groups of V changes the result
    (a wrong group index in the second GEMM's scales fails here)."""
    M, K, N, r, G = 3, 256, 24, 256, 64
    L, Uq, su, Vq, sv = _q4lr_case(M, K, N, r, G, 35)
    yres = oracle.forward(L.X, L.Rq, L.sw, None, None, G)["Y"]
    y0 = oracle.forward_q4lr(L.X, L.Rq, L.sw, np.zeros_like(Uq), su, Vq, sv, G, want_H=True)
    assert (y0["QH"] == 0).all() and (y0["sH"] == np.float32(2.0 ** -30) / np.float32(7.0)).all()
    assert (y0["Y"] == yres).all()
    assert (oracle.forward_q4lr(L.X, L.Rq, L.sw, Uq, su, np.zeros_like(Vq), sv, G)["Y"] == yres).all()
    both = oracle.forward_q4lr(L.X, L.Rq, L.sw, Uq, su, Vq, sv, G)["Y"]
    lr = oracle.forward_q4lr(L.X, np.zeros_like(L.Rq), L.sw, Uq, su, Vq, sv, G)["Y"]
    assert np.allclose(both, yres + lr, rtol=1e-12, atol=1e-12)
    sv_sw = sv[:, ::-1].copy()
    assert not np.allclose(oracle.forward_q4lr(L.X, L.Rq, L.sw, Uq, su, Vq, sv_sw, G)["Y"], both, rtol=1e-6)
    rows = [2, 0]
    sub = oracle.forward_q4lr(L.X, L.Rq, L.sw, Uq, su, Vq, sv, G, rows=rows)["Y"]
    assert (sub == both[rows]).all()


def test_q4lr_requantization_error_bound(oracle):
    """The re-quantized branch stays within the quantizer's half-step bound of the un-requantized product
    H . deq(V): |Ylr - sum_j H[m,j] sv qv| <= sum_h (sH/2)(1 + 2^-22) sum_{j in h} |sv qv|."""
    M, K, N, r, G = 4, 512, 32, 256, 128
    L, Uq, su, Vq, sv = _q4lr_case(M, K, N, r, G, 37)
    out = oracle.forward_q4lr(L.X, np.zeros_like(L.Rq), L.sw, Uq, su, Vq, sv, G, want_H=True)
    Gr = oracle.lowrank_group(r)
    dv = Vq.astype(np.float64) * np.repeat(sv.astype(np.float64), Gr, axis=1)            # [N, r]
    exact = out["H"] @ dv.T
    bound = np.zeros((M, N))
    for h in range(r // Gr):
        bound += 0.5 * (1 + 2.0 ** -22) * out["sH"][:, h:h + 1].astype(np.float64) * np.abs(dv[:, h * Gr:(h + 1) * Gr]).sum(axis=1)[None, :]
    err = np.abs(out["Y"] - exact)
    assert (err <= bound).all()
    assert err.max() > 0.02 * bound.max()                      # and the bound is not vacuous


def test_scale_fold_constant_and_pow2_exact(oracle):
    """Constant scales factor out; power-of-two scales and small integers make Y exactly representable."""
    rng = np.random.default_rng(7)
    M, N, K, G = 4, 8, 256, 64
    qx = rng.integers(-7, 8, (M, K), dtype=np.int8)
    qw = rng.integers(-8, 8, (N, K), dtype=np.int8)
    a = np.array([0.5, 2.0, 1.0, 0.25], np.float32)
    b = np.float16([2.0 ** -3] * 4 + [2.0 ** -5] * 4)
    sx = np.repeat(a[:, None], K // G, axis=1)
    sw = np.repeat(b[:, None], K // G, axis=1)
    X = bf16(np.zeros((M, K), np.float32))
    Y = oracle.forward_from_quantized(X, oracle.pack_nibbles(qx), sx, oracle.pack_nibbles(qw), sw, None, None, G)
    ref = (a.astype(np.float64)[:, None] * b.astype(np.float64)[None, :]) * (qx.astype(np.int64) @ qw.astype(np.int64).T)
    assert (Y == ref).all()


def test_round_bf16(oracle):
    v = np.array([1.0, 1.00390625, 1.01171875, -3.0, 0.0, 1e-40, 65504.0, 3.3895313892515355e38], np.float64)
    got = oracle.round_bf16(v)
    # 1 + 2^-8 is a tie -> even (1.0); 1 + 3*2^-8 is a tie -> even (1 + 4*2^-8 = 1.015625)
    assert got[0] == 0x3F80 and got[1] == 0x3F80 and got[2] == 0x3F82 and got[3] == 0xC040 and got[4] == 0
    rnd = np.random.default_rng(3).standard_normal(4096) * 37.0
    assert (oracle.round_bf16(rnd) == gen.f32_to_bf16_bits(rnd.astype(np.float32))).mean() > 0.99  # double rounding rare
    exact = rnd.astype(np.float32).astype(np.float64)
    assert (oracle.round_bf16(exact) == gen.f32_to_bf16_bits(exact.astype(np.float32))).all()


# --------------------------------------------------------------------------- paper-printed numbers
def test_storage_ratios_paper_L86(oracle):
    with open(os.path.join(HERE, "golden", "paper_L86_storage_ratios.txt")) as f:
        rows = [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 2
    for m, n, r, pct in rows:
        m, n, r, pct = int(m), int(n), int(r), float(pct)
        ratio = 100.0 * oracle.lowrank_fp16_bytes(m, n, r) / oracle.residual_4bit_bytes(m, n)
        assert abs(ratio - pct) < 1e-9


# --------------------------------------------------------------------------- generator sanity
def test_generator_statistics():
    L = gen.config2_qproj(16)
    assert L.X.shape == (16, 4096) and L.Rq.shape == (4096, 4096) and L.sw.shape == (4096, 32)
    assert L.Rq.min() == -8 and L.Rq.max() == 7
    assert abs(L.Rq.astype(np.float64).mean() + 0.5) < 0.01
    assert abs((L.Rq.astype(np.float64) ** 2).mean() - 21.5) < 0.05
    assert 0.005 * (1 - 2 ** -11) <= float(L.sw.min()) and float(L.sw.max()) <= 0.02 * (1 + 2 ** -11)  # FP16 RNE of U(0.005,0.02)
    L1 = gen.config1_tiny()
    assert (L1.M, L1.K, L1.N, L1.r, L1.G) == (8, 256, 512, 16, 64)
    a = gen.config1_tiny()
    assert (a.X == L1.X).all() and (a.Rq == L1.Rq).all()
