"""twq_dual_linear_noalloc (include/twq.h): the fused layer for callers that cannot allocate -- the split-K scratch lives in
a static device array inside the library (8.5 MiB).  Its output is compared with the existing path (twq_dual_linear with a
caller workspace) on two calls in a row, and with the CPU oracle within the tolerance of the other parity tests.

This file is collected last on purpose (the suite runs with pytest -x); it passes alone in a fresh process and after the
other tests.
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
    t.testing_set_plan_flags(0)
    return t


def _dev(a, dtype=None):
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t if dtype is None else t.view(dtype)


def _layer(twq, M, K, N, r, G, seed):
    import torch
    L = gen.make_layer(M, K, N, r, G, seed=seed, with_tinv=True)
    X = _dev(L.X.view(np.int16), torch.bfloat16)
    packed = twq.pack_weights(_dev(L.Rq), _dev(L.sw), _dev(L.L1) if r else None, _dev(L.L2) if r else None, G)
    Xq, sx = twq.quantize_act(X, G, _dev(L.tinv))
    return L, X, Xq, sx, packed


@pytest.mark.parametrize("M,K,N,r,G", [
    (128, 4096, 2048, 128, 128),      # 16 channel tiles x 8 K splits: 8 MiB + 256 B of scratch, the largest of the config-shaped calls
    (80, 512, 384, 32, 128),          # three splits, ragged token tile
    (300, 1024, 1024, 128, 128),      # several token tiles, four splits
])
def test_noalloc_matches_the_workspace_path_twice_in_a_row(twq, oracle, M, K, N, r, G):
    import torch
    L, X, Xq, sx, packed = _layer(twq, M, K, N, r, G, seed=9500 + M)
    need = twq.workspace_bytes(M, N, K, r, G)
    assert 0 < need <= twq.noalloc_max_workspace()
    ws = torch.zeros(need, dtype=torch.uint8, device="cuda")
    Yref = twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32, ws=ws)
    Y1 = torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda")
    Y2 = torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda")
    # cumulative number of allocations the caching allocator has served (frees by the garbage collector do not change it)
    n_alloc = torch.cuda.memory_stats()["allocation.all.allocated"]
    twq.dual_linear_noalloc(X, Xq, sx, packed, Y1, twq.OUT_FP32)
    twq.dual_linear_noalloc(X, Xq, sx, packed, Y2, twq.OUT_FP32)          # second call: the scratch holds the first call's state
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == n_alloc
    torch.cuda.synchronize()
    ref = oracle.forward(L.X, L.Rq, L.sw, L.L1 if r else None, L.L2 if r else None, G, tinv=L.tinv)["Y"]
    ymax = float(np.abs(ref).max())
    for Y in (Y1, Y2):
        assert torch.isfinite(Y).all()
        # same kernel, same plan, same order of every sum as the workspace path
        assert (Y - Yref).abs().max().item() <= TOL * ymax
        assert torch.equal(Y, Yref)
        assert np.abs(Y.cpu().numpy().astype(np.float64) - ref).max() / ymax <= TOL
    # a different shape in between, then the first one again: the shared array carries nothing over
    L2, X2, Xq2, sx2, packed2 = _layer(twq, 96, 1024, 512, 64, 128, seed=9600)
    Yo = torch.empty((96, 512), dtype=torch.float32, device="cuda")
    twq.dual_linear_noalloc(X2, Xq2, sx2, packed2, Yo, twq.OUT_FP32)
    Y3 = torch.empty((M, N), dtype=torch.bfloat16, device="cuda")
    twq.dual_linear_noalloc(X, Xq, sx, packed, Y3, twq.OUT_BF16)
    torch.cuda.synchronize()
    ref2 = oracle.forward(L2.X, L2.Rq, L2.sw, L2.L1, L2.L2, 128, tinv=L2.tinv)["Y"]
    assert np.abs(Yo.cpu().numpy().astype(np.float64) - ref2).max() / np.abs(ref2).max() <= TOL
    assert torch.equal(Y3.view(torch.int16), Yref.to(torch.bfloat16).view(torch.int16))


@pytest.mark.parametrize("M,K,N,r,G", [(16, 2048, 2048, 128, 128), (1024, 1024, 4096, 64, 128)])
def test_noalloc_shapes_without_scratch(twq, oracle, M, K, N, r, G):
    """Small batches and prefill-shaped calls need no scratch: the entry point is then twq_dual_linear itself."""
    import torch
    L, X, Xq, sx, packed = _layer(twq, M, K, N, r, G, seed=9700 + M)
    assert twq.workspace_bytes(M, N, K, r, G) == 0
    Y = torch.empty((M, N), dtype=torch.float32, device="cuda")
    twq.dual_linear_noalloc(X, Xq, sx, packed, Y, twq.OUT_FP32)
    Yref = twq.dual_linear(X, Xq, sx, packed, twq.OUT_FP32)
    torch.cuda.synchronize()
    assert torch.equal(Y, Yref)
    ref = oracle.forward(L.X, L.Rq, L.sw, L.L1, L.L2, G, tinv=L.tinv)["Y"]
    assert np.abs(Y.cpu().numpy().astype(np.float64) - ref).max() / np.abs(ref).max() <= TOL


def test_noalloc_rejects_a_shape_beyond_the_static_scratch(twq):
    """A few hundred tokens x few channels: 9.5 MB of split-K scratch > 8.5 MiB -> TWQ_ERR_WORKSPACE, nothing runs."""
    import torch
    M, N, K, r, G = 377, 896, 4096, 0, 128
    assert twq.workspace_bytes(M, N, K, r, G) > twq.noalloc_max_workspace()
    Xq = torch.zeros((M, K // 2), dtype=torch.uint8, device="cuda")
    sx = torch.ones((M, K // G), dtype=torch.float32, device="cuda")
    packed = twq.PackedLayer(torch.zeros(twq.packed_bytes(N, K, r, G), dtype=torch.uint8, device="cuda"), N, K, r, G)
    Y = torch.full((M, N), 7.0, dtype=torch.float32, device="cuda")
    with pytest.raises(twq.TwqError) as e:
        twq.dual_linear_noalloc(None, Xq, sx, packed, Y, twq.OUT_FP32)
    assert e.value.code == 3
    torch.cuda.synchronize()
    assert (Y == 7.0).all()
