"""-m gpu parity of haste_forward_topk (fused top-k inference, Eq. 4: P@k needs the k best labels of
a row) against the fp64 oracle: the oracle's logits (oracle.tail_forward / tail_points, the definition of),
sorted with numpy.  Values must match to fp32 accumulation; the label set must match wherever the oracle's k-th and
(k+1)-th logits are further apart than that accumulation error (ties and near-ties may legitimately swap)."""
import numpy as np
import pytest
import torch

from paper_2606_01117_b200 import synth

pytestmark = pytest.mark.gpu


def _check_topk(z_ref, got_val, got_idx, k, label_offset=0, tol=2e-5):
    """z_ref [n, L] fp64 logits of the rows under test; got_val / got_idx [n, k]."""
    n, L = z_ref.shape
    order = np.argsort(-z_ref, axis=1, kind="stable")
    for i in range(n):
        want_v = z_ref[i, order[i, :k]]
        scale = max(1.0, np.abs(want_v).max())
        kk = min(k, L)
        assert np.all(np.diff(got_val[i, :kk]) <= 0), "values must be descending"
        assert np.allclose(got_val[i, :kk], want_v[:kk], rtol=0, atol=tol * scale), (i, got_val[i], want_v)
        ids = got_idx[i, :kk] - label_offset
        assert np.all((ids >= 0) & (ids < L)) and len(set(ids.tolist())) == kk
        # every returned label really has (almost) the value returned, and nothing clearly better was left out
        assert np.allclose(z_ref[i, ids], got_val[i, :kk], rtol=0, atol=tol * scale)
        if L > kk:
            assert z_ref[i, order[i, kk]] <= got_val[i, kk - 1] + tol * scale
        if kk < k:
            assert np.all(got_idx[i, kk:] == -1) and np.all(np.isneginf(got_val[i, kk:]))


@pytest.mark.parametrize("shape", [(300, 768, 64 * 23 + 11, 64, 128), (130, 256, 32 * 40 + 5, 32, 64), (64, 512, 128 * 5 + 3, 128, 128),
                                   (257, 768, 64 * 300 + 1, 64, 64), (33, 256, 5, 64, 64),
                                   (200, 256, 16 * 90 + 7, 16, 64), (130, 384, 8 * 150 + 3, 8, 128)])
@pytest.mark.parametrize("k", [1, 5, 8])
def test_forward_topk_small(oracle, shape, k):
    from gpu_util import TailRun
    B, d, L, G, K = shape
    off = 1000
    inp = synth.small_case(90 + B, B, d, L, G, K, dtype="bf16", with_bias=(B % 2 == 0), w_std=0.2, label_offset=off, L_total=off + L)
    run = TailRun(inp, G, want_logits=False, label_offset=off)
    assert run.layer.kernel_family == 1
    val = torch.full((B, k), float("nan"), device=run.X.device)
    ind = torch.full((B, k), -7, dtype=torch.int64, device=run.X.device)
    run.layer.forward_topk(B, run.X, run.idx, run.W, run.bias, k, val, ind)
    z = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G, label_offset=off)["z"]
    _check_topk(z, val.cpu().numpy().astype(np.float64), ind.cpu().numpy(), k, label_offset=off)
    # a second call on the same handle gives the same answer (the candidate workspace is rewritten, not accumulated)
    val2, ind2 = torch.empty_like(val), torch.empty_like(ind)
    run.layer.forward_topk(B, run.X, run.idx, run.W, run.bias, k, val2, ind2)
    assert torch.equal(val, val2) and torch.equal(ind, ind2)


def test_forward_topk_ties_go_to_the_smaller_label(oracle):
    """Integer inputs: many exactly equal logits.  The library's rule: larger value first, then the smaller label id."""
    from gpu_util import TailRun
    B, d, L, G, K = 140, 256, 64 * 9 + 7, 64, 64
    inp = synth.small_case(5, B, d, L, G, K, dtype="bf16", with_bias=False)
    rng = np.random.RandomState(2)
    Xi = rng.randint(-1, 2, size=(B, d)).astype(np.float32)
    Wi = rng.randint(-1, 2, size=(L, K)).astype(np.float32)
    inp.X, inp.W = Xi, Wi
    inp.bits["X"], inp.bits["W"] = synth.round_bf16(Xi)[0].reshape(B, d), synth.round_bf16(Wi)[0].reshape(L, K)
    run = TailRun(inp, G, want_logits=False)
    k = 8
    val = torch.empty(B, k, device=run.X.device)
    ind = torch.empty(B, k, dtype=torch.int64, device=run.X.device)
    run.layer.forward_topk(B, run.X, run.idx, run.W, None, k, val, ind)
    z = oracle.tail_forward(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, G)["z"]
    order = np.lexsort((np.arange(L)[None, :].repeat(B, 0), -z), axis=1)[:, :k]     # value descending, then label ascending
    assert np.array_equal(ind.cpu().numpy(), order)
    assert np.array_equal(val.cpu().numpy().astype(np.float64), np.take_along_axis(z, order, axis=1))


def test_forward_topk_config3_full_size(oracle):
    """Config 3 (653 707 tail labels, B = 512) in the launch configuration of the forward kernel: the top-5 of sampled
    batch rows (one per 128-row tile and the last row) against the oracle's logits over ALL labels of those rows."""
    from gpu_util import to_dev, t32
    from paper_2606_01117_b200 import haste
    cfg = synth.CONFIGS["670k"]
    inp = synth.make_inputs(cfg, with_head=False)
    B, d, L, G, K = cfg.B, cfg.d, cfg.L_t, cfg.G, cfg.K
    dev = torch.device("cuda:0")
    layer = haste.HasteLayer(d, L, G, K, B, "bf16", label_offset=cfg.L_h, flags=haste.HASTE_IDX_SORTED_DISTINCT)
    X, W, idx = to_dev(inp, "X"), to_dev(inp, "W"), t32(inp.idx)
    k = 5
    val = torch.empty(B, k, device=dev)
    ind = torch.empty(B, k, dtype=torch.int64, device=dev)
    layer.forward_topk(B, X, idx, W, None, k, val, ind)
    rows = np.array([3, 130, 300, 450, B - 1], dtype=np.int32)
    z = np.empty((rows.size, L))
    labs = np.arange(L, dtype=np.int64)
    for n_, r in enumerate(rows):
        z[n_] = oracle.tail_points(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, G, np.full(L, r, dtype=np.int32), labs,
                                   label_offset=cfg.L_h)["z"]
    sel = torch.from_numpy(rows.astype(np.int64)).to(dev)
    _check_topk(z, val[sel].cpu().numpy().astype(np.float64), ind[sel].cpu().numpy(), k, label_offset=cfg.L_h)
    # every row: descending, distinct, inside the layer's id range
    v, i = val.cpu().numpy(), ind.cpu().numpy()
    assert np.all(np.diff(v, axis=1) <= 0) and np.all((i >= cfg.L_h) & (i < cfg.L_h + L))
    assert all(len(set(r.tolist())) == k for r in i)
