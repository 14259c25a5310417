"""-m gpu parity of the dense head (haste_head_forward_loss / haste_head_backward)
against the fp64 oracle."""
import numpy as np
import pytest
import torch

from paper_2606_01117_b200 import synth

pytestmark = pytest.mark.gpu


def _case(seed, B, d, Lh, dtype, with_bias, n_pos=4, w_std=0.05, L_total=None):
    X = synth.normal(seed, synth.STREAM_XHEAD, B * d).astype(np.float32).reshape(B, d)
    W = (synth.normal(seed, synth.STREAM_WHEAD, Lh * d) * w_std).astype(np.float32).reshape(Lh, d)
    bits = {}
    if dtype == "bf16":
        bits["X"], X = synth.round_bf16(X)
        bits["W"], W = synth.round_bf16(W)
        X, W = X.reshape(B, d), W.reshape(Lh, d)
        bits["X"], bits["W"] = bits["X"].reshape(B, d), bits["W"].reshape(Lh, d)
    bias = (synth.normal(seed, synth.STREAM_BIAS_HEAD, Lh) * 0.1).astype(np.float32) if with_bias else None
    rowptr, col = synth.draw_targets(seed, B, L_total or Lh, 0, n_pos, None, n_fixed=min(n_pos, Lh))
    return X, W, bias, rowptr, col, bits


def _dev(a, bits=None):
    dev = torch.device("cuda:0")
    if a is None:
        return None
    if bits is not None:
        return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(dev).view(torch.bfloat16)
    return torch.from_numpy(np.ascontiguousarray(a)).to(dev)


HEAD_CASES = [
    (32, 128, 300, "f32", True), (7, 40, 50, "f32", False),
    (64, 128, 256, "bf16", True), (130, 256, 1000, "bf16", False), (256, 768, 4096, "bf16", True),
    (512, 768, 2048 + 24, "bf16", False), (100, 200, 77, "bf16", True),
]


@pytest.mark.parametrize("force_simt", [False, True])
@pytest.mark.parametrize("case", HEAD_CASES, ids=lambda c: "B%d_d%d_L%d_%s" % c[:4])
def test_head_parity(oracle, case, force_simt):
    from paper_2606_01117_b200 import haste
    B, d, Lh, dt, with_bias = case
    tol = 1e-5 if dt == "f32" else 5e-3
    X, W, bias, rowptr, col, bits = _case(41 + B, B, d, Lh, dt, with_bias, L_total=Lh + 100)
    dev = torch.device("cuda:0")
    head = haste.HasteHead(d, Lh, B, dt, flags=haste.HASTE_FORCE_SIMT if force_simt else 0)
    Xd, Wd = _dev(X, bits.get("X")), _dev(W, bits.get("W"))
    bd, rp, cl = _dev(bias), _dev(rowptr), _dev(col)
    loss = torch.full((1,), float("nan"), device=dev)
    dY = torch.full((B, Lh), float("nan"), dtype=head.tdtype, device=dev)
    z = torch.full((B, Lh), float("nan"), device=dev)
    head.forward_loss(B, Xd, Wd, bd, rp, cl, loss=loss, dY=dY, logits_out=z)
    assert head.last_launch_count > 0
    ref = oracle.head_forward(X, W, bias, rowptr, col)
    assert abs(loss.item() - ref["loss"]) <= tol * abs(ref["loss"])
    assert oracle.rel_l2(z.cpu().numpy(), ref["z"]) <= 1e-5
    dYn = dY.float().cpu().numpy()
    assert np.all(np.isfinite(dYn))
    assert oracle.rel_l2(dYn, ref["dY"]) <= tol
    rows = np.repeat(np.arange(B), np.diff(rowptr))
    keep = col < Lh
    assert keep.any() and not keep.all()
    assert oracle.rel_l2(dYn[rows[keep], col[keep]], ref["dY"][rows[keep], col[keep]]) <= tol
    dW = torch.full((Lh, d), float("nan"), dtype=head.tdtype, device=dev)
    db = torch.full((Lh,), float("nan"), device=dev)
    dX = torch.full((B, d), float("nan"), device=dev)
    head.backward(B, Xd, Wd, dY, dWh=dW, dbias=db, dX=dX)
    bref = oracle.head_backward(X, W, ref["dY"])
    assert oracle.rel_l2(dW.float().cpu().numpy(), bref["dW"]) <= tol
    assert oracle.rel_l2(db.cpu().numpy(), bref["db"]) <= tol
    assert oracle.rel_l2(dX.cpu().numpy(), bref["dX"]) <= tol
    # accumulate_dX adds to the existing contents
    dX2 = torch.ones(B, d, device=dev)
    head.backward(B, Xd, Wd, dY, dWh=None, dbias=None, dX=dX2, accumulate_dX=True)
    assert oracle.rel_l2(dX2.cpu().numpy() - 1.0, bref["dX"]) <= max(tol, 1e-4)


@pytest.mark.parametrize("B,Lh", [(512, 128 * 100), (300, 128 * 120 + 40)])
def test_head_many_tiles_per_cta_heavy_rows(oracle, B, Lh):
    """Several output tiles per CTA and 40 positives per row: the forward epilogue keeps a cursor into each CSR row while
    a CTA's tiles move up in n with a fixed m tile (B = 512: 4 m tiles, 148 % 4 == 0) and resets it when the m tile
    changes from tile to tile (B = 300: 3 m tiles).  dY at the positive pairs is the gate that sees the targets."""
    from paper_2606_01117_b200 import haste
    d = 256
    X, W, bias, rowptr, col, bits = _case(7 + B, B, d, Lh, "bf16", True, n_pos=40, L_total=Lh + 500)
    dev = torch.device("cuda:0")
    head = haste.HasteHead(d, Lh, B, "bf16")
    assert head.kernel_family == 1
    loss = torch.full((1,), float("nan"), device=dev)
    dY = torch.full((B, Lh), float("nan"), dtype=head.tdtype, device=dev)
    head.forward_loss(B, _dev(X, bits["X"]), _dev(W, bits["W"]), _dev(bias), _dev(rowptr), _dev(col), loss=loss, dY=dY)
    ref = oracle.head_forward(X, W, bias, rowptr, col)
    assert abs(loss.item() - ref["loss"]) <= 5e-3 * abs(ref["loss"])
    dYn = dY.float().cpu().numpy()
    assert oracle.rel_l2(dYn, ref["dY"]) <= 5e-3
    rows = np.repeat(np.arange(B), np.diff(rowptr))
    keep = col < Lh
    assert keep.sum() > 30 * B
    assert oracle.rel_l2(dYn[rows[keep], col[keep]], ref["dY"][rows[keep], col[keep]]) <= 5e-3
    # every positive moved dY by -s: a missed or misplaced target shows as an error of the order of s = 1/B
    s = 1.0 / B
    assert np.max(np.abs(dYn[rows[keep], col[keep]] - ref["dY"][rows[keep], col[keep]])) < 0.02 * s
    neg = np.ones((B, Lh), dtype=bool)
    neg[rows[keep], col[keep]] = False
    assert np.max(np.abs(dYn[neg] - ref["dY"][neg])) < 0.02 * s


def test_head_empty():
    from paper_2606_01117_b200 import haste
    dev = torch.device("cuda:0")
    head = haste.HasteHead(16, 0, 8, "f32")
    loss = torch.full((1,), 3.0, device=dev)
    head.forward_loss(8, torch.zeros(8, 16, device=dev), torch.zeros(1, 16, device=dev), None, None, None, loss=loss)
    assert loss.item() == 0.0


@pytest.mark.parametrize("force_simt", [False, True])
def test_head_trained_regime_confident_negatives(oracle, force_simt):
    """Same gate as tests/test_gpu_tail.py::test_trained_regime_confident_negatives for the dense head: logits in
    [-12, -4] with a few confident positives; dY elementwise, loss by relative error."""
    from paper_2606_01117_b200 import haste
    B, d, Lh = 256, 256, 128 * 5 + 24
    X, W, bias, rowptr, col, bits = _case(91, B, d, Lh, "bf16", True, w_std=0.01, L_total=Lh + 50)
    rng = np.random.RandomState(4)
    bias = rng.uniform(-12.0, -4.0, size=Lh).astype(np.float32)
    bias[7::89] = 6.0
    bias[13::83] = -1.0
    dev = torch.device("cuda:0")
    head = haste.HasteHead(d, Lh, B, "bf16", flags=haste.HASTE_FORCE_SIMT if force_simt else 0)
    loss = torch.full((1,), float("nan"), device=dev)
    dY = torch.full((B, Lh), float("nan"), dtype=head.tdtype, device=dev)
    head.forward_loss(B, _dev(X, bits["X"]), _dev(W, bits["W"]), _dev(bias), _dev(rowptr), _dev(col), loss=loss, dY=dY)
    ref = oracle.head_forward(X, W, bias, rowptr, col)
    assert np.all((ref["z"] < -3.0) | (ref["z"] > -2.4))
    assert abs(loss.item() - ref["loss"]) <= 1e-3 * abs(ref["loss"]), (loss.item(), ref["loss"])
    dYn = dY.float().cpu().numpy()
    rel = np.abs(dYn - ref["dY"]) / np.abs(ref["dY"])
    assert rel.max() <= 6e-3, rel.max()
    assert np.all(np.sign(dYn) == np.sign(ref["dY"]))
