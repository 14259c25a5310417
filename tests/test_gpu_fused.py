"""-m gpu: haste_forward_loss_dw (include/haste.h, first slice) against the oracle, element by element
through the C ABI: loss, dY, dW and db of ONE kernel (forward + fused BCE + weight gradient, tc_fused.cu) must be what
the oracle's forward and backward give -- and what haste_forward_loss followed by haste_backward give: dY bit for bit (the
same arithmetic), the loss up to the order of its partial sums, dW up to the order the batch is accumulated in."""
import numpy as np
import pytest
import torch

from paper_2606_01117_b200 import synth

pytestmark = pytest.mark.gpu

SHAPES = [
    # B, d, L, G, K, dw_dtype, bias
    (512, 768, 64 * 300 + 11, 64, 128, "bf16", True),     # config-3 tile shape: 4 batch tiles, ~2 groups per CTA, ragged last group
    (300, 256, 64 * 40 + 5, 64, 64, "f32", False),        # 3 tiles, the last one ragged; K = 64; fp32 dW
    (128, 384, 64 * 500 + 1, 64, 128, "f32", True),       # one tile; several groups per CTA (both D_w buffers, both tile parities)
    (256, 256, 64 * 450 + 3, 64, 64, "bf16", True),       # two tiles, three groups per CTA
    (33, 128, 64 * 3, 64, 64, "bf16", True),              # fewer groups than SMs, one partial tile
    (200, 256, 32 * 20 + 3, 32, 64, "bf16", True),        # a shape the fused kernel does not cover: the two kernels run
    (600, 256, 64 * 9 + 3, 64, 128, "bf16", False),       # B > 512: the two kernels run
]


@pytest.mark.parametrize("shape", SHAPES, ids=lambda s: "B%d_d%d_L%d_G%d_K%d_%s_%s" % (s[0], s[1], s[2], s[3], s[4], s[5], "bias" if s[6] else "nobias"))
def test_forward_loss_dw(oracle, shape):
    from paper_2606_01117_b200 import haste
    from gpu_util import dev, to_dev, t32
    B, d, L, G, K, dwt, with_bias = shape
    inp = synth.small_case(41 + B, B, d, L, G, K, dtype="bf16", n_pos=4, with_bias=with_bias, w_std=0.05)
    layer = haste.HasteLayer(d, L, G, K, B, "bf16", dw_dtype=dwt, flags=haste.HASTE_IDX_SORTED_DISTINCT)
    assert layer.kernel_family == 1
    X, W, idx, bias = to_dev(inp, "X"), to_dev(inp, "W"), t32(inp.idx), t32(inp.bias)
    rowptr, col = t32(inp.rowptr), t32(inp.col)
    tdt = torch.bfloat16 if dwt == "bf16" else torch.float32

    def run(fused):
        loss = torch.full((1,), float("nan"), device=dev())
        dY = layer.alloc_dy(B); dY.fill_(float("nan"))
        dW = torch.full((L, K), float("nan"), dtype=tdt, device=dev())
        db = torch.full((L,), float("nan"), device=dev())
        if fused:
            layer.forward_loss_dw(B, X, idx, W, bias, rowptr, col, loss=loss, dY=dY, dW=dW, dbias=db)
            n = layer.last_launch_count
        else:
            layer.forward_loss(B, X, idx, W, bias, rowptr, col, loss=loss, dY=dY)
            layer.backward(B, X, idx, W, dY, dW=dW, dbias=db)
            n = None
        dYf = torch.empty(B, L, device=dev())
        layer.dy_unpack(B, dY, dYf)
        torch.cuda.synchronize()
        return dict(loss=float(loss.item()), dY=dYf.cpu().numpy(), dYraw=dY.clone(), dW=dW.float().cpu().numpy(), db=db.cpu().numpy(), n=n)

    f = run(True)
    if G == 64 and B <= 512:
        assert f["n"] == 2                                    # the transpose and ONE kernel
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G)
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], G)
    assert abs(f["loss"] - ref["loss"]) <= 2e-5 * abs(ref["loss"])
    assert np.all(np.isfinite(f["dY"])) and np.all(np.isfinite(f["dW"])) and np.all(np.isfinite(f["db"]))
    assert oracle.rel_l2(f["dY"], ref["dY"]) <= 5e-3
    assert oracle.rel_l2(f["dW"], bref["dW"]) <= 5e-3
    assert oracle.rel_l2(f["db"], bref["db"]) <= 5e-3
    # dY at the positive pairs only, and the partial last group on its own (where whole-tensor norms are blind)
    rows = np.repeat(np.arange(B), np.diff(inp.rowptr))
    assert oracle.rel_l2(f["dY"][rows, inp.col], ref["dY"][rows, inp.col]) <= 5e-3
    last = (L - 1) // G * G
    assert oracle.rel_l2(f["dW"][last:], bref["dW"][last:]) <= 5e-3
    # against the two separate kernels: dY is the same arithmetic, the loss and dW the same sums in another order
    s = run(False)
    assert torch.equal(f["dYraw"], s["dYraw"])
    assert abs(f["loss"] - s["loss"]) <= 1e-6 * abs(s["loss"])
    assert oracle.rel_l2(f["dW"], s["dW"]) <= (1e-5 if dwt == "f32" else 3e-3)
    assert oracle.rel_l2(f["db"], s["db"]) <= 1e-5


def test_forward_loss_dw_exact_sums(oracle):
    """Exactness where it exists: W = 0, b = 0 and a power-of-two loss scale give dY = s/2 - s y exactly in bf16, and with
    small-integer X the weight gradient dW = dY^T H and db = dY^T 1 are sums of exact products below 2^24: the fused kernel
    must reproduce the oracle's dW and db EXACTLY, whatever its accumulation order (operand addressing through both
    descriptors of the shared H image, the ones rows, the zeroed rows past the batch)."""
    from paper_2606_01117_b200 import haste
    from gpu_util import dev, t32
    B, d, L, G, K = 300, 128, 64 * 150 + 7, 64, 64
    inp = synth.small_case(5, B, d, L, G, K, dtype="bf16", n_pos=3, with_bias=False)
    rng = np.random.RandomState(2)
    Xi = rng.randint(-4, 5, size=(B, d)).astype(np.float32)
    Wz = np.zeros((L, K), dtype=np.float32)
    layer = haste.HasteLayer(d, L, G, K, B, "bf16", dw_dtype="f32", loss_scale=2.0 ** -6, flags=haste.HASTE_IDX_SORTED_DISTINCT)
    X = torch.from_numpy(Xi).to(dev()).to(torch.bfloat16)
    W = torch.zeros(L, K, dtype=torch.bfloat16, device=dev())
    idx, rowptr, col = t32(inp.idx), t32(inp.rowptr), t32(inp.col)
    loss = torch.zeros(1, device=dev())
    dY = layer.alloc_dy(B)
    dW = torch.full((L, K), float("nan"), device=dev())
    db = torch.full((L,), float("nan"), device=dev())
    layer.forward_loss_dw(B, X, idx, W, None, rowptr, col, loss=loss, dY=dY, dW=dW, dbias=db)
    torch.cuda.synchronize()
    assert layer.last_launch_count == 2
    ref = oracle.tail_forward(Xi.astype(np.float64), inp.idx, Wz.astype(np.float64), None, inp.rowptr, inp.col, G, s=2.0 ** -6)
    bref = oracle.tail_backward(Xi.astype(np.float64), inp.idx, Wz.astype(np.float64), ref["dY"], G)
    assert np.array_equal(dW.cpu().numpy().astype(np.float64), bref["dW"])
    assert np.array_equal(db.cpu().numpy().astype(np.float64), bref["db"])


def test_forward_loss_dw_heavy_rows_and_trained_regime(oracle):
    """Rows with many positives (the per-tile target cursors walk) and confident logits (the wide sigmoid evaluation) through
    the fused kernel."""
    from paper_2606_01117_b200 import haste
    from gpu_util import dev, to_dev, t32
    B, d, L, G, K = 260, 256, 64 * 160 + 9, 64, 128
    inp = synth.small_case(77, B, d, L, G, K, dtype="bf16", n_pos=40, with_bias=True, w_std=0.05)
    inp.bias = (inp.bias - 7.0).astype(np.float32)              # logits around -7: sigma ~ 1e-3
    layer = haste.HasteLayer(d, L, G, K, B, "bf16", dw_dtype="f32")
    X, W, idx, bias = to_dev(inp, "X"), to_dev(inp, "W"), t32(inp.idx), t32(inp.bias)
    rowptr, col = t32(inp.rowptr), t32(inp.col)
    loss = torch.zeros(1, device=dev()); dY = layer.alloc_dy(B)
    dW = torch.empty(L, K, device=dev()); db = torch.empty(L, device=dev())
    layer.forward_loss_dw(B, X, idx, W, bias, rowptr, col, loss=loss, dY=dY, dW=dW, dbias=db)
    dYf = torch.empty(B, L, device=dev())
    layer.dy_unpack(B, dY, dYf)
    torch.cuda.synchronize()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G)
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], G)
    got = dYf.cpu().numpy().astype(np.float64)
    assert abs(float(loss.item()) - ref["loss"]) <= 2e-5 * abs(ref["loss"])
    neg = np.ones((B, L), dtype=bool)
    rows = np.repeat(np.arange(B), np.diff(inp.rowptr))
    neg[rows, inp.col] = False
    rel = np.abs(got[neg] - ref["dY"][neg]) / np.abs(ref["dY"][neg])
    assert rel.max() <= 6e-3, rel.max()                          # elementwise: bf16 rounding of dY, no tanh.approx error
    assert oracle.rel_l2(got[rows, inp.col], ref["dY"][rows, inp.col]) <= 5e-3
    assert oracle.rel_l2(dW.cpu().numpy(), bref["dW"]) <= 5e-3
    assert oracle.rel_l2(db.cpu().numpy(), bref["db"]) <= 5e-3


def test_forward_loss_dw_optional_arguments(oracle):
    """dW alone, db alone, no loss, no targets, a label offset: each output must be what the full call gives."""
    from paper_2606_01117_b200 import haste
    from gpu_util import dev, to_dev, t32
    B, d, L, G, K, off = 200, 256, 64 * 170 + 3, 64, 128, 5000
    inp = synth.small_case(9, B, d, L, G, K, dtype="bf16", n_pos=4, with_bias=True, w_std=0.05)
    col = (inp.col + off).astype(np.int32)
    layer = haste.HasteLayer(d, L, G, K, B, "bf16", dw_dtype="f32", label_offset=off)
    X, W, idx, bias = to_dev(inp, "X"), to_dev(inp, "W"), t32(inp.idx), t32(inp.bias)
    rowptr, colt = t32(inp.rowptr), t32(col)

    def call(want_loss=True, want_dw=True, want_db=True, targets=True):
        loss = torch.full((1,), float("nan"), device=dev()) if want_loss else None
        dY = layer.alloc_dy(B)
        dW = torch.full((L, K), float("nan"), device=dev()) if want_dw else None
        db = torch.full((L,), float("nan"), device=dev()) if want_db else None
        layer.forward_loss_dw(B, X, idx, W, bias, rowptr if targets else None, colt if targets else None, loss=loss, dY=dY, dW=dW, dbias=db)
        torch.cuda.synchronize()
        return loss, dY, dW, db

    loss, dY, dW, db = call()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, col, G, label_offset=off)
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], G)
    assert abs(float(loss.item()) - ref["loss"]) <= 2e-5 * abs(ref["loss"])
    assert oracle.rel_l2(dW.cpu().numpy(), bref["dW"]) <= 5e-3 and oracle.rel_l2(db.cpu().numpy(), bref["db"]) <= 5e-3
    l2, dY2, dW2, db2 = call(want_loss=False, want_db=False)
    assert db2 is None and torch.equal(dY2, dY) and torch.equal(dW2, dW)
    l3, dY3, dW3, db3 = call(want_dw=False)
    assert dW3 is None and torch.equal(dY3, dY) and torch.equal(db3, db) and float(l3.item()) == float(loss.item())
    # no targets: every label is a negative
    l4, dY4, dW4, db4 = call(targets=False)
    ref4 = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, np.zeros(B + 1, dtype=np.int32), np.zeros(0, dtype=np.int32), G)
    bref4 = oracle.tail_backward(inp.X, inp.idx, inp.W, ref4["dY"], G)
    assert abs(float(l4.item()) - ref4["loss"]) <= 2e-5 * abs(ref4["loss"])
    assert oracle.rel_l2(dW4.cpu().numpy(), bref4["dW"]) <= 5e-3 and oracle.rel_l2(db4.cpu().numpy(), bref4["db"]) <= 5e-3
