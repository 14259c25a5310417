"""-m gpu parity of the sparse tail (haste_forward_loss / haste_backward through the C-ABI) against the
fp64 oracle, element by element on the same seeded inputs.

Bars (BASELINE.json north_star): rel-L2 <= 1e-5 per tensor for fp32, <= 5e-3 for bf16; index handling
bit-exact (integer-valued inputs must reproduce the oracle exactly).  Extra gates close the blind spots
of those bars: dY at the positive pairs, dW/db of labels that have positives, the
partial last group on its own, stage-isolated backward at 1e-4.
"""
import numpy as np
import pytest
import torch

from paper_2606_01117_b200 import synth

pytestmark = pytest.mark.gpu

TOL = {"f32": 1e-5, "bf16": 5e-3}


@pytest.fixture(scope="module")
def H():
    from paper_2606_01117_b200 import haste
    return haste


def _rel(oracle, a, ref):
    return oracle.rel_l2(a, ref)


def _check_forward(oracle, out, ref, tol, inp, label_offset=0):
    assert np.isfinite(out["loss"])
    assert abs(out["loss"] - ref["loss"]) <= tol * abs(ref["loss"]), (out["loss"], ref["loss"])
    if "z" in out:
        assert np.all(np.isfinite(out["z"]))
        # logits are fp32 accumulations of exact products: hold them to the fp32 bar even for bf16 storage
        assert _rel(oracle, out["z"], ref["z"]) <= 1e-5
    assert np.all(np.isfinite(out["dY"]))
    assert _rel(oracle, out["dY"], ref["dY"]) <= tol
    # gate (i): dY at the positive (row,label) pairs only
    B, L = ref["dY"].shape
    rows, labs = [], []
    for i in range(B):
        for p in range(inp.rowptr[i], inp.rowptr[i + 1]):
            l = int(inp.col[p]) - label_offset
            if 0 <= l < L:
                rows.append(i)
                labs.append(l)
    if rows:
        assert _rel(oracle, out["dY"][rows, labs], ref["dY"][rows, labs]) <= tol


def _check_backward(oracle, out, ref, tol, G):
    for k in ("dW", "db", "dX"):
        if ref.get(k) is None or out.get(k) is None:
            continue
        assert np.all(np.isfinite(out[k])), k
        assert _rel(oracle, out[k], ref[k]) <= tol, (k, _rel(oracle, out[k], ref[k]))
    L = ref["dW"].shape[0]
    last = (L - 1) // G * G
    assert _rel(oracle, out["dW"][last:], ref["dW"][last:]) <= tol   # partial last group on its own


SMALL = [
    # B, d, L, G, K, dtype, sorted_distinct, bias
    (32, 128, 4096, 16, 32, "f32", True, False),      # BASELINE config 1 shape
    (7, 40, 50, 3, 5, "f32", False, True),            # odd everything, unsorted + duplicated idx (R4)
    (33, 64, 130, 16, 8, "f32", True, True),          # ragged batch tile and last group
    (16, 32, 19, 1, 12, "f32", True, True),           # G = 1: per-label fixed fan-in
    (9, 24, 40, 8, 24, "f32", True, False),           # K = d: dense layer
    (64, 128, 64 * 5 + 11, 64, 64, "bf16", True, True),
    (130, 256, 32 * 9 + 7, 32, 64, "bf16", True, False),
    (200, 300, 32 * 8 + 5, 32, 64, "bf16", True, True),      # odd number of groups: the paired dW kernel has an unpaired last group
    (256, 256, 128 * 3 + 5, 128, 128, "bf16", True, True),
    (512, 768, 64 * 40 + 11, 64, 128, "bf16", True, True),   # config-3 tile shape, several tiles, ragged tail
    (100, 200, 64 * 3 + 1, 64, 24, "bf16", False, True),     # shape outside the tensor-core family
    (130, 256, 16 * 19 + 5, 16, 64, "bf16", True, True),     # narrow groups on the tensor cores: G = 16 ...
    (300, 384, 16 * 40 + 9, 16, 128, "bf16", True, False),
    (200, 256, 8 * 37 + 3, 8, 64, "bf16", True, True),       # ... and G = 8 (MMA N = 16, half of it unused)
    (129, 512, 8 * 50 + 1, 8, 128, "bf16", False, True),     # unsorted idx rows: dX takes the L2 path for every slot
]


@pytest.mark.parametrize("force_simt", [False, True])
@pytest.mark.parametrize("case", SMALL, ids=lambda c: "B%d_d%d_L%d_G%d_K%d_%s_%s" % (c[0], c[1], c[2], c[3], c[4], c[5], "sd" if c[6] else "any"))
def test_small_cases(oracle, H, case, force_simt):
    from gpu_util import TailRun
    B, d, L, G, K, dt, sd, with_bias = case
    inp = synth.small_case(11 + B + L, B, d, L, G, K, dtype=dt, n_pos=3, sorted_distinct=sd, with_bias=with_bias,
                           w_std=0.5 if dt == "f32" else 0.05)
    flags = (H.HASTE_FORCE_SIMT if force_simt else 0) | (H.HASTE_IDX_SORTED_DISTINCT if sd else 0)
    run = TailRun(inp, G, flags=flags)
    if force_simt:
        assert run.layer.kernel_family == 0
    out = run.forward()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G)
    _check_forward(oracle, out, ref, TOL[dt], inp)
    bout = run.backward()
    # the oracle's backward consumes the oracle's own fp64 dY (end-to-end bar) ...
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], G)
    _check_backward(oracle, bout, bref, TOL[dt], G)
    assert run.fwd_launches > 0 and run.bwd_launches > 0


@pytest.mark.parametrize("force_simt", [False, True])
def test_stage_isolated_backward(oracle, H, force_simt):
    """P11: feed haste_backward the oracle's dY rounded to bf16; compare with the oracle run on that
    rounded dY.  Only accumulation order and the bf16 rounding of dW remain, so the gate is tight."""
    from gpu_util import TailRun, dy_rounded
    B, d, L, G, K = 256, 256, 64 * 9 + 11, 64, 128
    inp = synth.small_case(5, B, d, L, G, K, dtype="bf16", w_std=0.05)
    run = TailRun(inp, G, flags=(H.HASTE_FORCE_SIMT if force_simt else 0) | H.HASTE_IDX_SORTED_DISTINCT, dw_dtype="f32")
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G)
    dYr = dy_rounded(inp, ref["dY"])
    out = run.backward(dY_BL=dYr)
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, dYr.astype(np.float64), G)
    for k in ("dW", "db", "dX"):
        assert oracle.rel_l2(out[k], bref[k]) <= 1e-4, (k, oracle.rel_l2(out[k], bref[k]))


@pytest.mark.parametrize("force_simt", [False, True])
@pytest.mark.parametrize("shape", [(64, 96, 64 * 3 + 5, 64, 64), (40, 64, 77, 8, 16), (128, 256, 32 * 5 + 3, 32, 64),
                                   (200, 128, 16 * 9 + 3, 16, 64), (130, 256, 8 * 21 + 5, 8, 128)])
def test_integer_exactness(oracle, H, shape, force_simt):
    """P7: small-integer X, W, dY (exact in bf16, every partial sum < 2^24): logits, dW and dX must
    equal the oracle EXACTLY whatever the accumulation or atomic order -- gather/scatter addressing
    is bit-exact."""
    from gpu_util import TailRun
    B, d, L, G, K = shape
    inp = synth.small_case(3, B, d, L, G, K, dtype="bf16", with_bias=False)
    rng = np.random.RandomState(1)
    Xi = rng.randint(-4, 5, size=(B, d)).astype(np.float32)
    Xi[: min(B, d)] = 0
    Xi[np.arange(min(B, d)), np.arange(min(B, d))] = 1.0          # one-hot rows: the logit names the feature read
    Wi = rng.randint(-4, 5, size=(L, K)).astype(np.float32)
    inp.X, inp.W = Xi, Wi
    inp.bits["X"], inp.bits["W"] = synth.round_bf16(Xi)[0].reshape(B, d), synth.round_bf16(Wi)[0].reshape(L, K)
    run = TailRun(inp, G, flags=(H.HASTE_FORCE_SIMT if force_simt else 0) | H.HASTE_IDX_SORTED_DISTINCT, dw_dtype="f32")
    out = run.forward()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, G)
    assert np.array_equal(out["z"].astype(np.float64), ref["z"])
    dYi = rng.randint(-3, 4, size=(B, L)).astype(np.float32)
    bout = run.backward(dY_BL=dYi)
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, dYi.astype(np.float64), G)
    assert np.array_equal(bout["dW"].astype(np.float64), bref["dW"])
    assert np.array_equal(bout["dX"].astype(np.float64), bref["dX"])
    assert np.array_equal(bout["db"].astype(np.float64), bref["db"])


@pytest.mark.parametrize("force_simt", [False, True])
def test_saturation_and_bias(oracle, H, force_simt):
    """Large |z| (W x50, bias +-100 on a few labels): softplus/sigmoid branches that the synthetic
    N(0,0.02^2) weights never reach.  Outputs finite, parity holds."""
    from gpu_util import TailRun
    B, d, L, G, K = 128, 128, 64 * 4 + 9, 64, 64
    inp = synth.small_case(17, B, d, L, G, K, dtype="bf16", w_std=1.0, with_bias=True)
    inp.bias[::7] = 100.0
    inp.bias[3::11] = -100.0
    run = TailRun(inp, G, flags=(H.HASTE_FORCE_SIMT if force_simt else 0) | H.HASTE_IDX_SORTED_DISTINCT)
    out = run.forward()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G)
    _check_forward(oracle, out, ref, 5e-3, inp)
    bout = run.backward()
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], G)
    _check_backward(oracle, bout, bref, 5e-3, G)


@pytest.mark.parametrize("force_simt", [False, True])
def test_label_offset_filter_and_loss_scale(oracle, H, force_simt):
    """One CSR over global ids serves head and tail: ids outside [offset, offset+L) are ignored (R7);
    loss_scale given explicitly is used as is (R1)."""
    from gpu_util import TailRun
    B, d, L, G, K, off = 64, 128, 64 * 6 + 3, 64, 64, 1000
    inp = synth.small_case(23, B, d, L, G, K, dtype="bf16", n_pos=6, w_std=0.05, label_offset=off, L_total=off + L + 500)
    run = TailRun(inp, G, flags=(H.HASTE_FORCE_SIMT if force_simt else 0), label_offset=off, loss_scale=0.25)
    out = run.forward()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G, label_offset=off, s=0.25)
    _check_forward(oracle, out, ref, 5e-3, inp, label_offset=off)
    inside = ((inp.col >= off) & (inp.col < off + L)).sum()
    assert 0 < inside < inp.col.size


@pytest.mark.parametrize("force_simt", [False, True])
def test_targets_heavy_rows(oracle, H, force_simt):
    """Many positives per row and per group (every group has positives; some rows hold dozens)."""
    from gpu_util import TailRun
    B, d, L, G, K = 128, 128, 64 * 8, 64, 64
    inp = synth.small_case(29, B, d, L, G, K, dtype="bf16", n_pos=60, w_std=0.05)
    run = TailRun(inp, G, flags=(H.HASTE_FORCE_SIMT if force_simt else 0))
    out = run.forward()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G)
    _check_forward(oracle, out, ref, 5e-3, inp)


def test_accumulate_dx_and_batch_smaller_than_bmax(oracle, H):
    from gpu_util import TailRun
    B, d, L, G, K = 48, 64, 100, 16, 16
    inp = synth.small_case(31, B, d, L, G, K, dtype="f32")
    run = TailRun(inp, G, B_max=200)
    out = run.forward()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G)
    _check_forward(oracle, out, ref, 1e-5, inp)
    base = np.arange(B * d, dtype=np.float32).reshape(B, d) / 100.0
    bout = run.backward(accumulate_into=base)
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], G)
    assert oracle.rel_l2(bout["dX"] - base, bref["dX"]) <= 1e-4


def test_empty_and_degenerate(H):
    dev = torch.device("cuda:0")
    layer = H.HasteLayer(16, 0, 4, 8, 8, "f32")            # no labels
    loss = torch.full((1,), 7.0, device=dev)
    X = torch.zeros(8, 16, device=dev)
    idx = torch.zeros(1, 8, dtype=torch.int32, device=dev)
    W = torch.zeros(1, 8, device=dev)
    layer.forward_loss(8, X, idx, W, None, None, None, loss=loss, dY=None)
    assert loss.item() == 0.0
    layer2 = H.HasteLayer(16, 12, 4, 8, 8, "f32")          # B = 0
    loss.fill_(7.0)
    layer2.forward_loss(0, X, idx, W, None, None, None, loss=loss, dY=None)
    assert loss.item() == 0.0
    with pytest.raises(H.HasteError) as ei:
        layer2.forward_loss(9, X, idx, W, None, None, None, loss=loss, dY=None)   # B > B_max
    assert ei.value.status == H.HASTE_ERR_INVALID_ARG


def test_validate_index(H):
    dev = torch.device("cuda:0")
    layer = H.HasteLayer(16, 8, 4, 4, 8, "f32", flags=H.HASTE_IDX_SORTED_DISTINCT)
    good = torch.tensor([[0, 3, 7, 15], [1, 2, 3, 4]], dtype=torch.int32, device=dev)
    layer.validate_index(good)
    for bad in ([[0, 3, 7, 16], [1, 2, 3, 4]], [[0, 3, 3, 15], [1, 2, 3, 4]], [[-1, 3, 7, 15], [1, 2, 3, 4]]):
        with pytest.raises(H.HasteError) as ei:
            layer.validate_index(torch.tensor(bad, dtype=torch.int32, device=dev))
        assert ei.value.status == H.HASTE_ERR_BAD_INDEX


def test_w_zero_closed_form(H):
    """P5 on the GPU: W = 0, b = 0 -> loss = s*B*L*ln2 exactly (to fp32), dY = s*(1/2 - y)."""
    from gpu_util import TailRun
    B, d, L, G, K = 64, 128, 64 * 5, 64, 64
    inp = synth.small_case(37, B, d, L, G, K, dtype="bf16", with_bias=False)
    inp.W[:] = 0
    inp.bits["W"][:] = 0
    out = TailRun(inp, G).forward()
    assert abs(out["loss"] - L * np.log(2.0)) <= 1e-5 * L * np.log(2.0)
    Y = np.zeros((B, L))
    for i in range(B):
        Y[i, inp.col[inp.rowptr[i]:inp.rowptr[i + 1]]] = 1
    assert np.allclose(out["dY"], (0.5 - Y) / B, rtol=0, atol=1e-7)


@pytest.mark.parametrize("force_simt", [False, True])
def test_trained_regime_confident_negatives(oracle, H, force_simt):
    """The regime of a trained XMC layer: almost every logit is a confident negative (z in [-12, -4], sigma 1e-5 .. 2e-2),
    a few labels are confident positives.  dY = s sigma(z) and the loss terms ln(1 + e^z) are then tiny numbers, and an
    evaluation of sigma with a fixed ABSOLUTE error (1/2 + 1/2 tanh.approx: 2.4e-4) is wrong by multiples of their
    value.  Gate: ELEMENTWISE relative error of dY (bf16 rounding 2^-9 plus the approximation), the loss by relative
    error, and the backward from the kernel's own dY."""
    from gpu_util import TailRun
    B, d, L, G, K = 256, 128, 64 * 9 + 5, 64, 64
    inp = synth.small_case(61, B, d, L, G, K, dtype="bf16", w_std=0.02, with_bias=True, n_pos=4)
    rng = np.random.RandomState(3)
    inp.bias = rng.uniform(-12.0, -4.0, size=L).astype(np.float32)
    inp.bias[5::97] = 6.0                                   # a few confident positives
    inp.bias[11::101] = -1.0                                # and some labels in the middle (both evaluations inside one group)
    run = TailRun(inp, G, flags=(H.HASTE_FORCE_SIMT if force_simt else 0) | H.HASTE_IDX_SORTED_DISTINCT)
    out = run.forward()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G)
    assert np.all((ref["z"] < -3.0) | (ref["z"] > -2.4))
    assert abs(out["loss"] - ref["loss"]) <= 1e-3 * abs(ref["loss"]), (out["loss"], ref["loss"])
    rel = np.abs(out["dY"] - ref["dY"]) / np.abs(ref["dY"])
    assert rel.max() <= 6e-3, (rel.max(), np.unravel_index(rel.argmax(), rel.shape))
    assert np.all(np.sign(out["dY"]) == np.sign(ref["dY"]))
    neg = ref["z"] < -3.0
    assert oracle.rel_l2(out["dY"][neg], ref["dY"][neg]) <= 5e-3           # the confident negatives on their own
    bout = run.backward()
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], G)
    _check_backward(oracle, bout, bref, 5e-3, G)


@pytest.mark.parametrize("shape", [(300, 768, 64 * 23 + 11, 64, 128), (130, 256, 32 * 9 + 5, 32, 64), (64, 512, 128 * 5 + 3, 128, 128),
                                   (200, 256, 16 * 30 + 7, 16, 64), (130, 384, 8 * 50 + 3, 8, 128)])
@pytest.mark.parametrize("with_bias", [False, True])
def test_forward_logits_only(oracle, H, shape, with_bias):
    """haste_forward_logits: z = bias + sum_j W[l,j] X[i, idx[l/G, j]] rounded once to bf16, in the library
    layout; padding labels of the last group are written as zero; nothing else is needed (no targets)."""
    from gpu_util import TailRun
    B, d, L, G, K = shape
    inp = synth.small_case(70 + B, B, d, L, G, K, dtype="bf16", with_bias=with_bias, w_std=0.2)
    run = TailRun(inp, G, want_logits=False)
    assert run.layer.kernel_family == 1
    Z = run.layer.alloc_dy(B)
    Z.fill_(float("nan"))
    run.layer.forward_logits(B, run.X, run.idx, run.W, run.bias, Z)
    zf = torch.empty(B, L, device=Z.device)
    run.layer.dy_unpack(B, Z, zf)
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G)["z"]
    want = synth.round_bf16(ref.astype(np.float32))[1].reshape(B, L)          # the fp64 logits rounded once to bf16
    got = zf.cpu().numpy()
    # fp32 accumulation before the rounding can move a value across a bf16 rounding boundary: allow one bf16 step there
    assert np.max(np.abs(got - want) / np.maximum(np.abs(want), 1e-3)) <= 2.0 ** -7
    assert oracle.rel_l2(got, ref) <= 3e-3
    NG = -(-L // G)
    if NG * G > L:
        assert torch.count_nonzero(Z.view(NG, B, G)[NG - 1, :, L - (NG - 1) * G:]).item() == 0


def test_xt_from_forward_flag(oracle, H):
    """HASTE_XT_FROM_FORWARD: the backward reuses the forward's transposed copy of X (same handle, same X and B); results
    are those of the default path, bit for bit (dW, db) -- and the default path does not depend on an earlier forward."""
    from gpu_util import TailRun
    B, d, L, G, K = 200, 256, 64 * 7 + 9, 64, 64
    inp = synth.small_case(83, B, d, L, G, K, dtype="bf16", w_std=0.05)
    a = TailRun(inp, G, flags=H.HASTE_XT_FROM_FORWARD, dw_dtype="f32")
    fa = a.forward()
    ba = a.backward()
    b = TailRun(inp, G, dw_dtype="f32")
    fb = b.forward()
    bb = b.backward()
    assert np.array_equal(fa["dY"], fb["dY"])
    assert np.array_equal(ba["dW"], bb["dW"]) and np.array_equal(ba["db"], bb["db"])
    assert a.bwd_launches == b.bwd_launches - 1
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G)
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], G)
    _check_backward(oracle, ba, bref, 5e-3, G)
    # default path: a backward after a forward with ANOTHER X on the same handle still uses its own X
    inp2 = synth.small_case(84, B, d, L, G, K, dtype="bf16", w_std=0.05)
    from gpu_util import to_dev
    b.layer.forward_loss(B, to_dev(inp2, "X"), b.idx, b.W, b.bias, b.rowptr, b.col, loss=None, dY=b.layer.alloc_dy(B))
    bb2 = b.backward()
    assert np.array_equal(bb2["dW"], bb["dW"])


@pytest.mark.parametrize("shape", [(5000, 256, 64 * 37 + 5, 64, 64), (4100, 192, 16 * 90 + 3, 16, 64), (20000, 128, 32 * 9, 32, 64)],
                         ids=lambda s: "B%d_d%d_L%d_G%d_K%d" % s)
def test_large_batch(oracle, H, shape):
    """Batches of many 128-row tiles: 40 tile pairs in the forward, 40 and 33 batch tiles x few group stripes in dX, and
    (B = 20000) more batch tiles than SMs, where the tcgen05 dX kernel declines and the CUDA-core one runs; the transposes'
    grids span several waves (they release their dependent kernel only when the last wave runs)."""
    from gpu_util import TailRun
    B, d, L, G, K = shape
    inp = synth.small_case(9, B, d, L, G, K, dtype="bf16", with_bias=True, w_std=0.05)
    run = TailRun(inp, G, flags=H.HASTE_IDX_SORTED_DISTINCT)
    assert run.layer.kernel_family == 1
    out = run.forward()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, inp.bias, inp.rowptr, inp.col, G)
    _check_forward(oracle, out, ref, TOL["bf16"], inp)
    bout = run.backward()
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], G)
    _check_backward(oracle, bout, bref, TOL["bf16"], G)
