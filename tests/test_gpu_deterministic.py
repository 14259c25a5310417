"""-m gpu: HASTE_DETERMINISTIC (include/haste.h) -- dX without float atomics.  The sparse tail's dX kernel then accumulates into
private per-CTA tiles with one writer per word and the tiles are summed in stripe order; the dense head's dX uses one label
slab.  Gates: bit-identical results from run to run, exact agreement with the fp64 oracle on integer inputs (which also
covers unsorted / duplicated index rows and several groups per CTA), closeness on real inputs, and a clean refusal
where no atomic-free kernel exists."""
import numpy as np
import pytest
import torch

from paper_2606_01117_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("shape", [(300, 768, 64 * 700 + 3, 64, 128), (200, 1024, 64 * 300 + 9, 64, 64), (130, 768, 32 * 401, 32, 64),
                                   (200, 768, 16 * 500 + 3, 16, 64), (130, 512, 8 * 700 + 1, 8, 128)])
def test_tail_dx_deterministic(oracle, shape):
    from paper_2606_01117_b200 import haste
    from gpu_util import TailRun, dy_rounded
    B, d, L, G, K = shape
    inp = synth.small_case(9 + B, B, d, L, G, K, dtype="bf16", with_bias=False, w_std=0.05)
    rng = np.random.RandomState(B)
    inp.idx[3] = np.sort(rng.choice(d, size=K, replace=True))      # duplicates -> the group takes the (now plain) L path
    inp.idx[5] = rng.permutation(d)[:K]                            # unsorted
    Wi = rng.randint(-4, 5, size=(L, K)).astype(np.float32)
    dYi = rng.randint(-3, 4, size=(B, L)).astype(np.float32)
    inp.W = Wi
    inp.bits["W"] = synth.round_bf16(Wi)[0].reshape(L, K)
    run = TailRun(inp, G, flags=haste.HASTE_DETERMINISTIC, dw_dtype="f32")
    assert run.layer.kernel_family == 1
    out = run.backward(dY_BL=dYi)
    ref = oracle.tail_backward(inp.X, inp.idx, inp.W, dYi.astype(np.float64), G)
    assert np.array_equal(out["dX"].astype(np.float64), ref["dX"])
    # real values: bit-identical from run to run, and close to the oracle
    Wr = (rng.standard_normal((L, K)) * 0.05).astype(np.float32)
    bits, Wr = synth.round_bf16(Wr)
    inp.W, inp.bits["W"] = Wr.reshape(L, K), bits.reshape(L, K)
    dYq = dy_rounded(inp, (rng.standard_normal((B, L)) / B).astype(np.float32))
    run = TailRun(inp, G, flags=haste.HASTE_DETERMINISTIC, dw_dtype="f32")
    a = run.backward(dY_BL=dYq)["dX"]
    for _ in range(3):
        b = run.backward(dY_BL=dYq)["dX"]
        assert np.array_equal(a.view(np.uint32), b.view(np.uint32))
    ref = oracle.tail_backward(inp.X, inp.idx, inp.W, dYq.astype(np.float64), G)
    assert oracle.rel_l2(a, ref["dX"]) <= 1e-4
    # and the default (atomic) path agrees with it to accumulation order
    c = TailRun(inp, G, dw_dtype="f32").backward(dY_BL=dYq)["dX"]
    assert oracle.rel_l2(c, a.astype(np.float64)) <= 1e-5


def test_deterministic_refused_without_atomic_free_kernel():
    from paper_2606_01117_b200 import haste
    with pytest.raises(haste.HasteError) as e:
        haste.HasteLayer(128, 4096, 16, 32, 32, "f32", flags=haste.HASTE_DETERMINISTIC)     # config 1: CUDA-core family only
    assert e.value.status == haste.HASTE_ERR_UNSUPPORTED


def test_head_dx_deterministic(oracle):
    """dX_h = dY_h W_h without float atomics: bit-identical from run to run, and equal to the oracle's
    head_backward on the same seeded bf16 inputs to accumulation order."""
    from paper_2606_01117_b200 import haste
    dev = torch.device("cuda:0")
    B, d, Lh = 512, 768, 4096
    seed = 77
    Xb, X = synth.round_bf16(synth.normal(seed, synth.STREAM_XHEAD, B * d).astype(np.float32))
    Wb, W = synth.round_bf16((synth.normal(seed, synth.STREAM_WHEAD, Lh * d) * 0.05).astype(np.float32))
    dYb, dYv = synth.round_bf16((synth.normal(seed, synth.STREAM_BIAS_HEAD, B * Lh) / B).astype(np.float32))
    X, W, dYv = X.reshape(B, d), W.reshape(Lh, d), dYv.reshape(B, Lh)

    def dv(bits, shape):
        return torch.from_numpy(np.ascontiguousarray(bits.reshape(shape)).view(np.int16)).to(dev).view(torch.bfloat16)

    Xd, Wd, dYd = dv(Xb, (B, d)), dv(Wb, (Lh, d)), dv(dYb, (B, Lh))
    head = haste.HasteHead(d, Lh, B, "bf16", flags=haste.HASTE_DETERMINISTIC)
    outs = []
    for _ in range(3):
        dX = torch.full((B, d), float("nan"), device=dev)
        head.backward(B, Xd, Wd, dYd, dWh=None, dX=dX)
        outs.append(dX.cpu().numpy())
    assert np.array_equal(outs[0].view(np.uint32), outs[1].view(np.uint32)) and np.array_equal(outs[0].view(np.uint32), outs[2].view(np.uint32))
    ref = oracle.head_backward(X, W, dYv.astype(np.float64))
    assert oracle.rel_l2(outs[0], ref["dX"]) <= 1e-5
