"""-m gpu parity of haste_backward_sgd: the SGD-with-momentum step of the output layer (heavy-ball form,
DESIGN.md reading R13) fused into the weight-gradient kernel.  Reference: the oracle's tail_backward (dW, db in fp64 from the
same bf16 dY) followed by the oracle's sgd_momentum.  The momentum is fp32 (compared by relative L2); W is bf16, updated by
one rounding of the fp32 result: it must be the bf16 rounding of the oracle's W' up to one bf16 step where the fp32 value
sits next to a rounding boundary."""
import numpy as np
import pytest
import torch

from paper_2606_01117_b200 import synth

pytestmark = pytest.mark.gpu


def _bf16_step(x):
    """Size of one bf16 step at |x| (8 significant bits)."""
    return 2.0 ** (np.floor(np.log2(np.maximum(np.abs(x), 1e-30))) - 7)


@pytest.mark.parametrize("shape", [(300, 768, 64 * 23 + 11, 64, 128), (130, 256, 32 * 40 + 5, 32, 64), (64, 512, 128 * 5 + 3, 128, 128),
                                   (257, 768, 64 * 200 + 1, 64, 64), (200, 512, 128 * 9, 128, 64),
                                   (130, 256, 32 * 21 + 5, 32, 128), (200, 256, 16 * 50 + 7, 16, 64), (130, 384, 8 * 90 + 3, 8, 128)])
@pytest.mark.parametrize("with_bias", [False, True])
def test_backward_sgd_two_steps(oracle, shape, with_bias):
    from gpu_util import TailRun, dy_rounded
    from paper_2606_01117_b200 import haste
    B, d, L, G, K = shape
    inp = synth.small_case(120 + B, B, d, L, G, K, dtype="bf16", with_bias=with_bias, w_std=0.05)
    run = TailRun(inp, G, want_logits=False)
    assert run.layer.kernel_family == 1
    dev = run.X.device
    lr, mu, wd = 0.5, 0.9, 0.01
    rng = np.random.RandomState(B)
    W_ref = inp.W.astype(np.float64)
    v_ref = rng.standard_normal((L, K)) * 0.01                     # a non-zero momentum buffer to start from
    mom = torch.from_numpy(v_ref.astype(np.float32)).to(dev)
    v_ref = mom.cpu().numpy().astype(np.float64)
    b_ref = None if not with_bias else inp.bias.astype(np.float64)
    vb_ref = None if not with_bias else np.zeros(L)
    bias = None if not with_bias else run.bias.clone()
    bmom = None if not with_bias else torch.zeros(L, device=dev)
    W = run.W.clone()
    for step in range(2):
        # the same dY on both sides: the kernel's own forward output would do, a seeded one isolates this call
        dYq = dy_rounded(inp, (np.random.RandomState(step + 7).standard_normal((B, L)) / B).astype(np.float32))
        dY = run.layer.alloc_dy(B)
        run.layer.dy_pack(B, torch.from_numpy(dYq).to(dev), dY)
        W_before = W.float().cpu().numpy().astype(np.float64)
        dX = torch.full((B, d), float("nan"), device=dev)
        run.layer.backward_sgd(B, run.X, run.idx, W, dY, mom, lr, mu, weight_decay=wd, bias=bias, bias_momentum=bmom, dX=dX)
        torch.cuda.synchronize()
        ref = oracle.tail_backward(inp.X, inp.idx, W_before, dYq.astype(np.float64), G)
        # dX comes from W as it was BEFORE the update
        assert oracle.rel_l2(dX.cpu().numpy(), ref["dX"]) <= 1e-4
        W_new, v_ref = oracle.sgd_momentum(W_before, ref["dW"], v_ref, lr, mu, wd)
        assert oracle.rel_l2(mom.cpu().numpy(), v_ref) <= 1e-5
        got = W.float().cpu().numpy().astype(np.float64)
        # one bf16 step of the result, plus what fp32 arithmetic can differ from fp64 by where the terms of w - lr v cancel:
        # the rounding of the operands, and the fp32 accumulation of the gradient (B terms; bounded through the sum of their
        # magnitudes, which the oracle gives when fed |X| and |dY|)
        gabs = oracle.tail_backward(np.abs(inp.X), inp.idx, W_before, np.abs(dYq).astype(np.float64), G, want_db=False)["dW"]
        allowed = _bf16_step(W_new) * (1.0 + 1e-6) + 2.0 ** -22 * (np.abs(W_before) + lr * np.abs(v_ref)) + lr * 2.0 ** -21 * gabs
        assert np.all(np.abs(got - W_new) <= allowed), np.max(np.abs(got - W_new) / allowed)
        assert oracle.rel_l2(got, W_new) <= 4e-3                   # bf16 rounding of the result
        assert np.mean(got == synth.round_bf16(W_new.astype(np.float32))[1].reshape(L, K)) > 0.99   # almost everywhere THE rounding
        if with_bias:
            b_ref, vb_ref = oracle.sgd_momentum(b_ref, ref["db"], vb_ref, lr, mu, 0.0)
            assert oracle.rel_l2(bmom.cpu().numpy(), vb_ref) <= 1e-5
            assert oracle.rel_l2(bias.cpu().numpy(), b_ref) <= 1e-5
        # the momentum the next step starts from is the device's (fp32) one on both sides
        v_ref = mom.cpu().numpy().astype(np.float64)
        if with_bias:
            vb_ref, b_ref = bmom.cpu().numpy().astype(np.float64), bias.cpu().numpy().astype(np.float64)


def test_backward_sgd_refusals():
    from paper_2606_01117_b200 import haste
    dev = torch.device("cuda:0")
    layer = haste.HasteLayer(128, 4096, 16, 32, 32, "f32")          # CUDA-core family: no fused kernel
    z = torch.zeros(16, device=dev)
    with pytest.raises(haste.HasteError) as e:
        layer.backward_sgd(32, z, z, z, z, z, 0.1, 0.9)
    assert e.value.status == haste.HASTE_ERR_UNSUPPORTED
    layer = haste.HasteLayer(256, 64 * 4, 64, 64, 64, "bf16")
    with pytest.raises(haste.HasteError) as e:
        layer.backward_sgd(64, z, z, z, z, z, 0.1, 0.9, bias=z)   # bias without its momentum
    assert e.value.status == haste.HASTE_ERR_INVALID_ARG
