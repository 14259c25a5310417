"""-m gpu: the hot calls are asynchronous stream work only (include/haste.h, "Asynchrony"): no call of the step
synchronises, allocates or reads back, so one whole step -- haste_forward_loss + haste_backward (+ the dense head) --
can be captured into a CUDA graph and replayed.  The replay must give what the plain stream launches give: loss, dY and
dW bit for bit (they have one writer per element), dX up to the order of its float atomics."""
import numpy as np
import pytest
import torch

from paper_2606_01117_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("shape", [(300, 768, 64 * 40 - 5, 64, 128), (64, 128, 16 * 50, 16, 32)],
                         ids=["tcgen05_family", "cuda_core_family"])
def test_step_captures_into_a_cuda_graph(shape):
    from paper_2606_01117_b200 import haste
    from gpu_util import dev, to_dev, t32
    B, d, L, G, K = shape
    Lh = 256
    dtype = "bf16" if G >= 32 else "f32"
    inp = synth.small_case(321, B, d, L, G, K, dtype=dtype, with_bias=True)
    X, W, idx, bias = to_dev(inp, "X"), to_dev(inp, "W"), t32(inp.idx), t32(inp.bias)
    rowptr, col = t32(inp.rowptr), t32(inp.col)
    layer = haste.HasteLayer(d, L, G, K, B, dtype)
    head = haste.HasteHead(d, Lh, B, dtype, label_offset=0)
    tdt = torch.bfloat16 if dtype == "bf16" else torch.float32
    rng = np.random.RandomState(3)
    Wh = torch.from_numpy((rng.standard_normal((Lh, d)) * 0.02).astype(np.float32)).to(dev()).to(tdt)
    out = dict(loss=torch.zeros(2, device=dev()), dY=layer.alloc_dy(B), dW=torch.empty(L, K, dtype=tdt, device=dev()),
               db=torch.empty(L, device=dev()), dX=torch.empty(B, d, device=dev()),
               dYh=torch.empty(B, Lh, dtype=tdt, device=dev()), dWh=torch.empty(Lh, d, dtype=tdt, device=dev()),
               dXh=torch.empty(B, d, device=dev()))

    def step():
        layer.forward_loss(B, X, idx, W, bias, rowptr, col, loss=out["loss"][0:1], dY=out["dY"])
        layer.backward(B, X, idx, W, out["dY"], dW=out["dW"], dbias=out["db"], dX=out["dX"])
        head.forward_loss(B, X, Wh, None, rowptr, col, loss=out["loss"][1:2], dY=out["dYh"])
        head.backward(B, X, Wh, out["dYh"], dWh=out["dWh"], dbias=None, dX=out["dXh"])

    step()
    torch.cuda.synchronize()
    ref = {k: v.clone() for k, v in out.items()}

    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        step()                                   # first call on this stream outside the capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):          # capture_error_mode "global": any synchronising or allocating call fails here
        step()
    for k, v in out.items():
        v.fill_(float("nan")) if v.is_floating_point() else v.zero_()
    for _ in range(3):                           # replays reuse the handles' workspaces: they must be re-zeroed per call
        g.replay()
    torch.cuda.synchronize()
    for k in ("loss", "dY", "dW", "db", "dYh", "dWh"):
        assert torch.equal(out[k], ref[k]), k
    for k in ("dX", "dXh"):
        assert torch.allclose(out[k], ref[k], rtol=1e-4, atol=1e-6), k


@pytest.mark.parametrize("route", ["two_kernels", "one_kernel"])
def test_back_to_back_steps_are_reproducible(route):
    """The step's kernels are launched with programmatic stream serialization (common.cuh): each starts while the one
    before is still draining and must not touch global memory before its griddepcontrol.wait.  A kernel that did would
    read a half-written dY, X^T or dX^T now and then.  40 steps back to back with inputs that change from step to step
    (so that a stale read is a different value), each compared with the same step run alone: loss, dY, dW, db bit for
    bit, dX up to the order of its float atomics -- and the workspace the transpose-out kernel zeroes behind itself
    must be clean every time (dX would accumulate otherwise)."""
    from paper_2606_01117_b200 import haste
    from gpu_util import dev, to_dev, t32
    B, d, L, G, K, Lh = 512, 768, 64 * 1200 + 7, 64, 128, 2048
    inp = synth.small_case(77, B, d, L, G, K, dtype="bf16", with_bias=True)
    W, idx, bias = to_dev(inp, "W"), t32(inp.idx), t32(inp.bias)
    rowptr, col = t32(inp.rowptr), t32(inp.col)
    layer = haste.HasteLayer(d, L, G, K, B, "bf16", flags=haste.HASTE_XT_FROM_FORWARD)
    head = haste.HasteHead(d, Lh, B, "bf16", label_offset=0)
    g = torch.Generator(device="cpu").manual_seed(5)
    Xs = [(torch.randn(B, d, generator=g) * (0.5 + 0.25 * i)).to(torch.bfloat16).to(dev()) for i in range(4)]
    Wh = (torch.randn(Lh, d, generator=g) * 0.02).to(torch.bfloat16).to(dev())

    def new_out():
        return dict(loss=torch.zeros(2, device=dev()), dY=layer.alloc_dy(B), dW=torch.empty(L, K, dtype=torch.bfloat16, device=dev()),
                    db=torch.empty(L, device=dev()), dX=torch.empty(B, d, device=dev()),
                    dYh=torch.empty(B, Lh, dtype=torch.bfloat16, device=dev()), dWh=torch.empty(Lh, d, dtype=torch.bfloat16, device=dev()),
                    dXh=torch.empty(B, d, device=dev()))

    def step(X, o):
        if route == "one_kernel":       # forward + dW in one kernel (tc_fused.cu), then dX: the route bench.py's step takes
            layer.forward_loss_dw(B, X, idx, W, bias, rowptr, col, loss=o["loss"][0:1], dY=o["dY"], dW=o["dW"], dbias=o["db"])
            layer.backward(B, X, idx, W, o["dY"], dX=o["dX"])
        else:
            layer.forward_loss(B, X, idx, W, bias, rowptr, col, loss=o["loss"][0:1], dY=o["dY"])
            layer.backward(B, X, idx, W, o["dY"], dW=o["dW"], dbias=o["db"], dX=o["dX"])
        head.forward_loss(B, X, Wh, None, rowptr, col, loss=o["loss"][1:2], dY=o["dYh"])
        head.backward(B, X, Wh, o["dYh"], dWh=o["dWh"], dbias=None, dX=o["dXh"])

    refs = []
    for X in Xs:                                  # each step alone, a synchronize on both sides
        o = new_out()
        torch.cuda.synchronize()
        step(X, o)
        torch.cuda.synchronize()
        refs.append(o)
    outs = [new_out() for _ in range(4)]
    torch.cuda.synchronize()
    for it in range(40):                          # back to back, no synchronize: kernels of neighbouring steps overlap
        step(Xs[it % 4], outs[it % 4])
    torch.cuda.synchronize()
    for i in range(4):
        for k in ("loss", "dY", "dW", "db", "dYh", "dWh"):
            assert torch.equal(outs[i][k], refs[i][k]), (i, k)
        for k in ("dX", "dXh"):
            assert torch.allclose(outs[i][k], refs[i][k], rtol=1e-4, atol=1e-6), (i, k)
