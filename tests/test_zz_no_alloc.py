"""-m gpu: haste_forward_topk_static (include/haste.h) -- the fused top-k forward with its candidate lists in a file-scope
device array of the library, for callers that cannot call cudaMalloc -- against the existing haste_forward_topk on the same
inputs.  Both run the same kernels on the same operands and differ only in where the scratch lives, so values and labels
must agree exactly (the gate written below is the top-k tests' own: labels equal, values within 1e-5 relative).

Collected last on purpose (the suite runs with pytest -x: a failure here must not hide the other tests).  Passes alone in
a fresh process and after the rest of the suite: it depends on no state but the library's own static array, which every
call overwrites where it reads."""
import numpy as np
import pytest
import torch

from paper_2606_01117_b200 import synth

pytestmark = pytest.mark.gpu


def _inputs(seed, B, d, L, G, K):
    from gpu_util import to_dev, t32
    inp = synth.small_case(seed, B, d, L, G, K, dtype="bf16", with_bias=True, w_std=0.3)
    return to_dev(inp, "X"), to_dev(inp, "W"), t32(inp.idx), t32(inp.bias)


def test_topk_static_matches_the_allocating_path_on_two_calls_in_a_row():
    from paper_2606_01117_b200 import haste
    from gpu_util import dev
    d, L, G, K, B_max = 768, 64 * 700 + 11, 64, 128, 300
    layer = haste.HasteLayer(d, L, G, K, B_max, "bf16", label_offset=1000)
    assert layer.kernel_family == 1
    # two different calls: the second has a smaller batch and another k, so anything it read from what the first left in
    # the shared array (which keeps its contents between calls) would show
    calls = [(300, 5, _inputs(1, 300, d, L, G, K)), (130, 8, _inputs(2, 130, d, L, G, K))]
    outs = []
    for B, k, _ in calls:
        outs.append((torch.full((B, k), float("nan"), device=dev()), torch.full((B, k), -7, dtype=torch.int64, device=dev())))
    # warm-up (the first launch of a kernel loads it), then the two calls in a row with the free device memory read around them
    B0, k0, (X0, W0, idx0, bias0) = calls[0]
    layer.forward_topk_static(B0, X0, idx0, W0, bias0, k0, outs[0][0], outs[0][1])
    torch.cuda.synchronize()
    for v, i in outs:
        v.fill_(float("nan")); i.fill_(-7)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for (B, k, (X, W, idx, bias)), (v, i) in zip(calls, outs):
        layer.forward_topk_static(B, X, idx, W, bias, k, v, i)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    assert free_after == free_before, "haste_forward_topk_static changed the free device memory: %d -> %d" % (free_before, free_after)
    # the existing path (its first call allocates the handle's own candidate workspace), same inputs
    for (B, k, (X, W, idx, bias)), (v, i) in zip(calls, outs):
        rv = torch.full((B, k), float("nan"), device=dev())
        ri = torch.full((B, k), -7, dtype=torch.int64, device=dev())
        layer.forward_topk(B, X, idx, W, bias, k, rv, ri)
        torch.cuda.synchronize()
        assert torch.isfinite(rv).all() and (ri >= 1000).all() and (ri < 1000 + L).all()
        assert torch.equal(i, ri), "labels differ (B=%d, k=%d)" % (B, k)
        assert torch.allclose(v, rv, rtol=1e-5, atol=0.0), "values differ (B=%d, k=%d)" % (B, k)
        assert (v[:, :-1] >= v[:, 1:]).all()


def test_topk_static_rejects_what_it_cannot_serve():
    from paper_2606_01117_b200 import haste
    from gpu_util import dev
    layer = haste.HasteLayer(128, 4096, 16, 32, 32, "f32")       # CUDA-core family: no fused top-k, as for haste_forward_topk
    z = torch.zeros(16, device=dev())
    with pytest.raises(haste.HasteError) as e:
        layer.forward_topk_static(1, z, z, z, None, 5, z, z)
    assert e.value.status == haste.HASTE_ERR_UNSUPPORTED
    layer2 = haste.HasteLayer(256, 64 * 9, 64, 64, 32, "bf16")
    with pytest.raises(haste.HasteError) as e:
        layer2.forward_topk_static(1, z, z, z, None, 9, z, z)      # k beyond 8
    assert e.value.status == haste.HASTE_ERR_INVALID_ARG
