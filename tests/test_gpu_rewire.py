"""-m gpu parity of haste_rewire (Algorithm 3, group-shared rewiring) against the oracle's rewire: integer
and byte work (which slots are pruned, the regrown features, the row order after the re-sort) and the reinitialised weights
must be BIT-EXACT; untouched entries must be untouched."""
import numpy as np
import pytest
import torch

from paper_2606_01117_b200 import synth

pytestmark = pytest.mark.gpu


def _run(oracle, B, d, L, G, K, dtype, rho, init_random, resort, with_mom, seed, w_std=0.3, ties=False):
    from gpu_util import TailRun, to_dev, t32
    inp = synth.small_case(200 + L % 97, B, d, L, G, K, dtype=dtype, w_std=w_std, with_bias=False)
    if ties:      # many exactly equal scores: whole columns of equal magnitude, and zeros
        inp.W[:, ::3] = 0.25
        inp.W[:, 1::7] = 0.0
        if dtype == "bf16":
            inp.bits["W"] = synth.round_bf16(inp.W)[0].reshape(L, K)
    run = TailRun(inp, G, want_logits=False)
    dev = run.X.device
    rho = float(np.float32(rho))
    mom0 = np.random.RandomState(1).standard_normal((L, K)).astype(np.float32) if with_mom else None
    mom = None if mom0 is None else torch.from_numpy(mom0).to(dev)
    idx, W = run.idx.clone(), run.W.clone()
    m = run.layer.rewire(idx, W, rho, momentum=mom, init_random=init_random, seed=seed, resort=resort)
    torch.cuda.synchronize()
    ref = oracle.rewire(inp.idx, inp.W, G, d, rho, init_random=init_random, seed=seed, resort=resort, momentum=mom0)
    assert m == ref["m"]
    assert np.array_equal(idx.cpu().numpy(), ref["idx"])
    got_W = W.float().cpu().numpy()
    want_W = ref["W"] if dtype == "f32" else synth.round_bf16(ref["W"])[1].reshape(L, K)
    assert np.array_equal(got_W, want_W)
    if with_mom:
        assert np.array_equal(mom.cpu().numpy(), ref["momentum"])
    return inp, run, idx, W, ref


@pytest.mark.parametrize("shape", [(64, 768, 64 * 23 + 11, 64, 128, "bf16"), (32, 256, 32 * 40 + 5, 32, 64, "bf16"),
                                   (16, 128, 16 * 300 + 3, 16, 32, "f32"), (8, 64, 777, 1, 16, "f32"), (32, 512, 128 * 70, 128, 64, "bf16")])
@pytest.mark.parametrize("init_random", [False, True])
@pytest.mark.parametrize("resort", [False, True])
def test_rewire_bit_exact(oracle, shape, init_random, resort):
    B, d, L, G, K, dtype = shape
    _run(oracle, B, d, L, G, K, dtype, 0.15, init_random, resort, with_mom=True, seed=1234 + L)


def test_rewire_ties_and_extremes(oracle):
    # ties at the threshold (equal scores across many slots), then rho = 1 (everything goes) and rho = 0 (nothing does)
    _run(oracle, 16, 256, 64 * 50 + 9, 64, 64, "bf16", 0.2, False, True, True, 5, ties=True)
    _run(oracle, 16, 256, 64 * 50 + 9, 64, 64, "bf16", 0.37, True, True, False, 6, ties=True)
    _run(oracle, 16, 128, 64 * 9, 64, 64, "bf16", 1.0, True, True, True, 7)
    inp, run, idx, W, ref = _run(oracle, 16, 128, 64 * 9, 64, 64, "bf16", 0.0, True, True, True, 8)
    assert torch.equal(idx, run.idx) and torch.equal(W, run.W)


def test_rewired_layer_still_runs_through_the_kernels(oracle):
    """After a rewiring WITHOUT re-sort the idx rows are unsorted and may hold duplicates (R4): forward, dW and dX of the
    tcgen05 family must still match the oracle on the rewired layer."""
    from gpu_util import TailRun
    inp, run, idx, W, ref = _run(oracle, 200, 768, 64 * 23 + 11, 64, 128, "bf16", 0.3, True, False, False, 99)
    inp.idx = ref["idx"]
    bits, Wv = synth.round_bf16(ref["W"])
    inp.W, inp.bits["W"] = Wv.reshape(ref["W"].shape), bits.reshape(ref["W"].shape)
    run2 = TailRun(inp, 64, want_logits=True)
    out = run2.forward()
    r = oracle.tail_forward(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, 64)
    assert oracle.rel_l2(out["z"], r["z"]) <= 1e-5 and oracle.rel_l2(out["dY"], r["dY"]) <= 5e-3
    b = run2.backward()
    br = oracle.tail_backward(inp.X, inp.idx, inp.W, r["dY"], 64)
    for k in ("dW", "db", "dX"):
        assert oracle.rel_l2(b[k], br[k]) <= 5e-3, k


def test_rewire_config3_size_timing_sanity(oracle):
    """Config 3's tail (653 707 labels, 1.3 M slots): parity of the mask through the regrown idx at full size."""
    from paper_2606_01117_b200 import haste
    cfg = synth.CONFIGS["670k"]
    inp = synth.make_inputs(cfg, with_head=False)
    from gpu_util import to_dev, t32
    layer = haste.HasteLayer(cfg.d, cfg.L_t, cfg.G, cfg.K, 64, "bf16")
    idx, W = t32(inp.idx), to_dev(inp, "W")
    rho = float(np.float32(0.1))
    m = layer.rewire(idx, W, rho, init_random=True, seed=42, resort=True)
    ref = oracle.rewire(inp.idx, inp.W, cfg.G, cfg.d, rho, init_random=True, seed=42, resort=True)
    assert m == ref["m"] == int(np.floor(inp.idx.size * rho))
    assert np.array_equal(idx.cpu().numpy(), ref["idx"])
    assert np.array_equal(W.float().cpu().numpy(), synth.round_bf16(ref["W"])[1].reshape(ref["W"].shape))
