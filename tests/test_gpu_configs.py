"""-m gpu parity at BASELINE.json's configs, in the launch configuration bench.py times.

Configs 1-2: every element against the full fp64 oracle.  Configs 3-4 (670K / 3M labels): the total
loss against the oracle run over label slices (the objective is a plain sum over labels, Eq. 3), and
dY / dW / db / dX on sampled outputs the oracle computes one by one (oracle.tail_points,
tail_label_rows, tail_batch_rows), always including every positive pair, labels that own positives
and the partial last group.  Config 5: reduced-L sweep points with the same G, K.
"""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest
import torch

from paper_2606_01117_b200 import synth

pytestmark = pytest.mark.gpu


def _oracle_loss_sliced(oracle, inp, G, L_h, threads=None):
    """Full-size loss: the oracle's O2 forward on group-aligned label slices, summed (ctypes drops the GIL)."""
    L = inp.W.shape[0]
    NG = -(-L // G)
    threads = threads or min(32, os.cpu_count() or 1)
    nchunk = max(1, min(NG, threads * 4))
    bounds = [(NG * c // nchunk) for c in range(nchunk + 1)]
    B = inp.X.shape[0]

    def one(c):
        g0, g1 = bounds[c], bounds[c + 1]
        l0, l1 = g0 * G, min(L, g1 * G)
        if l1 <= l0:
            return 0.0
        b = None if inp.bias is None else inp.bias[l0:l1]
        return oracle.tail_forward(inp.X, inp.idx[g0:g1], inp.W[l0:l1], b, inp.rowptr, inp.col, G,
                                   label_offset=L_h + l0, s=1.0 / B, want_z=False, want_dY=False)["loss"]

    with ThreadPoolExecutor(threads) as ex:
        return float(sum(ex.map(one, range(nchunk))))


def _packed_index(rows, labels, B, G):
    rows = np.asarray(rows, dtype=np.int64)
    labels = np.asarray(labels, dtype=np.int64)
    return ((labels // G) * B + rows) * G + labels % G


def _positive_pairs(inp, L_h, L):
    rows = np.repeat(np.arange(inp.X.shape[0]), np.diff(inp.rowptr))
    lab = inp.col.astype(np.int64) - L_h
    keep = (lab >= 0) & (lab < L)
    return rows[keep].astype(np.int32), lab[keep]


def test_config1_tiny_f32(oracle):
    from gpu_util import TailRun
    cfg = synth.CONFIGS["tiny_f32"]
    inp = synth.make_inputs(cfg)
    run = TailRun(inp, cfg.G)
    out = run.forward()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, cfg.G)
    assert abs(out["loss"] - ref["loss"]) <= 1e-5 * abs(ref["loss"])
    assert oracle.rel_l2(out["z"], ref["z"]) <= 1e-5
    assert oracle.rel_l2(out["dY"], ref["dY"]) <= 1e-5
    bout = run.backward()
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], cfg.G)
    for k in ("dW", "db", "dX"):
        assert oracle.rel_l2(bout[k], bref[k]) <= 1e-5, k


def test_config2_mid_bf16_full(oracle):
    from gpu_util import TailRun
    from paper_2606_01117_b200 import haste
    cfg = synth.CONFIGS["mid_bf16"]
    inp = synth.make_inputs(cfg, with_head=False)
    run = TailRun(inp, cfg.G, flags=haste.HASTE_IDX_SORTED_DISTINCT, label_offset=cfg.L_h, want_logits=False)
    out = run.forward()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, cfg.G, label_offset=cfg.L_h, want_z=False)
    assert abs(out["loss"] - ref["loss"]) <= 5e-3 * abs(ref["loss"])
    assert oracle.rel_l2(out["dY"], ref["dY"]) <= 5e-3
    pr, pl = _positive_pairs(inp, cfg.L_h, cfg.L_t)
    assert pr.size > 0
    assert oracle.rel_l2(out["dY"][pr, pl], ref["dY"][pr, pl]) <= 5e-3
    bout = run.backward()
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], cfg.G)
    for k in ("dW", "db", "dX"):
        assert oracle.rel_l2(bout[k], bref[k]) <= 5e-3, (k, oracle.rel_l2(bout[k], bref[k]))
    pl_u = np.unique(pl)
    assert oracle.rel_l2(bout["dW"][pl_u], bref["dW"][pl_u]) <= 5e-3      # gate (ii): labels that own positives
    assert oracle.rel_l2(bout["db"][pl_u], bref["db"][pl_u]) <= 5e-3


@pytest.mark.parametrize("name", ["670k", "3m"])
def test_full_size_sampled(oracle, name):
    from gpu_util import to_dev, t32
    from paper_2606_01117_b200 import haste
    cfg = synth.CONFIGS[name]
    inp = synth.make_inputs(cfg, with_head=False)
    B, d, L, G, K = cfg.B, cfg.d, cfg.L_t, cfg.G, cfg.K
    dev = torch.device("cuda:0")
    layer = haste.HasteLayer(d, L, G, K, B, "bf16", label_offset=cfg.L_h, flags=haste.HASTE_IDX_SORTED_DISTINCT)
    X, W, idx = to_dev(inp, "X"), to_dev(inp, "W"), t32(inp.idx)
    rowptr, col = t32(inp.rowptr), t32(inp.col)
    loss = torch.zeros(1, device=dev)
    dY = layer.alloc_dy(B)
    layer.forward_loss(B, X, idx, W, None, rowptr, col, loss=loss, dY=dY)
    dW = torch.empty(L, K, dtype=torch.bfloat16, device=dev)
    db = torch.empty(L, device=dev)
    dX = torch.empty(B, d, device=dev)
    layer.backward(B, X, idx, W, dY, dW=dW, dbias=db, dX=dX)
    torch.cuda.synchronize()

    # total loss (Eq. 3) against the oracle over label slices
    ref_loss = _oracle_loss_sliced(oracle, inp, G, cfg.L_h)
    assert abs(loss.item() - ref_loss) <= 5e-3 * abs(ref_loss), (loss.item(), ref_loss)

    # dY: random points + every positive pair + the whole partial last group
    rng = np.random.RandomState(cfg.seed)
    n = 20000
    rows = rng.randint(0, B, size=n).astype(np.int32)
    labs = rng.randint(0, L, size=n).astype(np.int64)
    pr, pl = _positive_pairs(inp, cfg.L_h, L)
    last0 = (L - 1) // G * G
    lr, ll = np.meshgrid(np.arange(B, dtype=np.int32), np.arange(last0, L, dtype=np.int64), indexing="ij")
    rows_all = np.concatenate([rows, pr, lr.ravel()])
    labs_all = np.concatenate([labs, pl, ll.ravel()])
    ref = oracle.tail_points(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, G, rows_all, labs_all, label_offset=cfg.L_h)
    got = dY[torch.from_numpy(_packed_index(rows_all, labs_all, B, G)).to(dev)].float().cpu().numpy()
    assert oracle.rel_l2(got[:n], ref["dY"][:n]) <= 5e-3
    assert pr.size > 0
    assert oracle.rel_l2(got[n:n + pr.size], ref["dY"][n:n + pr.size]) <= 5e-3
    assert oracle.rel_l2(got[n + pr.size:], ref["dY"][n + pr.size:]) <= 5e-3
    # padding labels of the last group (>= L) are written as zero
    NG = -(-L // G)
    if NG * G > L:
        tailpad = dY.view(NG, B, G)[NG - 1, :, L - last0:]
        assert torch.count_nonzero(tailpad).item() == 0

    # dW / db: random labels + labels that own positives + the last group
    labels = np.unique(np.concatenate([rng.randint(0, L, size=192), np.unique(pl)[:256], np.arange(last0, L)])).astype(np.int64)
    refl = oracle.tail_label_rows(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, G, labels, label_offset=cfg.L_h)
    sel = torch.from_numpy(labels).to(dev)
    assert oracle.rel_l2(dW[sel].float().cpu().numpy(), refl["dW"]) <= 5e-3
    assert oracle.rel_l2(db[sel].cpu().numpy(), refl["db"]) <= 5e-3
    own = np.isin(labels, pl)
    assert oracle.rel_l2(dW[sel].float().cpu().numpy()[own], refl["dW"][own]) <= 5e-3
    lastm = labels >= last0
    assert oracle.rel_l2(dW[sel].float().cpu().numpy()[lastm], refl["dW"][lastm]) <= 5e-3

    # dX: sampled batch rows over ALL labels
    brow = np.array(sorted(set([0, B - 1] + rng.randint(0, B, size=4).tolist())), dtype=np.int32)
    refr = oracle.tail_batch_rows(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, G, brow, label_offset=cfg.L_h)
    assert oracle.rel_l2(dX[torch.from_numpy(brow.astype(np.int64)).to(dev)].cpu().numpy(), refr["dX"]) <= 5e-3

    # P6 Euler identity at full size, from GPU outputs only: sum_f X[i,f] dX[i,f] = sum_l dY[i,l] z[i,l]
    # is checked per sampled row through the oracle's exact dX row above; here: dX is finite everywhere.
    assert torch.isfinite(dX).all() and torch.isfinite(dW.float()).all() and torch.isfinite(db).all()


@pytest.mark.parametrize("B,G", [(64, 1), (64, 8), (64, 16), (256, 32), (1024, 64), (256, 128)])
def test_config5_sweep_reduced(oracle, B, G):
    """Kernel-sweep points (K=64, d=768) on a reduced L = 65536 + 11 with the same G, K."""
    from gpu_util import TailRun
    from paper_2606_01117_b200 import haste
    L = 8192 + 11 if G == 1 else 65536 + 11
    cfg = synth.sweep_config(B, G, L=L)
    inp = synth.make_inputs(cfg, with_head=False)
    run = TailRun(inp, G, flags=haste.HASTE_IDX_SORTED_DISTINCT, want_logits=False)
    out = run.forward()
    ref = oracle.tail_forward(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, G, want_z=False)
    assert abs(out["loss"] - ref["loss"]) <= 5e-3 * abs(ref["loss"])
    assert oracle.rel_l2(out["dY"], ref["dY"]) <= 5e-3
    bout = run.backward()
    bref = oracle.tail_backward(inp.X, inp.idx, inp.W, ref["dY"], G)
    for k in ("dW", "db", "dX"):
        assert oracle.rel_l2(bout[k], bref[k]) <= 5e-3, (k, oracle.rel_l2(bout[k], bref[k]))
