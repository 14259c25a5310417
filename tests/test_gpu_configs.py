"""-m gpu parity at BASELINE.json's configs, in the launch configuration bench.py times.

Configs 1-2: every element against the full fp64 oracle.  Configs 3-4 (670K / 3M labels): the total
loss against the oracle run over label slices (the objective is a plain sum over labels, Eq. 3), dY / logits /
dW / db / dX on sampled outputs the oracle computes one by one (oracle.tail_points, tail_label_rows,
tail_batch_rows: every positive pair, labels that own positives, the partial last group, one dX row from every
128-row tile x 32-row quadrant), and the two Euler identities over EVERY batch row and EVERY label from the GPU
tensors alone.  Config 5: full L = 670 091 at B = 64 for every G of the sweep, the same way; the other sweep
points at a reduced L with the same G, K, every element.
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


def _euler_identities(X, W, dY, z, dW, dX, B, L, G, NG):
    """P6 from GPU outputs only, over ALL rows and ALL labels, in fp64 on the device:
         row i  :  sum_f X[i,f] dX[i,f]  =  sum_l dY[i,l] z[i,l]        (z is bilinear in X and W; bias = 0 here)
         label l:  sum_j W[l,j] dW[l,j]  =  sum_i dY[i,l] z[i,l]
    dY is the library's group-blocked [NG][B][G] buffer, z the [B,L] logits of the same forward call.
    Returns (lhs_row, rhs_row, lhs_lab, rhs_lab, scale_lab) as fp64 numpy arrays."""
    dev = X.device
    rhs_row = torch.zeros(B, dtype=torch.float64, device=dev)
    rhs_lab = torch.empty(L, dtype=torch.float64, device=dev)
    abs_lab = torch.empty(L, dtype=torch.float64, device=dev)
    dYv = dY.view(NG, B, G)
    step = 512                                                   # groups per slice
    for g0 in range(0, NG, step):
        g1 = min(NG, g0 + step)
        l0, l1 = g0 * G, min(L, g1 * G)
        dy = dYv[g0:g1].permute(1, 0, 2).reshape(B, (g1 - g0) * G)[:, : l1 - l0].double()
        prod = dy * z[:, l0:l1].double()
        rhs_row += prod.sum(dim=1)
        rhs_lab[l0:l1] = prod.sum(dim=0)
        abs_lab[l0:l1] = prod.abs().sum(dim=0)
    lhs_row = (X.double() * dX.double()).sum(dim=1)
    wd = W.double() * dW.double()
    lhs_lab = wd.sum(dim=1)
    scale_lab = wd.abs().sum(dim=1) + abs_lab
    return [t.cpu().numpy() for t in (lhs_row, rhs_row, lhs_lab, rhs_lab, scale_lab)]


@pytest.mark.parametrize("name", ["670k", "3m"])
def test_full_size_sampled(oracle, name):
    from gpu_util import to_dev, t32
    from paper_2606_01117_b200 import haste
    cfg = synth.CONFIGS[name]
    inp = synth.make_inputs(cfg, with_head=False)
    B, d, L, G, K = cfg.B, cfg.d, cfg.L_t, cfg.G, cfg.K
    NG = -(-L // G)
    dev = torch.device("cuda:0")
    layer = haste.HasteLayer(d, L, G, K, B, "bf16", label_offset=cfg.L_h, flags=haste.HASTE_IDX_SORTED_DISTINCT)
    X, W, idx = to_dev(inp, "X"), to_dev(inp, "W"), t32(inp.idx)
    rowptr, col = t32(inp.rowptr), t32(inp.col)
    loss = torch.zeros(1, device=dev)
    dY = layer.alloc_dy(B)
    z = torch.empty(B, L, device=dev)                            # 1.3 GB (670k) / 3.0 GB (3m): for the identities below
    layer.forward_loss(B, X, idx, W, None, rowptr, col, loss=loss, dY=dY, logits_out=z)
    dW = torch.empty(L, K, dtype=torch.bfloat16, device=dev)
    db = torch.empty(L, device=dev)
    dX = torch.empty(B, d, device=dev)
    layer.backward(B, X, idx, W, dY, dW=dW, dbias=db, dX=dX)
    torch.cuda.synchronize()

    # total loss (Eq. 3) against the oracle over label slices
    ref_loss = _oracle_loss_sliced(oracle, inp, G, cfg.L_h)
    assert abs(loss.item() - ref_loss) <= 5e-3 * abs(ref_loss), (loss.item(), ref_loss)

    # dY and logits: random points + every positive pair + the whole partial last group
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
    gotz = z[torch.from_numpy(rows_all.astype(np.int64)).to(dev), torch.from_numpy(labs_all).to(dev)].cpu().numpy()
    assert oracle.rel_l2(gotz, ref["z"]) <= 1e-5                 # the logits the identities rest on
    # padding labels of the last group (>= L) are written as zero
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

    # dX: one batch row from EVERY (128-row batch tile, 32-row TMEM lane quadrant) of the launch (16 rows at B = 512, 8 at
    # B = 256), first and last row included, each over ALL labels through the oracle
    brow = sorted(set([0, B - 1] + [q0 + int(rng.randint(0, min(32, B - q0))) for q0 in range(0, B, 32)]))
    brow = np.array(brow, dtype=np.int32)
    assert all(((brow >= q0) & (brow < q0 + 32)).any() for q0 in range(0, B, 32))
    refr = oracle.tail_batch_rows(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, G, brow, label_offset=cfg.L_h)
    gx = dX[torch.from_numpy(brow.astype(np.int64)).to(dev)].cpu().numpy()
    assert oracle.rel_l2(gx, refr["dX"]) <= 5e-3
    for k in range(brow.size):                                   # and row by row: one bad quadrant cannot hide among the others
        assert oracle.rel_l2(gx[k], refr["dX"][k]) <= 5e-3, int(brow[k])

    # P6 Euler identities over the WHOLE output (every batch row, every label), from GPU tensors only.
    # Tolerances from the arithmetic: both sides of the row identity use the same bf16 dY and differ only by fp32
    # accumulation (dX: ~1e5 terms per entry, z: K terms) -> 2e-4 of a sum that is ~16 per row and well conditioned;
    # the label identity carries the bf16 rounding of dW (2^-9 per entry, independent over K entries): each label within
    # 4e-3 of the sum of magnitudes of its terms, all labels together within 2e-3 in relative L2.
    lhs_row, rhs_row, lhs_lab, rhs_lab, scale_lab = _euler_identities(X, W, dY, z, dW, dX, B, L, G, NG)
    assert np.all(np.isfinite(lhs_row)) and np.all(np.isfinite(lhs_lab))
    assert np.max(np.abs(lhs_row - rhs_row) / np.abs(rhs_row)) <= 2e-4, np.max(np.abs(lhs_row - rhs_row) / np.abs(rhs_row))
    assert np.max(np.abs(lhs_lab - rhs_lab) / scale_lab) <= 4e-3, np.max(np.abs(lhs_lab - rhs_lab) / scale_lab)
    assert oracle.rel_l2(lhs_lab, rhs_lab) <= 2e-3, oracle.rel_l2(lhs_lab, rhs_lab)
    # db against the same dY, every label: db[l] = sum_i dY[i,l]
    dbr = dY.view(NG, B, G).float().sum(dim=1).reshape(NG * G)[:L].double().cpu().numpy()
    assert oracle.rel_l2(db.double().cpu().numpy(), dbr) <= 1e-5


@pytest.mark.parametrize("G", [1, 8, 16, 32, 64, 128])
def test_config5_full_L_B64(oracle, G):
    """Config 5 at full L = 670 091 for B = 64, every G of the sweep: total loss against the oracle over
    label slices, dY / logits at sampled points + every positive pair + the partial last group, dW / db at sampled labels,
    dX at sampled batch rows (each over all labels)."""
    from gpu_util import to_dev, t32
    from paper_2606_01117_b200 import haste
    B, K = 64, 64
    cfg = synth.sweep_config(B, G)
    inp = synth.make_inputs(cfg, with_head=False)
    d, L = cfg.d, cfg.L_t
    NG = -(-L // G)
    dev = torch.device("cuda:0")
    layer = haste.HasteLayer(d, L, G, K, B, "bf16", flags=haste.HASTE_IDX_SORTED_DISTINCT)
    X, W, idx = to_dev(inp, "X"), to_dev(inp, "W"), t32(inp.idx)
    rowptr, col = t32(inp.rowptr), t32(inp.col)
    loss = torch.zeros(1, device=dev)
    dY = layer.alloc_dy(B)
    z = torch.empty(B, L, device=dev)
    layer.forward_loss(B, X, idx, W, None, rowptr, col, loss=loss, dY=dY, logits_out=z)
    dW = torch.empty(L, K, dtype=torch.bfloat16, device=dev)
    db = torch.empty(L, device=dev)
    dX = torch.empty(B, d, device=dev)
    layer.backward(B, X, idx, W, dY, dW=dW, dbias=db, dX=dX)
    torch.cuda.synchronize()
    ref_loss = _oracle_loss_sliced(oracle, inp, G, 0)
    assert abs(loss.item() - ref_loss) <= 5e-3 * abs(ref_loss), (loss.item(), ref_loss)
    rng = np.random.RandomState(500 + G)
    n = 20000
    rows = rng.randint(0, B, size=n).astype(np.int32)
    labs = rng.randint(0, L, size=n).astype(np.int64)
    pr, pl = _positive_pairs(inp, 0, L)
    last0 = (L - 1) // G * G
    lr, ll = np.meshgrid(np.arange(B, dtype=np.int32), np.arange(last0, L, dtype=np.int64), indexing="ij")
    rows_all = np.concatenate([rows, pr, lr.ravel()])
    labs_all = np.concatenate([labs, pl, ll.ravel()])
    ref = oracle.tail_points(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, G, rows_all, labs_all)
    got = dY[torch.from_numpy(_packed_index(rows_all, labs_all, B, G)).to(dev)].float().cpu().numpy()
    assert oracle.rel_l2(got[:n], ref["dY"][:n]) <= 5e-3
    assert pr.size > 0 and oracle.rel_l2(got[n:n + pr.size], ref["dY"][n:n + pr.size]) <= 5e-3
    assert oracle.rel_l2(got[n + pr.size:], ref["dY"][n + pr.size:]) <= 5e-3
    gotz = z[torch.from_numpy(rows_all.astype(np.int64)).to(dev), torch.from_numpy(labs_all).to(dev)].cpu().numpy()
    assert oracle.rel_l2(gotz, ref["z"]) <= 1e-5
    labels = np.unique(np.concatenate([rng.randint(0, L, size=192), np.unique(pl)[:256], np.arange(last0, L)])).astype(np.int64)
    refl = oracle.tail_label_rows(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, G, labels)
    sel = torch.from_numpy(labels).to(dev)
    assert oracle.rel_l2(dW[sel].float().cpu().numpy(), refl["dW"]) <= 5e-3
    assert oracle.rel_l2(db[sel].cpu().numpy(), refl["db"]) <= 5e-3
    brow = np.array(sorted(set([0, B - 1, int(rng.randint(0, 32)), 32 + int(rng.randint(0, 32))])), dtype=np.int32)
    refr = oracle.tail_batch_rows(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, G, brow)
    gx = dX[torch.from_numpy(brow.astype(np.int64)).to(dev)].cpu().numpy()
    for k in range(brow.size):
        assert oracle.rel_l2(gx[k], refr["dX"][k]) <= 5e-3, int(brow[k])
    # the Euler identities over the whole output, as at configs 3 and 4
    lhs_row, rhs_row, lhs_lab, rhs_lab, scale_lab = _euler_identities(X, W, dY, z, dW, dX, B, L, G, NG)
    assert np.max(np.abs(lhs_row - rhs_row) / np.abs(rhs_row)) <= 2e-4
    assert np.max(np.abs(lhs_lab - rhs_lab) / scale_lab) <= 4e-3
    assert oracle.rel_l2(lhs_lab, rhs_lab) <= 2e-3


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
