"""-m gpu parity of the on-chip accumulating dX kernel (csrc/tc_dx_acc.cu) on the cases its design turns on:
features of all three destination classes (TMEM columns / shared-memory rows / L2 reductions), slot ranges that
start and end exactly at the class boundaries, groups whose idx row is NOT strictly increasing (duplicates,
unsorted: reading R4, they take the atomic path) mixed with strictly increasing ones, ragged batch tiles, and
both fan-ins the kernel is built for.  dX = sum_g dY_g W_g scattered by idx_g.

Two gates per case, both through haste_dy_pack so that only the backward is under test:
  * small-integer dY and W: dX (and dW, db) must equal the fp64 oracle EXACTLY, whatever the order of additions;
  * real-valued dY rounded to bf16: rel-L2 <= 1e-4 against the oracle run on the same rounded dY.
"""
import numpy as np
import pytest

from paper_2606_01117_b200 import synth

pytestmark = pytest.mark.gpu


def _boundary_idx(rng, NG, K, d, kind):
    """idx rows [NG,K] int32 in [0,d) that stress the class boundaries of tc_dx_acc.cu (255/383 TMEM features for
    K = 128/64, then as many shared-memory rows as fit, then L2)."""
    tf = 512 - 2 * K - 1
    idx = np.empty((NG, K), dtype=np.int32)
    for g in range(NG):
        mode = g % 6 if kind == "mixed" else 0
        if mode == 0:      # strictly increasing, uniform over [0,d)
            row = np.sort(rng.choice(d, size=K, replace=False))
        elif mode == 1:    # a run of consecutive features straddling the TMEM / shared-memory boundary
            lo = max(0, min(d - K, tf - K // 2))
            row = np.arange(lo, lo + K)
        elif mode == 2:    # everything at the top of the feature range (L2 class when d is large), strictly increasing
            row = np.arange(d - K, d)
        elif mode == 3:    # duplicates inside the row (sorted, NOT strict): atomic path
            row = np.sort(rng.choice(d, size=K, replace=True))
            row[K // 2] = row[K // 2 - 1]
        elif mode == 4:    # unsorted, distinct
            row = rng.permutation(d)[:K]
            if np.all(np.diff(row) > 0):
                row = row[::-1]
        else:              # everything below the first boundary (one class owns the whole row)
            row = np.sort(rng.choice(min(d, max(K, tf // 2)), size=K, replace=False))
        idx[g] = row
    return idx


CASES = [
    # B, d, NG (L = G*NG - 5), G, K, kind
    (300, 768, 23, 64, 128, "mixed"),     # config-3 tile shape: 255 TMEM + ~295 smem + L2 features, ragged batch tile
    (128, 1024, 17, 64, 64, "mixed"),     # config-4 tile shape: 383 TMEM features, d = 1024
    (130, 768, 9, 128, 128, "mixed"),     # wide groups: two operand stages, fewer shared-memory rows
    (64, 400, 11, 128, 64, "mixed"),      # d barely above the TMEM class (383 features): 17 shared-memory rows, no L2 class
    (257, 768, 40, 64, 128, "strict"),    # every row strictly increasing (the fast path only)
    (200, 768, 21, 32, 64, "mixed"),      # config-2 tile shape: G = 32 (dY tile is a 64-byte-swizzle operand)
    (130, 768, 13, 32, 128, "mixed"),
    (200, 768, 41, 16, 64, "mixed"),      # narrow groups: the dY tile is a 32-byte-swizzle operand, one MMA per group
    (130, 1024, 37, 16, 128, "mixed"),
    (300, 768, 53, 8, 64, "mixed"),       # G = 8: labels 8-15 of the operands are zero padding (TMA fill / zeroed W rows)
    (129, 600, 29, 8, 128, "mixed"),
]


@pytest.mark.parametrize("case", CASES, ids=lambda c: "B%d_d%d_NG%d_G%d_K%d_%s" % c)
def test_dx_classes_exact_and_close(oracle, case):
    from paper_2606_01117_b200 import haste
    from gpu_util import TailRun, dy_rounded
    B, d, NG, G, K, kind = case
    L = G * NG - 5
    inp = synth.small_case(100 + B + d, B, d, L, G, K, dtype="bf16", with_bias=False, w_std=0.05)
    rng = np.random.RandomState(B + d + K)
    inp.idx = _boundary_idx(rng, NG, K, d, kind)
    flags = haste.HASTE_IDX_SORTED_DISTINCT if kind == "strict" else 0

    # ---- gate 1: integers, exact
    Wi = rng.randint(-4, 5, size=(L, K)).astype(np.float32)
    Xi = rng.randint(-4, 5, size=(B, d)).astype(np.float32)
    dYi = rng.randint(-3, 4, size=(B, L)).astype(np.float32)
    inp.X, inp.W = Xi, Wi
    inp.bits["X"], inp.bits["W"] = synth.round_bf16(Xi)[0].reshape(B, d), synth.round_bf16(Wi)[0].reshape(L, K)
    run = TailRun(inp, G, flags=flags, dw_dtype="f32")
    assert run.layer.kernel_family == 1
    out = run.backward(dY_BL=dYi)
    ref = oracle.tail_backward(inp.X, inp.idx, inp.W, dYi.astype(np.float64), G)
    assert np.array_equal(out["dX"].astype(np.float64), ref["dX"])
    assert np.array_equal(out["dW"].astype(np.float64), ref["dW"])
    assert np.array_equal(out["db"].astype(np.float64), ref["db"])
    # a second call on the same handle must give the same answer (accumulators are re-zeroed per call)
    out2 = run.backward(dY_BL=dYi)
    assert np.array_equal(out2["dX"], out["dX"])

    # ---- gate 2: real values, accumulation error only
    Wr = (rng.standard_normal((L, K)) * 0.05).astype(np.float32)
    dYr = (rng.standard_normal((B, L)) / B).astype(np.float32)
    bits, Wr = synth.round_bf16(Wr)
    inp.W, inp.bits["W"] = Wr.reshape(L, K), bits.reshape(L, K)
    run = TailRun(inp, G, flags=flags, dw_dtype="f32")
    dYq = dy_rounded(inp, dYr)
    out = run.backward(dY_BL=dYq)
    ref = oracle.tail_backward(inp.X, inp.idx, inp.W, dYq.astype(np.float64), G)
    for k in ("dX", "dW", "db"):
        err = oracle.rel_l2(out[k], ref[k])
        assert err <= 1e-4, (k, err)
    # per-class slices of dX on their own (a class that silently dropped its adds would hide in the global norm)
    tf = 512 - 2 * K - 1
    for lo, hi in ((0, min(d, tf)), (min(d, tf), min(d, tf + 120)), (max(0, d - 100), d)):
        if hi > lo and np.linalg.norm(ref["dX"][:, lo:hi]) > 0:
            assert oracle.rel_l2(out["dX"][:, lo:hi], ref["dX"][:, lo:hi]) <= 1e-4, (lo, hi)


# ---------------------------------------------------------------------------------------------------------------
# Batches of several 128-row tiles with index rows that put whole groups into one half of the feature range, one slot
# apart from the rest, runs across the middle of the range, duplicates and unsorted rows, and enough groups that a
# CTA's stripe holds many of them (written for the round-2 cluster kernel, kept as parity cases of the product kernel).
# ---------------------------------------------------------------------------------------------------------------
def _pair_idx(rng, NG, K, d, kind):
    half = (d + 1) // 2
    idx = np.empty((NG, K), dtype=np.int32)
    for g in range(NG):
        mode = g % 8 if kind == "mixed" else 0
        if mode == 0:      # strictly increasing, uniform
            row = np.sort(rng.choice(d, size=K, replace=False))
        elif mode == 1:    # consecutive run straddling the boundary between the two CTAs
            lo = max(0, min(d - K, half - K // 2 - (g % 5)))
            row = np.arange(lo, lo + K)
        elif mode == 2:    # everything in the FIRST CTA's half (its jobs: ceil(K / 48); the other CTA has none)
            row = np.sort(rng.choice(min(half, d), size=K, replace=False)) if half >= K else np.arange(K)
        elif mode == 3:    # everything in the SECOND CTA's half, at the top (L class when the half is large)
            row = np.arange(d - K, d)
        elif mode == 4:    # duplicates (sorted, not strict): split by position, atomic path
            row = np.sort(rng.choice(d, size=K, replace=True))
            row[K // 2] = row[K // 2 - 1]
        elif mode == 5:    # unsorted, distinct
            row = rng.permutation(d)[:K]
            if np.all(np.diff(row) > 0):
                row = row[::-1]
        elif mode == 6:    # consecutive run from a random start: hits the T/S and S/L boundaries of either half over the groups
            lo = rng.randint(0, d - K + 1)
            row = np.arange(lo, lo + K)
        elif d - half < K - 1:
            row = np.sort(rng.choice(d, size=K, replace=False))
        else:              # one slot in the first half, the rest in the second
            row = np.concatenate([[rng.randint(0, half)], np.sort(half + rng.choice(d - half, size=K - 1, replace=False))])
        idx[g] = row
    return idx


PAIR_CASES = [
    # B, d, NG (L = G*NG - 5), G, K, kind
    (300, 768, 23, 64, 128, "mixed"),     # config-3 shape; second 256-row tile ragged (44 rows)
    (600, 768, 100, 64, 128, "mixed"),    # 300 units on 74 pairs: a pair's range crosses tile boundaries (flush + clear)
    (256, 1024, 90, 64, 64, "mixed"),     # config-4 shape: one full tile, d = 1024, one job per unit
    (257, 768, 40, 64, 128, "strict"),
    (200, 768, 41, 32, 64, "mixed"),      # G = 32: 64-byte-swizzle dY image
    (130, 768, 13, 32, 128, "mixed"),
    (384, 768, 19, 128, 128, "mixed"),    # G = 128: two k-blocks per tile
    (129, 400, 11, 128, 64, "mixed"),     # d = 400: both halves fit on chip, no L class
    (512, 96, 9, 64, 64, "mixed"),        # d < 2K: every feature in most groups
]


@pytest.mark.parametrize("case", PAIR_CASES, ids=lambda c: "B%d_d%d_NG%d_G%d_K%d_%s" % c)
def test_dx_multi_tile_exact_and_close(oracle, case):
    from paper_2606_01117_b200 import haste
    from gpu_util import TailRun, dy_rounded
    B, d, NG, G, K, kind = case
    L = G * NG - 5
    inp = synth.small_case(300 + B + d, B, d, L, G, K, dtype="bf16", with_bias=False, w_std=0.05)
    rng = np.random.RandomState(B + d + K + 1)
    inp.idx = _pair_idx(rng, NG, K, d, kind)
    flags = haste.HASTE_IDX_SORTED_DISTINCT if kind == "strict" else 0

    Wi = rng.randint(-4, 5, size=(L, K)).astype(np.float32)
    Xi = rng.randint(-4, 5, size=(B, d)).astype(np.float32)
    dYi = rng.randint(-3, 4, size=(B, L)).astype(np.float32)
    inp.X, inp.W = Xi, Wi
    inp.bits["X"], inp.bits["W"] = synth.round_bf16(Xi)[0].reshape(B, d), synth.round_bf16(Wi)[0].reshape(L, K)
    run = TailRun(inp, G, flags=flags, dw_dtype="f32")
    assert run.layer.kernel_family == 1
    out = run.backward(dY_BL=dYi)
    ref = oracle.tail_backward(inp.X, inp.idx, inp.W, dYi.astype(np.float64), G)
    bad = np.argwhere(out["dX"].astype(np.float64) != ref["dX"])
    assert bad.size == 0, (bad[:8].tolist(), len(bad))
    out2 = run.backward(dY_BL=dYi)
    assert np.array_equal(out2["dX"], out["dX"])
    # accumulate_dX through the workspace layout
    base = rng.randint(-5, 6, size=(B, d)).astype(np.float32)
    out3 = run.backward(dY_BL=dYi, accumulate_into=base)
    assert np.array_equal(out3["dX"].astype(np.float64), ref["dX"] + base)

    Wr = (rng.standard_normal((L, K)) * 0.05).astype(np.float32)
    dYr = (rng.standard_normal((B, L)) / B).astype(np.float32)
    bits, Wr = synth.round_bf16(Wr)
    inp.W, inp.bits["W"] = Wr.reshape(L, K), bits.reshape(L, K)
    run = TailRun(inp, G, flags=flags, dw_dtype="f32")
    dYq = dy_rounded(inp, dYr)
    out = run.backward(dY_BL=dYq)
    ref = oracle.tail_backward(inp.X, inp.idx, inp.W, dYq.astype(np.float64), G)
    assert oracle.rel_l2(out["dX"], ref["dX"]) <= 1e-4
    for lo in range(0, d, 64):     # every 64-feature slice on its own: a class that dropped its adds cannot hide in the global norm
        hi = min(d, lo + 64)
        if np.linalg.norm(ref["dX"][:, lo:hi]) > 0:
            assert oracle.rel_l2(out["dX"][:, lo:hi], ref["dX"][:, lo:hi]) <= 1e-4, (lo, hi)
