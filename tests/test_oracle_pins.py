"""Pins of the fp64 CPU oracle (oracle/) against what the paper and the mathematics fix.

None of these retypes the oracle's own loops in the oracle's own form: each compares it with a
closed form, an independent statement (dense brute force, numpy matmul, per-label loop), an
invariant, or a finite difference of its own loss.  CPU only (-m "not gpu").
Pin numbering follows DESIGN.md "Oracle pins".
"""
import math
import os

import numpy as np
import pytest

from paper_2606_01117_b200 import synth

HERE = os.path.dirname(os.path.abspath(__file__))


def _close(a, b, tol=1e-12):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    scale = max(1.0, float(np.max(np.abs(b))) if b.size else 1.0)
    assert a.shape == b.shape
    assert float(np.max(np.abs(a - b))) <= tol * scale, float(np.max(np.abs(a - b)))


def _dense_targets(B, L, rowptr, col, off=0):
    Y = np.zeros((B, L))
    for i in range(B):
        for p in range(rowptr[i], rowptr[i + 1]):
            l = int(col[p]) - off
            if 0 <= l < L:
                Y[i, l] = 1.0
    return Y


# ---------------------------------------------------------------- golden worked example
def _load_golden():
    d = {}
    with open(os.path.join(HERE, "golden", "worked_example.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            d[k] = np.array([float(x) for x in v])
    return d


def test_golden_worked_example(oracle):
    """Hand-derived closed-form example (tests/golden/worked_example.txt)."""
    g = _load_golden()
    X = g["X"].reshape(2, 3).astype(np.float32)
    W = g["W"].reshape(2, 2).astype(np.float32)
    idx = g["idx"].astype(np.int32).reshape(1, 2)
    rowptr = g["rowptr"].astype(np.int32)
    col = g["col"].astype(np.int32)
    for fn in (oracle.tail_forward, oracle.bruteforce):
        r = fn(X, idx, W, None, rowptr, col, 2)
        # X is fp32 (ln 3, ln 4 rounded to fp32), so agreement is to fp32 rounding of the inputs
        _close(r["z"].ravel(), g["z"], 1e-7)
        assert abs(r["loss"] - g["loss"][0]) < 1e-7
        _close(r["dY"].ravel(), g["dY"], 1e-7)
    f = oracle.tail_forward(X, idx, W, None, rowptr, col, 2)
    b = oracle.tail_backward(X, idx, W, f["dY"], 2)
    _close(b["dW"].ravel(), g["dW"], 1e-7)
    _close(b["db"].ravel(), g["db"], 1e-7)
    _close(b["dX"].ravel(), g["dX"], 1e-7)
    bf = oracle.bruteforce(X, idx, W, None, rowptr, col, 2)
    _close(bf["dW"].ravel(), g["dW"], 1e-7)
    _close(bf["dX"].ravel(), g["dX"], 1e-7)


def test_scalar_closed_forms(oracle):
    """softplus(ln n) = ln(n+1), sigma(ln n) = n/(n+1); symmetric identities; no overflow (reading R5)."""
    for n in (1, 2, 3, 4, 9, 1000):
        assert abs(oracle.softplus(math.log(n)) - math.log(n + 1)) < 1e-14
        assert abs(oracle.sigmoid(math.log(n)) - n / (n + 1)) < 1e-15
    for z in (-700.0, -30.0, -1.5, 0.0, 0.3, 40.0, 800.0, 1e4):
        assert math.isfinite(oracle.softplus(z)) and math.isfinite(oracle.sigmoid(z))
        assert abs(oracle.softplus(z) - oracle.softplus(-z) - z) <= 1e-12 * max(1, abs(z))
        assert abs(oracle.sigmoid(z) + oracle.sigmoid(-z) - 1.0) < 1e-15
    assert oracle.softplus(1e4) == 1e4 and oracle.softplus(-1e4) == 0.0 or oracle.softplus(-1e4) < 1e-300


# ---------------------------------------------------------------- P1 brute force O1 == O2
CASES = [
    # B, d, L, G, K, sorted_distinct
    (5, 16, 24, 4, 8, True),
    (3, 12, 23, 4, 6, True),      # partial last group (23 = 5*4 + 3)
    (7, 32, 64, 16, 8, True),
    (4, 9, 10, 1, 3, True),       # G = 1
    (6, 10, 21, 8, 10, True),     # K = d
    (5, 8, 19, 4, 12, False),     # K > d forces duplicates; unsorted (reading R4)
    (2, 20, 33, 32, 5, False),
]


@pytest.mark.parametrize("B,d,L,G,K,sd", CASES)
def test_p1_bruteforce_equals_direct(oracle, B, d, L, G, K, sd):
    c = synth.small_case(11 + L, B, d, L, G, K, sorted_distinct=sd, with_bias=True, n_pos=2)
    o1 = oracle.bruteforce(c.X, c.idx, c.W, c.bias, c.rowptr, c.col, G)
    f = oracle.tail_forward(c.X, c.idx, c.W, c.bias, c.rowptr, c.col, G)
    b = oracle.tail_backward(c.X, c.idx, c.W, f["dY"], G)
    assert abs(o1["loss"] - f["loss"]) <= 1e-12 * abs(o1["loss"])
    _close(f["z"], o1["z"]); _close(f["dY"], o1["dY"])
    _close(b["dW"], o1["dW"]); _close(b["db"], o1["db"]); _close(b["dX"], o1["dX"])


def test_p1_numpy_dense_masked(oracle):
    """A third opinion: the dense masked W_full built with numpy and an ordinary dense layer via np.matmul."""
    B, d, L, G, K = 6, 14, 27, 4, 5
    c = synth.small_case(3, B, d, L, G, K, with_bias=True, n_pos=3)
    Wf = np.zeros((L, d))
    for l in range(L):
        for j in range(K):
            Wf[l, c.idx[l // G, j]] += float(c.W[l, j])
    X = c.X.astype(np.float64)
    Z = X @ Wf.T + c.bias.astype(np.float64)[None, :]
    Y = _dense_targets(B, L, c.rowptr, c.col)
    loss = (np.logaddexp(0.0, Z) - Y * Z).sum() / B
    dY = (1.0 / (1.0 + np.exp(-Z)) - Y) / B
    f = oracle.tail_forward(c.X, c.idx, c.W, c.bias, c.rowptr, c.col, G)
    b = oracle.tail_backward(c.X, c.idx, c.W, f["dY"], G)
    assert abs(f["loss"] - loss) < 1e-12 * abs(loss)
    _close(f["z"], Z); _close(f["dY"], dY)
    _close(b["dX"], dY @ Wf)
    dWf = dY.T @ X
    _close(b["dW"], np.stack([dWf[l, c.idx[l // G]] for l in range(L)]))
    _close(b["db"], dY.sum(0))


# ---------------------------------------------------------------- P2 G = 1: ordinary per-label fixed fan-in
def test_p2_g1_is_per_label_fixed_fan_in(oracle):
    """With G=1 every label owns its index row: z[i,l] = sum_j W[l,j] X[i, idx[l,j]]."""
    B, d, L, K = 5, 18, 13, 7
    c = synth.small_case(5, B, d, L, 1, K, with_bias=False)
    z = np.einsum("lj,ilj->il", c.W.astype(np.float64), c.X.astype(np.float64)[:, c.idx])
    f = oracle.tail_forward(c.X, c.idx, c.W, None, c.rowptr, c.col, 1)
    _close(f["z"], z)
    # and grouping = repeating the index row G times
    G = 4
    cg = synth.small_case(6, B, d, 12, G, K, with_bias=True)
    idx_rep = np.repeat(cg.idx, G, axis=0)[:12]
    fg = oracle.tail_forward(cg.X, cg.idx, cg.W, cg.bias, cg.rowptr, cg.col, G)
    f1 = oracle.tail_forward(cg.X, idx_rep, cg.W, cg.bias, cg.rowptr, cg.col, 1)
    _close(fg["z"], f1["z"]); _close(fg["dY"], f1["dY"])
    bg = oracle.tail_backward(cg.X, cg.idx, cg.W, fg["dY"], G)
    b1 = oracle.tail_backward(cg.X, idx_rep, cg.W, f1["dY"], 1)
    _close(bg["dW"], b1["dW"]); _close(bg["dX"], b1["dX"])


# ---------------------------------------------------------------- P3 K = d: a dense layer
def test_p3_full_support_is_dense_layer(oracle):
    """K = d, idx = 0..d-1 reduces to the textbook dense layer X W^T; also pins the head."""
    B, d, L, G = 6, 10, 20, 4
    c = synth.small_case(9, B, d, L, G, d, with_bias=True)
    assert (c.idx == np.arange(d)[None, :]).all()
    X = c.X.astype(np.float64); W = c.W.astype(np.float64)
    Z = X @ W.T + c.bias.astype(np.float64)
    f = oracle.tail_forward(c.X, c.idx, c.W, c.bias, c.rowptr, c.col, G)
    _close(f["z"], Z)
    b = oracle.tail_backward(c.X, c.idx, c.W, f["dY"], G)
    _close(b["dW"], f["dY"].T @ X); _close(b["dX"], f["dY"] @ W)
    h = oracle.head_forward(c.X, c.W, c.bias, c.rowptr, c.col)
    assert abs(h["loss"] - f["loss"]) < 1e-12 * abs(f["loss"])
    _close(h["z"], Z); _close(h["dY"], f["dY"])
    hb = oracle.head_backward(c.X, c.W, h["dY"])
    _close(hb["dW"], f["dY"].T @ X); _close(hb["dX"], f["dY"] @ W); _close(hb["db"], f["dY"].sum(0))


# ---------------------------------------------------------------- P4 finite differences
def test_p4_finite_differences(oracle):
    B, d, L, G, K = 3, 7, 10, 4, 3
    c = synth.small_case(21, B, d, L, G, K, with_bias=True, n_pos=2, w_std=0.7, sorted_distinct=False)
    # exact-in-fp32 perturbation: inputs are multiples of 2^-10 so +-h with h = 2^-10 stays exact
    q = lambda a: (np.round(a * 1024) / 1024).astype(np.float32)
    X, W, bias = q(c.X), q(c.W), q(c.bias)
    h = 1.0 / 1024

    def loss(X_, W_, b_):
        return oracle.tail_forward(X_, c.idx, W_, b_, c.rowptr, c.col, G, want_z=False, want_dY=False)["loss"]

    f = oracle.tail_forward(X, c.idx, W, bias, c.rowptr, c.col, G)
    bk = oracle.tail_backward(X, c.idx, W, f["dY"], G)

    def fd(arr, pos, which):
        # 4th-order central difference (error O(h^4) ~ 1e-12 * derivative scale)
        vals = []
        for k in (-2, -1, 1, 2):
            a = arr.copy(); a[pos] += np.float32(k * h)
            args = dict(X=X, W=W, b=bias); args[which] = a
            vals.append(loss(args["X"], args["W"], args["b"]))
        return (vals[0] - 8 * vals[1] + 8 * vals[2] - vals[3]) / (12 * h)

    for l in range(L):
        for j in range(K):
            assert abs(fd(W, (l, j), "W") - bk["dW"][l, j]) < 2e-9
        assert abs(fd(bias, (l,), "b") - bk["db"][l]) < 2e-9
    for i in range(B):
        for t in range(d):
            assert abs(fd(X, (i, t), "X") - bk["dX"][i, t]) < 2e-9


def test_p4_head_finite_differences(oracle):
    B, d, Lh = 3, 5, 6
    c = synth.small_case(22, B, d, Lh, 1, d, with_bias=True, n_pos=2, w_std=0.7)
    q = lambda a: (np.round(a * 1024) / 1024).astype(np.float32)
    X, W, bias = q(c.X), q(c.W), q(c.bias)
    h = 1.0 / 1024
    f = oracle.head_forward(X, W, bias, c.rowptr, c.col)
    bk = oracle.head_backward(X, W, f["dY"])
    L0 = lambda X_, W_, b_: oracle.head_forward(X_, W_, b_, c.rowptr, c.col, want_z=False, want_dY=False)["loss"]
    for (arr, name, grad) in ((W, "W", bk["dW"]), (X, "X", bk["dX"]), (bias, "b", bk["db"])):
        for pos in np.ndindex(arr.shape):
            v = []
            for k in (-2, -1, 1, 2):
                a = arr.copy(); a[pos] += np.float32(k * h)
                args = dict(X=X, W=W, b=bias); args[name] = a
                v.append(L0(args["X"], args["W"], args["b"]))
            assert abs((v[0] - 8 * v[1] + 8 * v[2] - v[3]) / (12 * h) - grad[pos]) < 2e-9


# ---------------------------------------------------------------- P5 W = 0 closed form
def test_p5_zero_weights_closed_form(oracle):
    B, d, L, G, K = 8, 16, 30, 4, 6
    c = synth.small_case(31, B, d, L, G, K, with_bias=False, n_pos=3)
    W0 = np.zeros_like(c.W)
    f = oracle.tail_forward(c.X, c.idx, W0, None, c.rowptr, c.col, G)
    s = 1.0 / B
    assert abs(f["loss"] - s * B * L * math.log(2.0)) < 1e-12
    Y = _dense_targets(B, L, c.rowptr, c.col)
    assert Y.sum() == 3 * B
    _close(f["dY"], s * (0.5 - Y))
    b = oracle.tail_backward(c.X, c.idx, W0, f["dY"], G)
    assert np.all(b["dX"] == 0.0)
    X = c.X.astype(np.float64)
    exp = np.stack([(s * (0.5 - Y[:, l]))[:, None] * X[:, c.idx[l // G]] for l in range(L)]).sum(1)
    _close(b["dW"], exp)


def test_targets_offset_and_out_of_range_ids(oracle):
    """Reading R7: CSR columns are global ids; ids outside [off, off+L) are ignored; repeated id counts once."""
    B, d, L, G, K = 4, 8, 12, 4, 4
    c = synth.small_case(41, B, d, L, G, K, with_bias=False, n_pos=2)
    off = 100
    rowptr = np.array([0, 3, 5, 5, 7], dtype=np.int32)
    col = np.array([5, 100, 111, 103, 103, 99, 112], dtype=np.int32)   # in-range: (0,0),(0,11),(1,3) only
    f = oracle.tail_forward(c.X, c.idx, c.W, None, rowptr, col, G, label_offset=off)
    f0 = oracle.tail_forward(c.X, c.idx, c.W, None, np.zeros(B + 1, np.int32), np.zeros(0, np.int32), G)
    diff = (f0["dY"] - f["dY"]) * B
    exp = np.zeros((B, L)); exp[0, 0] = exp[0, 11] = exp[1, 3] = 1.0
    _close(diff, exp)
    assert abs((f0["loss"] - f["loss"]) * B - (f["z"][0, 0] + f["z"][0, 11] + f["z"][1, 3])) < 1e-12


# ---------------------------------------------------------------- P6 Euler identities
def test_p6_euler_identities(oracle):
    """z - b is bilinear in (X, W): sum_f X dX = sum_l dY (z-b) per row; sum_j W dW = sum_i dY (z-b) per label."""
    B, d, L, G, K = 6, 20, 37, 8, 9
    c = synth.small_case(51, B, d, L, G, K, with_bias=True, sorted_distinct=False)
    f = oracle.tail_forward(c.X, c.idx, c.W, c.bias, c.rowptr, c.col, G)
    b = oracle.tail_backward(c.X, c.idx, c.W, f["dY"], G)
    zb = f["z"] - c.bias.astype(np.float64)[None, :]
    _close((c.X.astype(np.float64) * b["dX"]).sum(1), (f["dY"] * zb).sum(1))
    _close((c.W.astype(np.float64) * b["dW"]).sum(1), (f["dY"] * zb).sum(0))


# ---------------------------------------------------------------- P8 slot permutation, P9 duplicate additivity
def test_p8_slot_permutation_invariance(oracle):
    B, d, L, G, K = 5, 16, 16, 4, 6
    c = synth.small_case(61, B, d, L, G, K, with_bias=True)
    perm = np.array([3, 0, 5, 1, 4, 2])
    idx2 = c.idx.copy(); W2 = c.W.copy()
    idx2[1] = c.idx[1][perm]; W2[4:8] = c.W[4:8][:, perm]
    f = oracle.tail_forward(c.X, c.idx, c.W, c.bias, c.rowptr, c.col, G)
    f2 = oracle.tail_forward(c.X, idx2, W2, c.bias, c.rowptr, c.col, G)
    _close(f2["z"], f["z"], 1e-14)
    b = oracle.tail_backward(c.X, c.idx, c.W, f["dY"], G)
    b2 = oracle.tail_backward(c.X, idx2, W2, f["dY"], G)
    _close(b2["dX"], b["dX"], 1e-14)
    exp = b["dW"].copy(); exp[4:8] = b["dW"][4:8][:, perm]
    _close(b2["dW"], exp, 1e-14)


def test_p9_duplicate_index_additivity(oracle):
    B, d, L, G, K = 4, 12, 8, 4, 5
    c = synth.small_case(71, B, d, L, G, K, with_bias=False)
    W = (np.round(c.W * 64) / 64).astype(np.float32)       # exact sums in fp32
    idx_dup = c.idx.copy(); idx_dup[0, 3] = c.idx[0, 1]     # slot 3 now repeats slot 1's feature
    # equivalent distinct-support layer: slot 1 carries W[:,1]+W[:,3]; slot 3 points anywhere with weight 0
    W_eq = W.copy(); W_eq[0:4, 1] = W[0:4, 1] + W[0:4, 3]; W_eq[0:4, 3] = 0.0
    f = oracle.tail_forward(c.X, idx_dup, W, None, c.rowptr, c.col, G)
    g = oracle.tail_forward(c.X, c.idx, W_eq, None, c.rowptr, c.col, G)
    _close(f["z"], g["z"], 1e-14)
    b = oracle.tail_backward(c.X, idx_dup, W, f["dY"], G)
    g_b = oracle.tail_backward(c.X, c.idx, W_eq, f["dY"], G)
    _close(b["dX"], g_b["dX"], 1e-14)
    _close(b["dW"][0:4, 3], b["dW"][0:4, 1], 0.0)          # both slots see the same feature column


# ---------------------------------------------------------------- sampled statements agree with the full ones
def test_sampled_statements_match_full(oracle):
    B, d, L, G, K = 6, 24, 45, 8, 7
    off = 17
    c = synth.small_case(81, B, d, L, G, K, with_bias=True, label_offset=off, n_pos=4)
    f = oracle.tail_forward(c.X, c.idx, c.W, c.bias, c.rowptr, c.col, G, label_offset=off)
    b = oracle.tail_backward(c.X, c.idx, c.W, f["dY"], G)
    rows = np.array([0, 5, 2, 2], dtype=np.int32); labels = np.array([44, 0, 13, 40], dtype=np.int64)
    p = oracle.tail_points(c.X, c.idx, c.W, c.bias, c.rowptr, c.col, G, rows, labels, label_offset=off)
    _close(p["z"], f["z"][rows, labels]); _close(p["dY"], f["dY"][rows, labels])
    lr = oracle.tail_label_rows(c.X, c.idx, c.W, c.bias, c.rowptr, c.col, G, labels, label_offset=off)
    _close(lr["dYcol"], f["dY"][:, labels].T); _close(lr["dW"], b["dW"][labels]); _close(lr["db"], b["db"][labels])
    br = oracle.tail_batch_rows(c.X, c.idx, c.W, c.bias, c.rowptr, c.col, G, rows[:3], label_offset=off)
    _close(br["dX"], b["dX"][rows[:3]])
    allr = oracle.tail_batch_rows(c.X, c.idx, c.W, c.bias, c.rowptr, c.col, G, np.arange(B, dtype=np.int32),
                                  label_offset=off, want_dX=False)
    assert abs(allr["loss_rows"].sum() - f["loss"]) < 1e-12 * abs(f["loss"])


def test_oracle_rejects_bad_index(oracle):
    c = synth.small_case(91, 2, 8, 8, 4, 4)
    bad = c.idx.copy(); bad[1, 2] = 8
    with pytest.raises(ValueError):
        oracle.tail_forward(c.X, bad, c.W, None, c.rowptr, c.col, 4)


# ---------------------------------------------------------------- P10 expected value at the paper-shaped distribution
def test_p10_expected_softplus_scale(oracle):
    """X~N(0,1), W~N(0,0.02^2): E[softplus(z)] ~ ln2 + K*0.02^2/8 (second-order expansion), s = 1/B."""
    cfg = synth.Config("p10", 0, B=64, d=128, L=2048, L_h=0, G=16, K=32, dtype="f32", n_fixed=3)
    inp = synth.make_inputs(cfg)
    f = oracle.tail_forward(inp.X, inp.idx, inp.W, None, inp.rowptr, inp.col, cfg.G, want_z=True, want_dY=False)
    per_logit = (f["loss"] * cfg.B + f["z"][_dense_targets(cfg.B, cfg.L, inp.rowptr, inp.col) > 0].sum()) / (cfg.B * cfg.L)
    assert abs(per_logit - (math.log(2.0) + cfg.K * 0.02 ** 2 / 8)) < 2e-4


# ------------------------------------------------------------------------------------------------------------------
# SGD with momentum on the output layer (heavy-ball form, reading R13)
# ------------------------------------------------------------------------------------------------------------------
def test_sgd_momentum_closed_forms(oracle):
    rng = np.random.RandomState(11)
    w0 = rng.standard_normal((7, 5))
    g = rng.standard_normal((7, 5))
    lr, mu = 0.1, 0.9
    # mu = 0, wd = 0: plain gradient descent
    w1, v1 = oracle.sgd_momentum(w0, g, np.zeros_like(w0), lr, 0.0)
    assert np.allclose(w1, w0 - lr * g, rtol=0, atol=1e-15) and np.allclose(v1, g, rtol=0, atol=0)
    # constant gradient, n steps from v = 0:  v_n = g (1 - mu^n) / (1 - mu),  w_n = w_0 - lr g sum_{t=1..n} (1 - mu^t) / (1 - mu)
    w, v = w0.copy(), np.zeros_like(w0)
    for n in range(1, 6):
        w, v = oracle.sgd_momentum(w, g, v, lr, mu)
        assert np.allclose(v, g * (1 - mu ** n) / (1 - mu), rtol=1e-13, atol=0)
        assert np.allclose(w, w0 - lr * g * sum((1 - mu ** t) / (1 - mu) for t in range(1, n + 1)), rtol=1e-12, atol=1e-14)
        if n == 2:
            assert np.allclose(w, w0 - lr * g * (2 + mu), rtol=1e-13, atol=1e-15)      # the two-step form, by hand
    # g = 0, mu = 0: weight decay alone shrinks w by (1 - lr wd)
    w1, _ = oracle.sgd_momentum(w0, np.zeros_like(w0), np.zeros_like(w0), lr, 0.0, wd=0.05)
    assert np.allclose(w1, w0 * (1 - lr * 0.05), rtol=1e-15, atol=0)
    # a hand-computed scalar: w = 2, g = 0.5, v = 1, lr = 0.1, mu = 0.9, wd = 0.01 -> g' = 0.52, v' = 1.42, w' = 1.858
    w1, v1 = oracle.sgd_momentum(np.array([2.0]), np.array([0.5]), np.array([1.0]), 0.1, 0.9, wd=0.01)
    assert abs(v1[0] - 1.42) < 1e-15 and abs(w1[0] - 1.858) < 1e-15
    # the sign of the step: a positive gradient lowers the weight
    assert oracle.sgd_momentum(np.array([0.0]), np.array([1.0]), np.array([0.0]), 1.0, 0.5)[0][0] == -1.0


# ------------------------------------------------------------------------------------------------------------------
# Algorithm 3, group-shared rewiring
# ------------------------------------------------------------------------------------------------------------------
def test_rewire_generator_is_splitmix64(oracle):
    # SplitMix64 seeded with 0: the published first outputs of the reference generator (state += golden ratio, then mix)
    assert oracle.rewire_mix(0, 0) == 0xE220A8397B1DCDAF
    assert oracle.rewire_mix(0, 1) == 0x6E789E6AA1B965F4
    assert oracle.rewire_mix(0, 2) == 0x06C45D188009454F


def _rw_case(seed, L, G, K, d, w_std=0.3):
    inp = synth.small_case(seed, 4, d, L, G, K, dtype="f32", w_std=w_std, with_bias=False)
    return inp


@pytest.mark.parametrize("L,G,K,d", [(64 * 5 + 7, 64, 16, 40), (37, 8, 8, 24), (16 * 9, 16, 32, 64)])
def test_rewire_properties(oracle, L, G, K, d):
    inp = _rw_case(3, L, G, K, d)
    NG = -(-L // G)
    rho = 0.2
    out = oracle.rewire(inp.idx, inp.W, G, d, rho, init_random=False, seed=77, resort=False)
    m = int(np.floor(NG * K * rho))
    assert out["m"] == m and int(out["mask"].sum()) == m                       # exactly floor(NG K rho) slots
    # scores: the mean of |w| over the group's labels, against numpy in fp64 -- the fp32 order of additions moves
    # a score by a few ulp, it cannot move it further
    for k in range(NG):
        rows = inp.W[k * G:min(L, (k + 1) * G)]
        assert np.allclose(out["scores"][k], np.abs(rows.astype(np.float64)).mean(axis=0), rtol=1e-5, atol=0)
    # the mask holds the m smallest: nothing left out is smaller than anything taken
    S, M = out["scores"].ravel(), out["mask"].ravel().astype(bool)
    assert S[M].max() <= S[~M].min()
    # untouched slots keep idx and weights; touched slots: idx in range, weights zero for EVERY label of the group
    keep = ~out["mask"].astype(bool)
    assert np.array_equal(out["idx"][keep], inp.idx[keep])
    assert np.all((out["idx"] >= 0) & (out["idx"] < d))
    lab_mask = np.repeat(out["mask"], G, axis=0)[:L].astype(bool)
    assert np.all(out["W"][lab_mask] == 0) and np.array_equal(out["W"][~lab_mask], inp.W[~lab_mask])
    # the regrown feature is floor(d * h / 2^64) of the generator's word for that slot (Unif{0..H-1})
    for k, j in np.argwhere(out["mask"])[:20]:
        h = oracle.rewire_mix(77, int(k) * K + int(j))
        assert out["idx"][k, j] == (h * d) >> 64
    # zero-initialised slots contribute nothing: the layer computes what the old one computed with those weights zeroed
    z_new = oracle.tail_forward(inp.X, out["idx"], out["W"], None, inp.rowptr, inp.col, G)["z"]
    z_old = oracle.tail_forward(inp.X, inp.idx, np.where(lab_mask, 0.0, inp.W).astype(np.float32), None, inp.rowptr, inp.col, G)["z"]
    assert np.allclose(z_new, z_old, rtol=0, atol=1e-12)
    # rho = 0: nothing happens
    out0 = oracle.rewire(inp.idx, inp.W, G, d, 0.0)
    assert out0["m"] == 0 and np.array_equal(out0["idx"], inp.idx) and np.array_equal(out0["W"], inp.W)


def test_rewire_random_init_and_resort(oracle):
    L, G, K, d = 64 * 4 + 9, 64, 32, 200
    inp = _rw_case(5, L, G, K, d)
    mom = np.ones((L, K), dtype=np.float32)
    a = oracle.rewire(inp.idx, inp.W, G, d, 0.3, init_random=True, seed=9, resort=False, momentum=mom)
    b = oracle.rewire(inp.idx, inp.W, G, d, 0.3, init_random=True, seed=9, resort=True, momentum=mom)
    lab_mask = np.repeat(a["mask"], G, axis=0)[:L].astype(bool)
    r = 1.0 / np.sqrt(K)
    w = a["W"][lab_mask]
    assert np.all(np.abs(w) <= r) and abs(w.mean()) < 0.1 * r and w.std() > 0.4 * r   # Unif(-1/sqrt(F), 1/sqrt(F))
    assert np.all(a["momentum"][lab_mask] == 0) and np.all(a["momentum"][~lab_mask] == 1)
    # resort: every touched row ascending, same multiset of (feature, weight column) pairs, same function (pin P8)
    touched = a["mask"].any(axis=1)
    assert np.all(np.diff(b["idx"][touched], axis=1) >= 0)
    assert np.array_equal(np.sort(a["idx"], axis=1), np.sort(b["idx"], axis=1))
    za = oracle.tail_forward(inp.X, a["idx"], a["W"], None, inp.rowptr, inp.col, G)["z"]
    zb = oracle.tail_forward(inp.X, b["idx"], b["W"], None, inp.rowptr, inp.col, G)["z"]
    assert np.allclose(za, zb, rtol=0, atol=1e-12)
    assert np.array_equal(b["idx"][~touched], inp.idx[~touched])
    # ties: with all-equal scores the flat index decides -- the first m slots go
    Wc = np.full((L, K), 0.25, dtype=np.float32)
    t = oracle.rewire(inp.idx, Wc, G, d, 0.1, resort=False)
    assert np.array_equal(np.flatnonzero(t["mask"].ravel()), np.arange(t["m"]))
