"""ctypes front end of the fp64 CPU oracle (oracle/haste_oracle.cpp).

TEST INFRASTRUCTURE, not the product: argument marshalling only; every number is
computed by the C++ file, which states the paper passage each loop follows
(PAPER.md:72, :97-103, :107-111).  Inputs are numpy arrays; float inputs are
taken as float32 (bf16 configs pass the bf16-rounded values widened exactly),
all arithmetic and all outputs are float64.
"""
import ctypes
import numpy as np

from . import build as _build

__all__ = [
    "tail_forward", "tail_backward", "bruteforce", "head_forward", "head_backward",
    "tail_points", "tail_label_rows", "tail_batch_rows", "sgd_momentum", "rewire", "rewire_mix", "softplus", "sigmoid", "rel_l2",
]

_lib = None


def _L():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        _lib.haste_oracle_softplus.restype = ctypes.c_double
        _lib.haste_oracle_softplus.argtypes = [ctypes.c_double]
        _lib.haste_oracle_sigmoid.restype = ctypes.c_double
        _lib.haste_oracle_sigmoid.argtypes = [ctypes.c_double]
    return _lib


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _i64(a):
    return np.ascontiguousarray(a, dtype=np.int64)


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _chk(rc):
    if rc != 0:
        raise ValueError("oracle: index out of range (rc=%d)" % rc)


def softplus(z):
    return _L().haste_oracle_softplus(float(z))


def sigmoid(z):
    return _L().haste_oracle_sigmoid(float(z))


def rel_l2(a, ref):
    """||a - ref||_2 / ||ref||_2 in fp64 (absolute norm when ||ref|| = 0)."""
    a = np.asarray(a, dtype=np.float64).ravel()
    ref = np.asarray(ref, dtype=np.float64).ravel()
    den = np.linalg.norm(ref)
    num = np.linalg.norm(a - ref)
    return num / den if den > 0 else num


def _dims(X, idx, W, G):
    B, d = X.shape
    L, K = W.shape
    NG = -(-L // G)
    assert idx.shape == (NG, K), (idx.shape, NG, K)
    return B, d, L, K


def tail_forward(X, idx, W, bias, rowptr, col, G, label_offset=0, s=None, want_z=True, want_dY=True):
    """O2 forward.  Returns dict(loss, z [B,L] | None, dY [B,L] | None)."""
    X, W, bias = _f32(X), _f32(W), _f32(bias)
    idx, rowptr, col = _i32(idx), _i32(rowptr), _i32(col)
    B, d, L, K = _dims(X, idx, W, G)
    s = 1.0 / B if s is None else float(s)
    loss = ctypes.c_double(0.0)
    z = np.empty((B, L), dtype=np.float64) if want_z else None
    dY = np.empty((B, L), dtype=np.float64) if want_dY else None
    _chk(_L().haste_oracle_tail_forward(
        ctypes.c_int(B), ctypes.c_int(d), ctypes.c_int64(L), ctypes.c_int(G), ctypes.c_int(K),
        _p(X), _p(idx), _p(W), _p(bias), _p(rowptr), _p(col), ctypes.c_int64(label_offset),
        ctypes.c_double(s), ctypes.byref(loss), _p(z), _p(dY)))
    return dict(loss=loss.value, z=z, dY=dY)


def tail_backward(X, idx, W, dY, G, want_db=True):
    """O2 backward from dY [B,L] fp64.  Returns dict(dW [L,K], db [L] | None, dX [B,d])."""
    X, W = _f32(X), _f32(W)
    idx = _i32(idx)
    B, d, L, K = _dims(X, idx, W, G)
    dY = np.ascontiguousarray(dY, dtype=np.float64)
    assert dY.shape == (B, L)
    dW = np.empty((L, K), dtype=np.float64)
    db = np.empty((L,), dtype=np.float64) if want_db else None
    dX = np.empty((B, d), dtype=np.float64)
    _chk(_L().haste_oracle_tail_backward(
        ctypes.c_int(B), ctypes.c_int(d), ctypes.c_int64(L), ctypes.c_int(G), ctypes.c_int(K),
        _p(X), _p(idx), _p(W), _p(dY), _p(dW), _p(db), _p(dX)))
    return dict(dW=dW, db=db, dX=dX)


def bruteforce(X, idx, W, bias, rowptr, col, G, label_offset=0, s=None):
    """O1: dense masked W_full brute force (tiny only).  Returns loss, z, dY, dW, db, dX."""
    X, W, bias = _f32(X), _f32(W), _f32(bias)
    idx, rowptr, col = _i32(idx), _i32(rowptr), _i32(col)
    B, d, L, K = _dims(X, idx, W, G)
    if L * d > (1 << 24):
        raise ValueError("bruteforce is for tiny inputs")
    s = 1.0 / B if s is None else float(s)
    loss = ctypes.c_double(0.0)
    z = np.empty((B, L)); dY = np.empty((B, L)); dW = np.empty((L, K)); db = np.empty((L,)); dX = np.empty((B, d))
    _chk(_L().haste_oracle_bruteforce(
        ctypes.c_int(B), ctypes.c_int(d), ctypes.c_int64(L), ctypes.c_int(G), ctypes.c_int(K),
        _p(X), _p(idx), _p(W), _p(bias), _p(rowptr), _p(col), ctypes.c_int64(label_offset),
        ctypes.c_double(s), ctypes.byref(loss), _p(z), _p(dY), _p(dW), _p(db), _p(dX)))
    return dict(loss=loss.value, z=z, dY=dY, dW=dW, db=db, dX=dX)


def head_forward(X, Wh, bias, rowptr, col, label_offset=0, s=None, want_z=True, want_dY=True):
    X, Wh, bias = _f32(X), _f32(Wh), _f32(bias)
    rowptr, col = _i32(rowptr), _i32(col)
    B, d = X.shape
    Lh = Wh.shape[0]
    assert Wh.shape[1] == d
    s = 1.0 / B if s is None else float(s)
    loss = ctypes.c_double(0.0)
    z = np.empty((B, Lh)) if want_z else None
    dY = np.empty((B, Lh)) if want_dY else None
    _chk(_L().haste_oracle_head_forward(
        ctypes.c_int(B), ctypes.c_int(d), ctypes.c_int64(Lh), _p(X), _p(Wh), _p(bias), _p(rowptr), _p(col),
        ctypes.c_int64(label_offset), ctypes.c_double(s), ctypes.byref(loss), _p(z), _p(dY)))
    return dict(loss=loss.value, z=z, dY=dY)


def head_backward(X, Wh, dY, want_db=True):
    X, Wh = _f32(X), _f32(Wh)
    B, d = X.shape
    Lh = Wh.shape[0]
    dY = np.ascontiguousarray(dY, dtype=np.float64)
    assert dY.shape == (B, Lh)
    dWh = np.empty((Lh, d)); db = np.empty((Lh,)) if want_db else None; dX = np.empty((B, d))
    _chk(_L().haste_oracle_head_backward(
        ctypes.c_int(B), ctypes.c_int(d), ctypes.c_int64(Lh), _p(X), _p(Wh), _p(dY), _p(dWh), _p(db), _p(dX)))
    return dict(dW=dWh, db=db, dX=dX)


def tail_points(X, idx, W, bias, rowptr, col, G, rows, labels, label_offset=0, s=None):
    """Logit z and dY at n sampled (row, label) pairs."""
    X, W, bias = _f32(X), _f32(W), _f32(bias)
    idx, rowptr, col = _i32(idx), _i32(rowptr), _i32(col)
    B, d, L, K = _dims(X, idx, W, G)
    rows, labels = _i32(rows), _i64(labels)
    n = rows.shape[0]
    s = 1.0 / B if s is None else float(s)
    z = np.empty((n,)); dY = np.empty((n,))
    _chk(_L().haste_oracle_tail_points(
        ctypes.c_int(B), ctypes.c_int(d), ctypes.c_int64(L), ctypes.c_int(G), ctypes.c_int(K),
        _p(X), _p(idx), _p(W), _p(bias), _p(rowptr), _p(col), ctypes.c_int64(label_offset), ctypes.c_double(s),
        ctypes.c_int64(n), _p(rows), _p(labels), _p(z), _p(dY)))
    return dict(z=z, dY=dY)


def tail_label_rows(X, idx, W, bias, rowptr, col, G, labels, label_offset=0, s=None):
    """For n sampled labels: dY column [n,B], dW row [n,K], db [n] (fp64 end to end)."""
    X, W, bias = _f32(X), _f32(W), _f32(bias)
    idx, rowptr, col = _i32(idx), _i32(rowptr), _i32(col)
    B, d, L, K = _dims(X, idx, W, G)
    labels = _i64(labels)
    n = labels.shape[0]
    s = 1.0 / B if s is None else float(s)
    dYc = np.empty((n, B)); dW = np.empty((n, K)); db = np.empty((n,))
    _chk(_L().haste_oracle_tail_label_rows(
        ctypes.c_int(B), ctypes.c_int(d), ctypes.c_int64(L), ctypes.c_int(G), ctypes.c_int(K),
        _p(X), _p(idx), _p(W), _p(bias), _p(rowptr), _p(col), ctypes.c_int64(label_offset), ctypes.c_double(s),
        ctypes.c_int64(n), _p(labels), _p(dYc), _p(dW), _p(db)))
    return dict(dYcol=dYc, dW=dW, db=db)


def tail_batch_rows(X, idx, W, bias, rowptr, col, G, rows, label_offset=0, s=None, want_dX=True):
    """For n sampled batch rows: the row's loss term and its dX row [n,d], over ALL labels."""
    X, W, bias = _f32(X), _f32(W), _f32(bias)
    idx, rowptr, col = _i32(idx), _i32(rowptr), _i32(col)
    B, d, L, K = _dims(X, idx, W, G)
    rows = _i32(rows)
    n = rows.shape[0]
    s = 1.0 / B if s is None else float(s)
    lr = np.empty((n,)); dX = np.empty((n, d)) if want_dX else None
    _chk(_L().haste_oracle_tail_batch_rows(
        ctypes.c_int(B), ctypes.c_int(d), ctypes.c_int64(L), ctypes.c_int(G), ctypes.c_int(K),
        _p(X), _p(idx), _p(W), _p(bias), _p(rowptr), _p(col), ctypes.c_int64(label_offset), ctypes.c_double(s),
        ctypes.c_int64(n), _p(rows), _p(lr), _p(dX)))
    return dict(loss_rows=lr, dX=dX)


def sgd_momentum(w, g, v, lr, mu, wd=0.0):
    """One SGD-with-momentum step (heavy-ball form, reading R13) on arrays of any shape, fp64:
    v' = mu v + (g + wd w);  w' = w - lr v'.  Returns (w', v')."""
    w = np.ascontiguousarray(w, dtype=np.float64)
    g = np.ascontiguousarray(g, dtype=np.float64)
    v = np.ascontiguousarray(v, dtype=np.float64)
    assert w.shape == g.shape == v.shape
    w_out, v_out = np.empty_like(w), np.empty_like(v)
    _chk(_L().haste_oracle_sgd_momentum(ctypes.c_int64(w.size), _p(w), _p(g), _p(v), ctypes.c_double(lr), ctypes.c_double(mu),
                                        ctypes.c_double(wd), _p(w_out), _p(v_out)))
    return w_out, v_out


def rewire_mix(seed, counter):
    """The counter-based generator of the rewiring step (SplitMix64 finaliser), as a Python int."""
    f = _L().haste_oracle_rewire_mix
    f.restype = ctypes.c_uint64
    f.argtypes = [ctypes.c_uint64, ctypes.c_uint64]
    return int(f(seed & 0xFFFFFFFFFFFFFFFF, counter & 0xFFFFFFFFFFFFFFFF))


def rewire(idx, W, G, d, rho, init_random=False, seed=0, resort=True, momentum=None):
    """Algorithm 3, group-shared rewiring (readings in oracle/haste_oracle.cpp).  Returns a dict with
    the new idx [NG,K] int32, W [L,K] float32 (random weights NOT yet rounded to a storage type), momentum (or None),
    the fp32 scores [NG,K], the mask [NG,K] (uint8) and m."""
    idx = np.array(idx, dtype=np.int32, order="C", copy=True)
    W = np.array(W, dtype=np.float32, order="C", copy=True)
    L, K = W.shape
    NG = idx.shape[0]
    assert NG == -(-L // G) and idx.shape[1] == K
    mom = None if momentum is None else np.array(momentum, dtype=np.float32, order="C", copy=True)
    scores = np.empty((NG, K), dtype=np.float32)
    mask = np.empty((NG, K), dtype=np.uint8)
    f = _L().haste_oracle_rewire
    f.restype = ctypes.c_int64
    m = f(ctypes.c_int64(L), ctypes.c_int(G), ctypes.c_int(K), ctypes.c_int(d), _p(idx), _p(W), _p(mom), ctypes.c_double(rho),
          ctypes.c_int(1 if init_random else 0), ctypes.c_uint64(seed), ctypes.c_int(1 if resort else 0), _p(scores), _p(mask))
    if m < 0:
        raise ValueError("oracle.rewire failed")
    return dict(idx=idx, W=W, momentum=mom, scores=scores, mask=mask, m=int(m))
