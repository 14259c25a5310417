"""Seeded synthetic inputs with the shapes and statistics of the paper's workloads.

This module holds NONE of the method's arithmetic (no logits, no loss, no
gradients): it only draws X, W, idx, bias and CSR targets.  It is the one piece
the tests hand to both sides (the fp64 oracle and the CUDA path).  Host-side
numpy only.

Recipe (DESIGN.md "Input recipe"; shapes from PAPER.md:341-348 Table 7, :151
Fig. 4 caption, :145, :405; BASELINE.json configs):
  * PRNG: counter-based SplitMix64 hash of (seed, stream, element index) -- values do
    not depend on generation order.  seed = 1000 + config number; streams below.
  * normals by Box-Muller in fp64, one round-to-nearest-even to fp32 / bf16.
  * idx: each group draws K distinct features (Gumbel top-K on weights rank^-skew
    through a seeded rank->feature permutation; skew = 0 is uniform), sorted ascending.
  * targets: row i gets n_i = max(1, Poisson(avg)) distinct labels (or exactly n_fixed,
    uniform), drawn by popularity rank from Zipf(s) over 1..L by inverse CDF; rank r <= L_h
    maps to head id r-1, rank r > L_h to L_h + pi(r - L_h - 1) with pi a seeded
    permutation of the tail; columns sorted within each row.
No dataset item is reproduced; these stand in for Amazon-670K / Amazon-3M shaped data.
"""
from dataclasses import dataclass, field
import numpy as np

STREAM_X, STREAM_W, STREAM_IDX, STREAM_TGT, STREAM_WHEAD, STREAM_XHEAD, STREAM_BIAS, STREAM_PERM = 1, 2, 3, 4, 5, 6, 7, 8
STREAM_FPERM, STREAM_NPOS, STREAM_BIAS_HEAD = 9, 10, 11

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x):
    """SplitMix64 finaliser on a uint64 array (wrapping arithmetic)."""
    with np.errstate(over="ignore"):
        x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        x = ((x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        x = ((x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        return x ^ (x >> np.uint64(31))


def hash_u64(seed, stream, index):
    """Counter-based 64-bit hash of (seed, stream, index); index is an int array."""
    idx = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        key = _splitmix64(np.uint64(seed) * np.uint64(0x100000001B3) + np.uint64(stream))
        return _splitmix64(idx ^ key)


def uniform01(seed, stream, index):
    """Uniform in (0,1): 53 random bits, never exactly 0."""
    h = hash_u64(seed, stream, index)
    return ((h >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed, stream, n, start=0, chunk=1 << 24):
    """n standard normals (fp64) for element indices start..start+n-1 (Box-Muller on a pair of uniforms)."""
    out = np.empty(n, dtype=np.float64)
    for a in range(0, n, chunk):
        b = min(n, a + chunk)
        e = np.arange(start + a, start + b, dtype=np.uint64)
        u1 = uniform01(seed, stream, e * np.uint64(2))
        u2 = uniform01(seed, stream, e * np.uint64(2) + np.uint64(1))
        out[a:b] = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    return out


def round_bf16(a32):
    """Round-to-nearest-even fp32 -> bf16; returns (uint16 bit patterns, the rounded values as fp32)."""
    a32 = np.ascontiguousarray(a32, dtype=np.float32)
    u = a32.view(np.uint32)
    r = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    bits = ((u + r) >> np.uint32(16)).astype(np.uint16)
    vals = (bits.astype(np.uint32) << np.uint32(16)).view(np.float32)
    return bits, vals


def bf16_bits_to_f32(bits):
    return (np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def seeded_permutation(seed, stream, n):
    return np.argsort(hash_u64(seed, stream, np.arange(n, dtype=np.uint64)), kind="stable").astype(np.int64)


def draw_idx(seed, NG, d, K, skew=0.0, chunk_groups=4096):
    """idx [NG,K] int32: K distinct features per group, sorted; weights rank^-skew (skew=0: uniform)."""
    assert K <= d
    perm = seeded_permutation(seed, STREAM_FPERM, d)           # popularity rank -> feature id
    logw = np.empty(d, dtype=np.float64)
    logw[perm] = -skew * np.log(np.arange(1, d + 1, dtype=np.float64))
    out = np.empty((NG, K), dtype=np.int32)
    for g0 in range(0, NG, chunk_groups):
        g1 = min(NG, g0 + chunk_groups)
        e = (np.arange(g0, g1, dtype=np.uint64)[:, None] * np.uint64(d) + np.arange(d, dtype=np.uint64)[None, :])
        gumbel = -np.log(-np.log(uniform01(seed, STREAM_IDX, e)))
        keys = logw[None, :] + gumbel
        if K == d:
            top = np.tile(np.arange(d), (g1 - g0, 1))
        else:
            top = np.argpartition(-keys, K - 1, axis=1)[:, :K]
        out[g0:g1] = np.sort(top, axis=1).astype(np.int32)
    return out


def _poisson_from_uniform(u, lam):
    """Inverse-CDF Poisson(lam) from uniforms u."""
    kmax = int(lam + 12.0 * np.sqrt(lam) + 30)
    k = np.arange(kmax + 1, dtype=np.float64)
    from math import lgamma
    logp = -lam + k * np.log(lam) - np.array([lgamma(v + 1.0) for v in k])
    cdf = np.cumsum(np.exp(logp))
    return np.searchsorted(cdf, u, side="left").astype(np.int64)


def draw_targets(seed, B, L, L_h, avg_pos, zipf_s, n_fixed=None):
    """CSR multi-hot targets over global label ids [0,L).  Returns rowptr [B+1] int32, col [nnz] int32."""
    if n_fixed is not None:
        npos = np.full(B, int(n_fixed), dtype=np.int64)
    else:
        npos = np.maximum(1, _poisson_from_uniform(uniform01(seed, STREAM_NPOS, np.arange(B, dtype=np.uint64)), avg_pos))
    npos = np.minimum(npos, L)
    if zipf_s is None:
        cdf = None
    else:
        w = np.arange(1, L + 1, dtype=np.float64) ** (-float(zipf_s))
        cdf = np.cumsum(w)
        cdf /= cdf[-1]
    Lt = L - L_h
    pi = seeded_permutation(seed, STREAM_PERM, Lt) if Lt > 0 else None
    rowptr = np.zeros(B + 1, dtype=np.int32)
    cols = []
    MAX_TRY = 1 << 16
    for i in range(B):
        need = int(npos[i])
        got = []
        seen = set()
        t = 0
        while len(got) < need:
            m = max(16, 2 * (need - len(got)))
            e = np.uint64(i) * np.uint64(MAX_TRY) + np.arange(t, t + m, dtype=np.uint64)
            u = uniform01(seed, STREAM_TGT, e)
            if cdf is None:
                ranks = np.minimum((u * L).astype(np.int64), L - 1)          # 0-based, uniform
            else:
                ranks = np.minimum(np.searchsorted(cdf, u, side="left"), L - 1)   # 0-based popularity rank
            for r in ranks.tolist():
                lab = r if r < L_h else L_h + int(pi[r - L_h])
                if lab not in seen:
                    seen.add(lab)
                    got.append(lab)
                    if len(got) == need:
                        break
            t += m
            assert t < MAX_TRY
        got.sort()
        cols.extend(got)
        rowptr[i + 1] = len(cols)
    return rowptr, np.asarray(cols, dtype=np.int32)


@dataclass
class Config:
    name: str
    number: int
    B: int
    d: int
    L: int              # all labels (head + tail)
    L_h: int            # dense-head labels (the L_h most frequent); tail = L - L_h (reading R10)
    G: int
    K: int
    dtype: str          # "f32" | "bf16"
    idx_skew: float = 0.0
    zipf_s: float = None
    avg_pos: float = 5.0
    n_fixed: int = None
    w_std: float = 0.02

    @property
    def L_t(self):
        return self.L - self.L_h

    @property
    def NG(self):
        return -(-self.L_t // self.G)

    @property
    def seed(self):
        return 1000 + self.number


# BASELINE.json configs 1-4 (config 5 is a sweep: see sweep_config()).
CONFIGS = {
    "tiny_f32": Config("tiny_f32", 1, B=32, d=128, L=4096, L_h=0, G=16, K=32, dtype="f32", n_fixed=3),
    "mid_bf16": Config("mid_bf16", 2, B=256, d=768, L=131072, L_h=4096, G=32, K=64, dtype="bf16", zipf_s=1.1, avg_pos=5.0),
    "670k": Config("670k", 3, B=512, d=768, L=670091, L_h=16384, G=64, K=128, dtype="bf16", idx_skew=0.8, zipf_s=1.1, avg_pos=5.4),
    "3m": Config("3m", 4, B=256, d=1024, L=3000000, L_h=32768, G=64, K=64, dtype="bf16", zipf_s=1.0, avg_pos=36.0),
}


def sweep_config(B, G, L=670091, K=64, d=768):
    return Config("sweep_B%d_G%d" % (B, G), 5, B=B, d=d, L=L, L_h=0, G=G, K=K, dtype="bf16", zipf_s=1.1, avg_pos=5.4)


@dataclass
class Inputs:
    cfg: Config
    X: np.ndarray            # [B,d] fp32 values (bf16-rounded when dtype == bf16)
    W: np.ndarray            # [L_t,K] fp32 values
    idx: np.ndarray          # [NG,K] int32
    bias: np.ndarray         # [L_t] fp32 or None
    rowptr: np.ndarray       # [B+1] int32
    col: np.ndarray          # [nnz] int32 global ids
    X_head: np.ndarray = None   # [B,d]
    W_head: np.ndarray = None   # [L_h,d]
    bias_head: np.ndarray = None
    bits: dict = field(default_factory=dict)   # bf16 bit patterns (uint16) of X, W, X_head, W_head when dtype == bf16


def _draw_matrix(cfg, stream, shape, std, bits, key):
    n = int(np.prod(shape))
    a = (normal(cfg.seed, stream, n) * std).astype(np.float32)
    if cfg.dtype == "bf16":
        b, a = round_bf16(a)
        bits[key] = b.reshape(shape)
    return a.reshape(shape)


def make_inputs(cfg: Config, with_bias=False, with_head=True) -> Inputs:
    bits = {}
    X = _draw_matrix(cfg, STREAM_X, (cfg.B, cfg.d), 1.0, bits, "X")
    W = _draw_matrix(cfg, STREAM_W, (cfg.L_t, cfg.K), cfg.w_std, bits, "W")
    idx = draw_idx(cfg.seed, cfg.NG, cfg.d, cfg.K, cfg.idx_skew)
    rowptr, col = draw_targets(cfg.seed, cfg.B, cfg.L, cfg.L_h, cfg.avg_pos, cfg.zipf_s, cfg.n_fixed)
    bias = (normal(cfg.seed, STREAM_BIAS, cfg.L_t) * 0.1).astype(np.float32) if with_bias else None
    inp = Inputs(cfg, X, W, idx, bias, rowptr, col, bits=bits)
    if with_head and cfg.L_h > 0:
        inp.X_head = _draw_matrix(cfg, STREAM_XHEAD, (cfg.B, cfg.d), 1.0, bits, "X_head")
        inp.W_head = _draw_matrix(cfg, STREAM_WHEAD, (cfg.L_h, cfg.d), cfg.w_std, bits, "W_head")
        inp.bias_head = (normal(cfg.seed, STREAM_BIAS_HEAD, cfg.L_h) * 0.1).astype(np.float32) if with_bias else None
    return inp


def small_case(seed, B, d, L, G, K, dtype="f32", n_pos=3, sorted_distinct=True, with_bias=True, w_std=0.5,
               label_offset=0, L_total=None):
    """Free-form small case for parity/pin tests (any G, K, d; partial last group; optional duplicates)."""
    cfg = Config("small", 0, B=B, d=d, L=L, L_h=0, G=G, K=K, dtype=dtype, n_fixed=n_pos, w_std=w_std)
    bits = {}
    n = B * d
    X = normal(seed, STREAM_X, n).astype(np.float32).reshape(B, d)
    W = (normal(seed, STREAM_W, L * K) * w_std).astype(np.float32).reshape(L, K)
    if dtype == "bf16":
        bits["X"], X = round_bf16(X)
        bits["W"], W = round_bf16(W)
        bits["X"] = bits["X"].reshape(B, d)
        bits["W"] = bits["W"].reshape(L, K)
        X = X.reshape(B, d)
        W = W.reshape(L, K)
    NG = -(-L // G)
    if sorted_distinct:
        idx = draw_idx(seed, NG, d, K, 0.0)
    else:   # any values in [0,d): duplicates and arbitrary order allowed (reading R4)
        e = np.arange(NG * K, dtype=np.uint64)
        idx = np.minimum((uniform01(seed, STREAM_IDX, e) * d).astype(np.int32), d - 1).reshape(NG, K)
    Ltot = L_total if L_total is not None else label_offset + L
    rowptr, col = draw_targets(seed, B, Ltot, 0, n_pos, None, n_fixed=min(n_pos, Ltot))
    bias = (normal(seed, STREAM_BIAS, L) * 0.1).astype(np.float32) if with_bias else None
    return Inputs(cfg, X, W, idx, bias, rowptr, col, bits=bits)
