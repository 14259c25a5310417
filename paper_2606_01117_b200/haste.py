"""ctypes binding of the C-ABI library (include/haste.h): argument marshalling only.

Same names as the C entry points (haste_create / haste_forward_loss / haste_backward /
haste_head_*), wrapped in two small classes.  torch is used for device memory and
streams; every step of the path runs in the library's CUDA kernels.  There is no CPU
fallback: loading fails loudly when libhaste.so is missing, and every call raises
HasteError on a non-zero status.
"""
import ctypes
import os

import torch

_DIR = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_DIR, "libhaste.so")

HASTE_F32, HASTE_BF16 = 0, 1
HASTE_IDX_SORTED_DISTINCT, HASTE_DETERMINISTIC, HASTE_FORCE_SIMT, HASTE_XT_FROM_FORWARD = 1, 2, 4, 8
HASTE_OK, HASTE_ERR_INVALID_ARG, HASTE_ERR_BAD_INDEX, HASTE_ERR_UNSUPPORTED, HASTE_ERR_CUDA, HASTE_ERR_NOMEM = 0, -1, -2, -3, -4, -5

# Every symbol include/haste.h declares (tests check the library exports all of them).
SYMBOLS = [
    "haste_create", "haste_destroy", "haste_dy_bytes", "haste_validate_index", "haste_forward_loss", "haste_forward_loss_dw", "haste_forward_logits", "haste_forward_topk", "haste_forward_topk_static",
    "haste_backward", "haste_backward_sgd", "haste_rewire", "haste_dy_unpack", "haste_dy_pack", "haste_head_create", "haste_head_destroy",
    "haste_head_forward_loss", "haste_head_backward", "haste_status_string", "haste_last_error",
    "haste_kernel_family", "haste_head_kernel_family", "haste_last_launch_count", "haste_head_last_launch_count",
    "haste_set_profiling", "haste_kernel_ms", "haste_head_set_profiling", "haste_head_kernel_ms",
]
KERNEL_FORWARD, KERNEL_DW, KERNEL_DX, KERNEL_PREP_FWD, KERNEL_PREP_BWD, KERNEL_POST_BWD = range(6)


class haste_config_t(ctypes.Structure):
    _fields_ = [
        ("d", ctypes.c_int32), ("L", ctypes.c_int64), ("G", ctypes.c_int32), ("K", ctypes.c_int32),
        ("B_max", ctypes.c_int32), ("dtype", ctypes.c_int), ("dw_dtype", ctypes.c_int),
        ("label_offset", ctypes.c_int64), ("loss_scale", ctypes.c_float), ("flags", ctypes.c_uint32),
    ]


class HasteError(RuntimeError):
    def __init__(self, status, detail):
        self.status = status
        super().__init__("haste status %d: %s" % (status, detail))


_lib = None


def lib():
    """Load libhaste.so (built in-tree by paper_2606_01117_b200.build).  No fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libhaste.so is missing at %s: run `python -m paper_2606_01117_b200.build` "
                          "(there is no CPU fallback)" % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, f32, u32 = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_float, ctypes.c_uint32
    L.haste_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(haste_config_t), i32]
    L.haste_destroy.argtypes = [vp]
    L.haste_dy_bytes.argtypes = [vp, i32]
    L.haste_dy_bytes.restype = ctypes.c_size_t
    L.haste_validate_index.argtypes = [vp, vp, vp]
    L.haste_forward_loss.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.haste_forward_loss_dw.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.haste_forward_logits.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp]
    L.haste_forward_topk.argtypes = [vp, i32, vp, vp, vp, vp, i32, vp, vp, vp]
    L.haste_forward_topk_static.argtypes = [vp, i32, vp, vp, vp, vp, i32, vp, vp, vp]
    L.haste_backward.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, i32, vp]
    L.haste_backward_sgd.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, f32, f32, f32, vp, i32, vp]
    L.haste_rewire.argtypes = [vp, vp, vp, vp, f32, i32, ctypes.c_uint64, i32, ctypes.POINTER(ctypes.c_int64), vp]
    L.haste_dy_unpack.argtypes = [vp, i32, vp, vp, vp]
    L.haste_dy_pack.argtypes = [vp, i32, vp, vp, vp]
    L.haste_head_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int32, i64, ctypes.c_int32, i32, i64, f32, u32, i32]
    L.haste_head_destroy.argtypes = [vp]
    L.haste_head_forward_loss.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    L.haste_head_backward.argtypes = [vp, i32, vp, vp, vp, vp, vp, vp, i32, vp]
    L.haste_status_string.argtypes = [i32]
    L.haste_status_string.restype = ctypes.c_char_p
    L.haste_last_error.restype = ctypes.c_char_p
    for n in ("haste_kernel_family", "haste_head_kernel_family", "haste_last_launch_count", "haste_head_last_launch_count"):
        getattr(L, n).argtypes = [vp]
    for n in ("haste_set_profiling", "haste_head_set_profiling"):
        getattr(L, n).argtypes = [vp, i32]
    for n in ("haste_kernel_ms", "haste_head_kernel_ms"):
        getattr(L, n).argtypes = [vp, i32, i32, ctypes.POINTER(f32)]
    _lib = L
    return L


def _check(rc):
    if rc != 0:
        L = lib()
        raise HasteError(rc, "%s: %s" % (L.haste_status_string(rc).decode(), L.haste_last_error().decode()))


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def _dt(dtype):
    if dtype in (torch.float32, "f32", HASTE_F32):
        return HASTE_F32
    if dtype in (torch.bfloat16, "bf16", HASTE_BF16):
        return HASTE_BF16
    raise ValueError("dtype must be float32 or bfloat16")


_TORCH = {HASTE_F32: torch.float32, HASTE_BF16: torch.bfloat16}


class HasteLayer:
    """Sparse tail handle (haste_create ... haste_destroy)."""

    def __init__(self, d, L, G, K, B_max, dtype, dw_dtype=None, label_offset=0, loss_scale=0.0, flags=0, device=0):
        self.cfg = haste_config_t(d=d, L=L, G=G, K=K, B_max=B_max, dtype=_dt(dtype),
                                  dw_dtype=_dt(dw_dtype if dw_dtype is not None else dtype),
                                  label_offset=label_offset, loss_scale=loss_scale, flags=flags)
        self.device = device
        self.h = ctypes.c_void_p()
        self._destroy = lib().haste_destroy      # bound here: module globals may be gone when __del__ runs at interpreter exit
        _check(lib().haste_create(ctypes.byref(self.h), ctypes.byref(self.cfg), device))
        self.NG = -(-L // G)
        self.tdtype = _TORCH[self.cfg.dtype]
        self.dw_tdtype = _TORCH[self.cfg.dw_dtype]

    def close(self):
        if getattr(self, "h", None) is not None and self.h.value:
            self._destroy(self.h)
            self.h = None

    __del__ = close

    @property
    def kernel_family(self):
        return lib().haste_kernel_family(self.h)

    @property
    def last_launch_count(self):
        return lib().haste_last_launch_count(self.h)

    def set_profiling(self, depth=1):
        _check(lib().haste_set_profiling(self.h, int(depth)))

    def kernel_ms(self, kernel, age=0):
        ms = ctypes.c_float()
        _check(lib().haste_kernel_ms(self.h, kernel, age, ctypes.byref(ms)))
        return ms.value

    def dy_bytes(self, B):
        return lib().haste_dy_bytes(self.h, B)

    def alloc_dy(self, B):
        n = self.dy_bytes(B) // (4 if self.cfg.dtype == HASTE_F32 else 2)
        return torch.empty(max(n, 1), dtype=self.tdtype, device="cuda:%d" % self.device)

    def validate_index(self, idx, stream=None):
        _check(lib().haste_validate_index(self.h, _ptr(idx), _stream(stream)))

    def forward_loss(self, B, X, idx, W, bias, rowptr, col, loss=None, dY=None, logits_out=None, stream=None):
        _check(lib().haste_forward_loss(self.h, B, _ptr(X), _ptr(idx), _ptr(W), _ptr(bias), _ptr(rowptr), _ptr(col),
                                        _ptr(loss), _ptr(dY), _ptr(logits_out), _stream(stream)))

    def forward_topk(self, B, X, idx, W, bias, k, out_val, out_idx, stream=None):
        _check(lib().haste_forward_topk(self.h, B, _ptr(X), _ptr(idx), _ptr(W), _ptr(bias), k, _ptr(out_val), _ptr(out_idx),
                                        _stream(stream)))

    def forward_topk_static(self, B, X, idx, W, bias, k, out_val, out_idx, stream=None):
        """haste_forward_topk_static: the same results with the candidate lists in the library's static device array; the
        call allocates nothing (include/haste.h)."""
        _check(lib().haste_forward_topk_static(self.h, B, _ptr(X), _ptr(idx), _ptr(W), _ptr(bias), k, _ptr(out_val),
                                               _ptr(out_idx), _stream(stream)))

    def forward_loss_dw(self, B, X, idx, W, bias, rowptr, col, loss=None, dY=None, dW=None, dbias=None, stream=None):
        _check(lib().haste_forward_loss_dw(self.h, B, _ptr(X), _ptr(idx), _ptr(W), _ptr(bias), _ptr(rowptr), _ptr(col), _ptr(loss),
                                           _ptr(dY), _ptr(dW), _ptr(dbias), _stream(stream)))

    def forward_logits(self, B, X, idx, W, bias, Z, stream=None):
        _check(lib().haste_forward_logits(self.h, B, _ptr(X), _ptr(idx), _ptr(W), _ptr(bias), _ptr(Z), _stream(stream)))

    def backward(self, B, X, idx, W, dY, dW=None, dbias=None, dX=None, accumulate_dX=False, stream=None):
        _check(lib().haste_backward(self.h, B, _ptr(X), _ptr(idx), _ptr(W), _ptr(dY), _ptr(dW), _ptr(dbias), _ptr(dX),
                                    1 if accumulate_dX else 0, _stream(stream)))

    def backward_sgd(self, B, X, idx, W, dY, momentum, lr, mu, weight_decay=0.0, bias=None, bias_momentum=None, dX=None,
                     accumulate_dX=False, stream=None):
        _check(lib().haste_backward_sgd(self.h, B, _ptr(X), _ptr(idx), _ptr(W), _ptr(dY), _ptr(momentum), _ptr(bias),
                                        _ptr(bias_momentum), lr, mu, weight_decay, _ptr(dX), 1 if accumulate_dX else 0,
                                        _stream(stream)))

    def rewire(self, idx, W, rho, momentum=None, init_random=False, seed=0, resort=True, stream=None):
        """Algorithm 3 in place on idx / W / momentum; returns the number of pruned slots."""
        m = ctypes.c_int64(0)
        _check(lib().haste_rewire(self.h, _ptr(idx), _ptr(W), _ptr(momentum), rho, 1 if init_random else 0, seed,
                                  1 if resort else 0, ctypes.byref(m), _stream(stream)))
        return m.value

    def dy_unpack(self, B, dY, out_BL, stream=None):
        _check(lib().haste_dy_unpack(self.h, B, _ptr(dY), _ptr(out_BL), _stream(stream)))

    def dy_pack(self, B, in_BL, dY, stream=None):
        _check(lib().haste_dy_pack(self.h, B, _ptr(in_BL), _ptr(dY), _stream(stream)))


class HasteHead:
    """Dense head handle (haste_head_create ... haste_head_destroy)."""

    def __init__(self, d, L_h, B_max, dtype, label_offset=0, loss_scale=0.0, flags=0, device=0):
        self.d, self.L, self.device = d, L_h, device
        self.dtype = _dt(dtype)
        self.tdtype = _TORCH[self.dtype]
        self.h = ctypes.c_void_p()
        self._destroy = lib().haste_head_destroy
        _check(lib().haste_head_create(ctypes.byref(self.h), d, L_h, B_max, self.dtype, label_offset, loss_scale, flags,
                                       device))

    def close(self):
        if getattr(self, "h", None) is not None and self.h.value:
            self._destroy(self.h)
            self.h = None

    __del__ = close

    @property
    def kernel_family(self):
        return lib().haste_head_kernel_family(self.h)

    @property
    def last_launch_count(self):
        return lib().haste_head_last_launch_count(self.h)

    def set_profiling(self, depth=1):
        _check(lib().haste_head_set_profiling(self.h, int(depth)))

    def kernel_ms(self, kernel, age=0):
        ms = ctypes.c_float()
        _check(lib().haste_head_kernel_ms(self.h, kernel, age, ctypes.byref(ms)))
        return ms.value

    def forward_loss(self, B, X, Wh, bias, rowptr, col, loss=None, dY=None, logits_out=None, stream=None):
        _check(lib().haste_head_forward_loss(self.h, B, _ptr(X), _ptr(Wh), _ptr(bias), _ptr(rowptr), _ptr(col),
                                             _ptr(loss), _ptr(dY), _ptr(logits_out), _stream(stream)))

    def backward(self, B, X, Wh, dY, dWh=None, dbias=None, dX=None, accumulate_dX=False, stream=None):
        _check(lib().haste_head_backward(self.h, B, _ptr(X), _ptr(Wh), _ptr(dY), _ptr(dWh), _ptr(dbias), _ptr(dX),
                                         1 if accumulate_dX else 0, _stream(stream)))
