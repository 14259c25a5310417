"""Host-side checks of the C-ABI boundary that need no GPU: the library builds, loads,
exports every function include/haste.h declares, and fails loudly (no CPU fallback)."""
import ctypes
import os
import re

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    from paper_2606_01117_b200 import build
    return build.build()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "haste.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b(haste_[a-z_0-9]+)\s*\(", src)
    return sorted(set(names))


def test_header_declares_the_north_star_calls():
    names = _declared_functions()
    for n in ("haste_create", "haste_forward_loss", "haste_backward", "haste_head_create", "haste_head_forward_loss",
              "haste_head_backward", "haste_destroy", "haste_head_destroy"):
        assert n in names


def test_library_exports_every_declared_symbol(built):
    L = ctypes.CDLL(built)
    for n in _declared_functions():
        assert hasattr(L, n), "libhaste.so does not export %s" % n


def test_binding_lists_the_same_symbols(built):
    from paper_2606_01117_b200 import haste
    assert sorted(haste.SYMBOLS) == _declared_functions()
    L = haste.lib()
    assert L.haste_status_string(0) == b"HASTE_OK"
    assert L.haste_status_string(-2) == b"HASTE_ERR_BAD_INDEX"


def test_config_struct_matches_header_layout():
    from paper_2606_01117_b200 import haste
    # int32 d; int64 L; int32 G,K; int32 B_max; enum dtype; enum dw_dtype; int64 label_offset; float; uint32
    assert haste.haste_config_t.d.offset == 0
    assert haste.haste_config_t.L.offset == 8
    assert haste.haste_config_t.G.offset == 16
    assert haste.haste_config_t.K.offset == 20
    assert haste.haste_config_t.B_max.offset == 24
    assert haste.haste_config_t.dtype.offset == 28
    assert haste.haste_config_t.dw_dtype.offset == 32
    assert haste.haste_config_t.label_offset.offset == 40
    assert haste.haste_config_t.loss_scale.offset == 48
    assert haste.haste_config_t.flags.offset == 52
    assert ctypes.sizeof(haste.haste_config_t) == 56


def test_argument_errors_are_reported_before_any_launch(built):
    from paper_2606_01117_b200 import haste
    L = haste.lib()
    h = ctypes.c_void_p()
    assert L.haste_create(ctypes.byref(h), None, 0) == haste.HASTE_ERR_INVALID_ARG
    cfg = haste.haste_config_t(d=0, L=10, G=2, K=2, B_max=4, dtype=0, dw_dtype=0)
    assert L.haste_create(ctypes.byref(h), ctypes.byref(cfg), 0) == haste.HASTE_ERR_INVALID_ARG
    assert b"positive" in L.haste_last_error()
    assert L.haste_forward_loss(None, 1, None, None, None, None, None, None, None, None, None, None) == haste.HASTE_ERR_INVALID_ARG
    assert L.haste_dy_bytes(None, 4) == 0


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback(built):
    """Without a CUDA device the product path must fail loudly, never compute on the CPU."""
    from paper_2606_01117_b200 import haste
    with pytest.raises(haste.HasteError) as ei:
        haste.HasteLayer(d=16, L=8, G=2, K=4, B_max=4, dtype="f32")
    assert ei.value.status == haste.HASTE_ERR_CUDA
    with pytest.raises(haste.HasteError):
        haste.HasteHead(d=16, L_h=8, B_max=4, dtype="f32")


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_01117_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "haste_oracle" not in txt, f
