"""The C-ABI boundary (include/tabattn.h): the library loads, exports every declared symbol and
rejects bad arguments before touching the device.  No compute calls -- runs without a GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tab():
    from paper_2606_03681_b200 import build as _build
    _build.build()
    import paper_2606_03681_b200 as t
    return t


def _declared_symbols():
    names = []
    for fn in sorted(os.listdir(os.path.join(ROOT, "include"))):
        if fn.endswith(".h"):
            src = open(os.path.join(ROOT, "include", fn)).read()
            names += re.findall(r"TABATTN_API\s+[\w\s\*]+?\b(tabattn_\w+)\s*\(", src)
    return names


def test_every_declared_symbol_is_exported(tab):
    names = _declared_symbols()
    assert set(names) == set(tab.EXPORTS) and len(names) == 8
    L = ctypes.CDLL(tab.LIB_PATH)
    for n in names:
        assert getattr(L, n) is not None


def test_version_and_status_strings(tab):
    assert tab.version() == 100
    seen = {tab.status_string(i) for i in range(5)}
    assert len(seen) == 5 and all(seen)
    assert tab.status_string(99)


def test_shape_struct_matches_header(tab):
    # 5 x int32, 3 pointers (8-byte aligned after 20 bytes -> 24), float, padded to 8
    assert ctypes.sizeof(tab.TabattnShape) == 56
    assert tab.TabattnShape.n_train.offset == 24 and tab.TabattnShape.softmax_scale.offset == 48


def test_workspace_bytes(tab):
    s = tab.TabattnShape(32, 1024, 11, 6, 32, None, None, None, 0.0)
    assert tab.workspace_bytes(s, tab.OP_FEATURE_FWD) == 0
    assert tab.workspace_bytes(s, tab.OP_ITEM_FWD) % 16 == 0
    # D = rowsum(dO o O) as f32 [B,C,H,R] must fit
    assert tab.workspace_bytes(s, tab.OP_ITEM_BWD) >= 32 * 11 * 6 * 1024 * 4
    bad = tab.TabattnShape(32, 1024, 11, 6, 48, None, None, None, 0.0)
    assert tab.workspace_bytes(bad, tab.OP_ITEM_BWD) == 0
    assert tab.workspace_bytes(s, 7) == 0


def _call_fwd(tab, fn, shape, ptrs=(16, 16, 16, 16, 16), ws=None, nws=0):
    f = getattr(tab.lib(), fn)
    args = [ctypes.c_void_p(p) if p else None for p in ptrs]
    return f(ctypes.byref(shape) if shape is not None else None, *args, ws, nws, None)


@pytest.mark.parametrize("fn", ["tabattn_feature_fwd", "tabattn_item_fwd"])
def test_argument_errors_need_no_device(tab, fn):
    nt = (ctypes.c_int32 * 2)(3, 4)
    ntp = ctypes.cast(nt, ctypes.c_void_p).value
    ok = tab.TabattnShape(2, 8, 4, 2, 16, 4096, None, None, 0.0)
    assert _call_fwd(tab, fn, None) == tab.ERR_INVALID_ARG
    for field in ("B", "R", "C", "H", "dh"):
        s = tab.TabattnShape(2, 8, 4, 2, 16, 4096, None, None, 0.0)
        setattr(s, field, 0)
        assert _call_fwd(tab, fn, s) == tab.ERR_INVALID_ARG
    s = tab.TabattnShape(2, 8, 4, 2, 24, 4096, None, None, 0.0)
    assert _call_fwd(tab, fn, s) == tab.ERR_UNSUPPORTED
    assert _call_fwd(tab, fn, ok, ptrs=(0, 16, 16, 16, 16)) == tab.ERR_INVALID_ARG      # NULL Q
    assert _call_fwd(tab, fn, ok, ptrs=(16, 16, 24, 16, 16)) == tab.ERR_INVALID_ARG     # misaligned V
    if fn == "tabattn_item_fwd":
        s = tab.TabattnShape(2, 8, 4, 2, 16, None, None, None, 0.0)                     # NULL n_train
        assert _call_fwd(tab, fn, s) == tab.ERR_INVALID_ARG
        bad = (ctypes.c_int32 * 2)(3, 9)                                                # n_train > R
        s = tab.TabattnShape(2, 8, 4, 2, 16, 4096, ctypes.cast(bad, ctypes.c_void_p).value, None, 0.0)
        assert _call_fwd(tab, fn, s) == tab.ERR_INVALID_ARG
        zero = (ctypes.c_int32 * 2)(0, 4)                                               # n_train = 0
        s = tab.TabattnShape(2, 8, 4, 2, 16, 4096, ctypes.cast(zero, ctypes.c_void_p).value, None, 0.0)
        assert _call_fwd(tab, fn, s) == tab.ERR_INVALID_ARG
        # a good host copy passes validation (NULL Q is then the first error, still before any launch)
        s = tab.TabattnShape(2, 8, 4, 2, 16, 4096, ntp, None, 0.0)
        assert _call_fwd(tab, fn, s, ptrs=(0, 16, 16, 16, 16)) == tab.ERR_INVALID_ARG
    else:
        s = tab.TabattnShape(2, 8, 129, 2, 16, None, None, None, 0.0)                   # C too large
        assert _call_fwd(tab, fn, s) == tab.ERR_UNSUPPORTED


def test_item_bwd_workspace_is_checked(tab):
    s = tab.TabattnShape(2, 8, 4, 2, 16, 4096, None, None, 0.0)
    f = tab.lib().tabattn_item_bwd
    p = ctypes.c_void_p(16)
    assert f(ctypes.byref(s), p, p, p, p, p, p, p, p, p, None, 0, None) == tab.ERR_WORKSPACE
    assert f(ctypes.byref(s), p, p, p, p, p, p, p, p, p, p, 8, None) == tab.ERR_WORKSPACE


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_03681_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in src.replace("no CPU or PyTorch fallback", ""), fn
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".c")):
            assert "paper_2606_03681_b200/csrc" in open(os.path.join(ROOT, "oracle", fn)).read() or \
                "import paper_2606_03681_b200" not in open(os.path.join(ROOT, "oracle", fn)).read()
