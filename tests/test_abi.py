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
    assert set(names) == set(tab.EXPORTS) and len(names) == len(set(names)) >= 10
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
    # feature calls: per-table geometry for masked tables (a0), a few KB
    assert 32 * (16 + 128) <= tab.workspace_bytes(s, tab.OP_FEATURE_FWD) <= 32 * 256
    assert tab.workspace_bytes(s, tab.OP_FEATURE_BWD) == tab.workspace_bytes(s, tab.OP_FEATURE_FWD)
    # item forward: the a0 column list of masked calls, 4 bytes per (b, c) pair
    assert 32 * 11 * 4 <= tab.workspace_bytes(s, tab.OP_ITEM_FWD) <= 32 * 11 * 4 + 64
    # D = rowsum(dO o O) as f32 [B,C,H,R] must fit
    assert tab.workspace_bytes(s, tab.OP_ITEM_BWD) >= 32 * 11 * 6 * 1024 * 4
    bad = tab.TabattnShape(32, 1024, 11, 6, 48, None, None, None, 0.0)
    assert tab.workspace_bytes(bad, tab.OP_ITEM_BWD) == 0
    assert tab.workspace_bytes(s, 7) == 0


def _call_fwd(tab, fn, shape, ptrs=(16, 32, 48, 64, 80), ws=None, nws=0):
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
    assert _call_fwd(tab, fn, ok, ptrs=(0, 32, 48, 64, 80)) == tab.ERR_INVALID_ARG      # NULL Q
    assert _call_fwd(tab, fn, ok, ptrs=(16, 32, 56, 64, 80)) == tab.ERR_INVALID_ARG     # misaligned V
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
        assert _call_fwd(tab, fn, s, ptrs=(0, 32, 48, 64, 80)) == tab.ERR_INVALID_ARG
    else:
        s = tab.TabattnShape(2, 8, 129, 2, 16, None, None, None, 0.0)                   # C too large
        assert _call_fwd(tab, fn, s) == tab.ERR_UNSUPPORTED


def test_item_bwd_workspace_is_checked(tab):
    s = tab.TabattnShape(2, 8, 4, 2, 16, 4096, None, None, 0.0)
    f = tab.lib().tabattn_item_bwd
    p = [ctypes.c_void_p(16 * (i + 1)) for i in range(10)]
    assert f(ctypes.byref(s), *p[:9], None, 0, None) == tab.ERR_WORKSPACE
    assert f(ctypes.byref(s), *p[:9], p[9], 8, None) == tab.ERR_WORKSPACE


def test_output_aliasing_is_rejected(tab):
    """tabattn.h: no aliasing of an output with any other argument (equal pointers are detected)."""
    s = tab.TabattnShape(2, 8, 4, 2, 16, 4096, None, None, 0.0)
    for fn in ("tabattn_feature_fwd", "tabattn_item_fwd"):
        assert _call_fwd(tab, fn, s, ptrs=(16, 32, 48, 16, 80)) == tab.ERR_INVALID_ARG     # O over Q
    p = [ctypes.c_void_p(16 * (i + 1)) for i in range(10)]
    for fn in ("tabattn_feature_bwd", "tabattn_item_bwd"):
        f = getattr(tab.lib(), fn)
        a = list(p[:9])
        a[6] = a[0]                                                                         # dQ over Q
        assert f(ctypes.byref(s), *a, p[9], 1 << 20, None) == tab.ERR_INVALID_ARG
        a = list(p[:9])
        a[8] = a[7]                                                                         # dV over dK
        assert f(ctypes.byref(s), *a, p[9], 1 << 20, None) == tab.ERR_INVALID_ARG


def test_documented_limits_match_the_implementation(tab):
    """include/tabattn.h documents TABATTN_MAX_D and TABATTN_MAX_FEATURE_C; B*C has no limit of its own."""
    hdr = open(os.path.join(ROOT, "include", "tabattn.h")).read()
    max_d = int(re.search(r"#define TABATTN_MAX_D (\d+)", hdr).group(1))
    max_c = int(re.search(r"#define TABATTN_MAX_FEATURE_C (\d+)", hdr).group(1))
    ok = tab.TabattnShape(1, 8, 4, max_d // 16, 16, 4096, None, None, 0.0)
    assert tab.workspace_bytes(ok, tab.OP_ITEM_BWD) > 0
    bad = tab.TabattnShape(1, 8, 4, max_d // 16 + 1, 16, 4096, None, None, 0.0)
    assert tab.workspace_bytes(bad, tab.OP_ITEM_BWD) == 0
    wide = tab.TabattnShape(700, 8, 100, 2, 16, 4096, None, None, 0.0)     # B*C = 70000 > 65535
    assert tab.workspace_bytes(wide, tab.OP_ITEM_BWD) > 0
    assert _call_fwd(tab, "tabattn_feature_fwd", tab.TabattnShape(2, 8, max_c + 1, 2, 16, None, None, None, 0.0)) \
        == tab.ERR_UNSUPPORTED


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


def test_new_entry_points_reject_bad_arguments_without_a_device(tab):
    """The evaluation and sub-block calls validate before they touch the device."""
    L = tab.lib()
    P = lambda i: ctypes.c_void_p(16 * (i + 1))
    nt = (ctypes.c_int32 * 2)(3, 4)
    s = tab.TabattnShape(2, 8, 4, 2, 32, 4096, ctypes.cast(nt, ctypes.c_void_p).value, None, 0.0)
    # row range outside [0, R] or empty
    for r0, r1 in ((-1, 4), (4, 4), (6, 2), (0, 9)):
        assert L.tabattn_item_fwd_infer(ctypes.byref(s), P(0), P(1), P(2), P(3), r0, r1, None, 0, None) == tab.ERR_INVALID_ARG
        assert L.tabattn_feature_fwd_infer(ctypes.byref(s), P(0), P(1), P(2), P(3), r0, r1, None, 0, None) == tab.ERR_INVALID_ARG
    assert L.tabattn_item_fwd_infer(ctypes.byref(s), P(0), P(1), P(2), P(0), 0, 8, None, 0, None) == tab.ERR_INVALID_ARG  # O over Q
    # sub-blocks: e = H*dh must be a multiple of 64 (here 2 x 16 = 32), axis in {0, 1}, saved struct required
    s32 = tab.TabattnShape(2, 8, 4, 2, 16, 4096, None, None, 0.0)
    sv = tab.binding.TabattnAttnSaved(*[16 * (i + 20) for i in range(7)])
    assert L.tabattn_attn_block_fwd(ctypes.byref(s32), 0, 1.0, 0.0, P(0), P(1), P(2), P(3), P(4), ctypes.byref(sv), None, 0,
                                    None) == tab.ERR_UNSUPPORTED
    s64 = tab.TabattnShape(2, 8, 4, 2, 32, 4096, None, None, 0.0)
    assert L.tabattn_attn_block_fwd(ctypes.byref(s64), 2, 1.0, 0.0, P(0), P(1), P(2), P(3), P(4), ctypes.byref(sv), None, 0,
                                    None) == tab.ERR_INVALID_ARG
    assert L.tabattn_attn_block_fwd(ctypes.byref(s64), 0, 1.0, 0.0, P(0), P(1), P(2), P(3), P(4), None, None, 0,
                                    None) == tab.ERR_INVALID_ARG
    assert L.tabattn_attn_block_workspace_bytes(ctypes.byref(s64), 0, 1) > 2 * 8 * 4 * 64 * 2 * 5
    assert L.tabattn_attn_block_workspace_bytes(ctypes.byref(s64), 3, 1) == 0
    mv = tab.binding.TabattnMlpSaved(*[16 * (i + 30) for i in range(4)])
    assert L.tabattn_mlp_fwd(100, 96, 128, 1.0, 0.0, P(0), P(1), P(2), P(3), P(4), ctypes.byref(mv), None) == tab.ERR_UNSUPPORTED
    assert L.tabattn_mlp_fwd(0, 64, 128, 1.0, 0.0, P(0), P(1), P(2), P(3), P(4), ctypes.byref(mv), None) == tab.ERR_INVALID_ARG
    assert L.tabattn_mlp_fwd(100, 64, 128, 1.0, 0.0, P(0), P(1), P(2), P(3), P(0), ctypes.byref(mv), None) == tab.ERR_INVALID_ARG
    assert L.tabattn_mlp_workspace_bytes(100, 64, 128) > 100 * 128 * 4
    assert L.tabattn_mlp_workspace_bytes(100, 60, 128) == 0
    # Newton-Schulz: m <= n, multiples of 8, workspace checked
    assert L.tabattn_newton_schulz(2, 64, 32, P(0), P(1), 5, P(2), 1 << 20, None) == tab.ERR_UNSUPPORTED
    assert L.tabattn_newton_schulz(2, 60, 64, P(0), P(1), 5, P(2), 1 << 20, None) == tab.ERR_UNSUPPORTED
    assert L.tabattn_newton_schulz(2, 64, 64, P(0), P(0), 5, P(2), 1 << 20, None) == tab.ERR_INVALID_ARG
    assert L.tabattn_newton_schulz(2, 64, 64, P(0), P(1), 5, None, 0, None) == tab.ERR_WORKSPACE
    assert L.tabattn_newton_schulz_workspace_bytes(2, 64, 64) >= (2 * 64 * 64 * 3) * 2
