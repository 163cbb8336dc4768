"""ctypes front-end of the fp64 CPU oracle (oracle/tabattn_ref.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / ``--impl reference`` leg may import this module.  It
shares nothing with paper_2606_03681_b200/ and never imports it.

Inputs are ``[B,R,C,H,dh]`` numpy arrays, either ``uint16`` (bf16 bit
patterns, widened exactly) or ``float64``.  Outputs are ``float64``.
With ``rows=None`` / ``cols=None`` the full tensors come back in the library's
layouts (O/dQ/dK/dV ``[B,R,C,H,dh]``, feature LSE ``[B,R,H,C]``, item LSE
``[B,C,H,R]``); with a selection ``[[b, r], ...]`` / ``[[b, c], ...]`` only
those whole sequences are computed and returned compactly
(feature ``[n_sel,C,H,dh]`` + LSE ``[n_sel,H,C]``; item ``[n_sel,R,H,dh]`` + LSE
``[n_sel,H,R]``).  Definition followed: SURVEY.md §8(c) steps 1-7.
"""
import ctypes

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        _lib.ref_num_threads.restype = ctypes.c_int
    return _lib


def num_threads() -> int:
    return int(_load().ref_num_threads())


def _prep_in(*arrs):
    a0 = arrs[0]
    if a0.dtype == np.uint16:
        f64 = 0
    elif a0.dtype == np.float64:
        f64 = 1
    else:
        raise TypeError("oracle inputs must be uint16 (bf16 bits) or float64, got %s" % a0.dtype)
    out = []
    for a in arrs:
        if a.dtype != a0.dtype or a.shape != a0.shape or a.ndim != 5:
            raise ValueError("Q,K,V,dO must share dtype and the [B,R,C,H,dh] shape")
        out.append(np.ascontiguousarray(a))
    return f64, out


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p) if a is not None else None


def _mask(col_valid, B, C):
    if col_valid is None:
        return None
    m = np.ascontiguousarray(col_valid, dtype=np.uint8)
    if m.shape != (B, C):
        raise ValueError("col_valid must be [B,C]")
    return m


def _sel(sel, full_a, full_b):
    if sel is None:
        bb, xx = np.meshgrid(np.arange(full_a), np.arange(full_b), indexing="ij")
        sel = np.stack([bb.ravel(), xx.ravel()], axis=1)
    sel = np.asarray(sel, dtype=np.int32).reshape(-1, 2)
    return np.ascontiguousarray(sel[:, 0]), np.ascontiguousarray(sel[:, 1])


def feature_fwd(Q, K, V, col_valid=None, scale=0.0, rows=None, nthreads=0):
    f64, (Q, K, V) = _prep_in(Q, K, V)
    B, R, C, H, dh = Q.shape
    m = _mask(col_valid, B, C)
    sb, sr = _sel(rows, B, R)
    n = sb.size
    O = np.empty((n, C, H, dh), np.float64)
    LSE = np.empty((n, H, C), np.float64)
    rc = _load().ref_feature_fwd(_p(Q), _p(K), _p(V), f64, B, R, C, H, dh, _p(m), ctypes.c_double(scale),
                                 n, _p(sb), _p(sr), _p(O), _p(LSE), int(nthreads))
    if rc:
        raise ValueError("ref_feature_fwd rc=%d" % rc)
    if rows is None:
        return O.reshape(B, R, C, H, dh), LSE.reshape(B, R, H, C)
    return O, LSE


def feature_bwd(Q, K, V, dO, col_valid=None, scale=0.0, rows=None, nthreads=0):
    f64, (Q, K, V, dO) = _prep_in(Q, K, V, dO)
    B, R, C, H, dh = Q.shape
    m = _mask(col_valid, B, C)
    sb, sr = _sel(rows, B, R)
    n = sb.size
    dQ, dK, dV = (np.empty((n, C, H, dh), np.float64) for _ in range(3))
    rc = _load().ref_feature_bwd(_p(Q), _p(K), _p(V), _p(dO), f64, B, R, C, H, dh, _p(m),
                                 ctypes.c_double(scale), n, _p(sb), _p(sr), _p(dQ), _p(dK), _p(dV),
                                 int(nthreads))
    if rc:
        raise ValueError("ref_feature_bwd rc=%d" % rc)
    if rows is None:
        return tuple(x.reshape(B, R, C, H, dh) for x in (dQ, dK, dV))
    return dQ, dK, dV


def _ntrain(n_train, B):
    nt = np.ascontiguousarray(n_train, dtype=np.int32)
    if nt.shape != (B,):
        raise ValueError("n_train must be [B]")
    return nt


def item_fwd(Q, K, V, n_train, col_valid=None, scale=0.0, cols=None, nthreads=0):
    f64, (Q, K, V) = _prep_in(Q, K, V)
    B, R, C, H, dh = Q.shape
    m = _mask(col_valid, B, C)
    nt = _ntrain(n_train, B)
    sb, sc = _sel(cols, B, C)
    n = sb.size
    O = np.empty((n, R, H, dh), np.float64)
    LSE = np.empty((n, H, R), np.float64)
    rc = _load().ref_item_fwd(_p(Q), _p(K), _p(V), f64, B, R, C, H, dh, _p(nt), _p(m), ctypes.c_double(scale),
                              n, _p(sb), _p(sc), _p(O), _p(LSE), int(nthreads))
    if rc:
        raise ValueError("ref_item_fwd rc=%d" % rc)
    if cols is None:
        O = np.ascontiguousarray(O.reshape(B, C, R, H, dh).transpose(0, 2, 1, 3, 4))
        return O, LSE.reshape(B, C, H, R)
    return O, LSE


def item_bwd(Q, K, V, dO, n_train, col_valid=None, scale=0.0, cols=None, nthreads=0):
    f64, (Q, K, V, dO) = _prep_in(Q, K, V, dO)
    B, R, C, H, dh = Q.shape
    m = _mask(col_valid, B, C)
    nt = _ntrain(n_train, B)
    sb, sc = _sel(cols, B, C)
    n = sb.size
    dQ, dK, dV = (np.empty((n, R, H, dh), np.float64) for _ in range(3))
    rc = _load().ref_item_bwd(_p(Q), _p(K), _p(V), _p(dO), f64, B, R, C, H, dh, _p(nt), _p(m),
                              ctypes.c_double(scale), n, _p(sb), _p(sc), _p(dQ), _p(dK), _p(dV), int(nthreads))
    if rc:
        raise ValueError("ref_item_bwd rc=%d" % rc)
    if cols is None:
        return tuple(np.ascontiguousarray(x.reshape(B, C, R, H, dh).transpose(0, 2, 1, 3, 4))
                     for x in (dQ, dK, dV))
    return dQ, dK, dV
