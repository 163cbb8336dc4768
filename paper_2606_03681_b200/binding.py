"""Thin ctypes binding of libtabattn (include/tabattn.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used here for
device memory (``tensor.data_ptr()``) and the current stream, nothing else.  There is no CPU
fallback: if ``libtabattn.so`` has not been built (``python -m paper_2606_03681_b200.build``)
importing the library raises.

Tensors are ``[B,R,C,H,dh]`` torch.bfloat16 CUDA tensors, contiguous; ``n_train`` is an int32
CUDA tensor ``[B]``; ``col_valid`` an optional uint8 CUDA tensor ``[B,C]``.  Feature LSE is
``[B,R,H,C]`` f32, item LSE ``[B,C,H,R]`` f32.
"""
import contextlib
import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtabattn.so")

OP_FEATURE_FWD, OP_FEATURE_BWD, OP_ITEM_FWD, OP_ITEM_BWD = 0, 1, 2, 3
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_WORKSPACE, ERR_CUDA = 0, 1, 2, 3, 4

EXPORTS = ("tabattn_feature_fwd", "tabattn_feature_bwd", "tabattn_item_fwd", "tabattn_item_bwd",
           "tabattn_feature_fwd_infer", "tabattn_item_fwd_infer", "tabattn_workspace_bytes", "tabattn_status_string", "tabattn_version", "tabattn_launch_count")


class TabattnShape(ctypes.Structure):
    """Mirror of ``tabattn_shape`` (include/tabattn.h)."""
    _fields_ = [("B", ctypes.c_int32), ("R", ctypes.c_int32), ("C", ctypes.c_int32),
                ("H", ctypes.c_int32), ("dh", ctypes.c_int32),
                ("n_train", ctypes.c_void_p), ("n_train_host", ctypes.c_void_p),
                ("col_valid", ctypes.c_void_p), ("softmax_scale", ctypes.c_float)]


class TabattnError(RuntimeError):
    def __init__(self, status, what):
        self.status = int(status)
        super().__init__("%s: %s (status %d)" % (what, status_string(status), status))


_lib = None


def lib():
    """The loaded C-ABI library.  Raises if it has not been built: there is no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libtabattn.so is missing (%s): run `python -m paper_2606_03681_b200.build`; "
                              "there is no CPU or PyTorch fallback" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        vp, sz = ctypes.c_void_p, ctypes.c_size_t
        shp = ctypes.POINTER(TabattnShape)
        L.tabattn_feature_fwd.argtypes = [shp, vp, vp, vp, vp, vp, vp, sz, vp]
        L.tabattn_item_fwd.argtypes = [shp, vp, vp, vp, vp, vp, vp, sz, vp]
        L.tabattn_feature_bwd.argtypes = [shp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
        L.tabattn_item_bwd.argtypes = [shp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
        i32 = ctypes.c_int32
        L.tabattn_feature_fwd_infer.argtypes = [shp, vp, vp, vp, vp, i32, i32, vp, sz, vp]
        L.tabattn_item_fwd_infer.argtypes = [shp, vp, vp, vp, vp, i32, i32, vp, sz, vp]
        for f in (L.tabattn_feature_fwd, L.tabattn_item_fwd, L.tabattn_feature_bwd, L.tabattn_item_bwd,
                  L.tabattn_feature_fwd_infer, L.tabattn_item_fwd_infer):
            f.restype = ctypes.c_int
        L.tabattn_workspace_bytes.argtypes = [shp, ctypes.c_int]
        L.tabattn_workspace_bytes.restype = sz
        L.tabattn_status_string.argtypes = [ctypes.c_int]
        L.tabattn_status_string.restype = ctypes.c_char_p
        L.tabattn_version.argtypes = []
        L.tabattn_version.restype = ctypes.c_int
        L.tabattn_launch_count.argtypes = []
        L.tabattn_launch_count.restype = ctypes.c_uint64
        _lib = L
    return _lib


def status_string(status) -> str:
    return lib().tabattn_status_string(int(status)).decode()


def version() -> int:
    return int(lib().tabattn_version())


def launch_count() -> int:
    """Kernels launched by libtabattn in this process so far (tabattn.h: tabattn_launch_count)."""
    return int(lib().tabattn_launch_count())


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else None


def make_shape(Q, n_train=None, col_valid=None, n_train_host=None, softmax_scale=0.0):
    """Build the ``tabattn_shape`` for a ``[B,R,C,H,dh]`` tensor.  Returns (struct, keepalive)."""
    B, R, C, H, dh = Q.shape
    keep = [n_train, col_valid]
    nth = None
    if n_train_host is not None:
        nth = (ctypes.c_int32 * B)(*[int(x) for x in n_train_host])
        keep.append(nth)
    s = TabattnShape(B, R, C, H, dh,
                     n_train.data_ptr() if n_train is not None else None,
                     ctypes.cast(nth, ctypes.c_void_p).value if nth is not None else None,
                     col_valid.data_ptr() if col_valid is not None else None,
                     float(softmax_scale))
    return s, keep


def workspace_bytes(shape: TabattnShape, op: int) -> int:
    return int(lib().tabattn_workspace_bytes(ctypes.byref(shape), int(op)))


def _check_inputs(*ts):
    """Cell tensors (inputs and caller-provided outputs): contiguous CUDA bfloat16 [B,R,C,H,dh] on one device."""
    t0 = ts[0]
    if t0.dim() != 5:
        raise ValueError("expected [B,R,C,H,dh]")
    for t in ts:
        if t is None:
            continue
        if (t.dtype != torch.bfloat16 or not t.is_cuda or not t.is_contiguous() or t.shape != t0.shape
                or t.device != t0.device):
            raise ValueError("tensors must be contiguous CUDA bfloat16 of one shape [B,R,C,H,dh] on one device")


def _check_aux(Q, n_train=None, col_valid=None, LSE=None, lse_shape=None):
    """The non-cell arguments cross the ABI as raw pointers: a wrong dtype would be read as garbage
    (torch's default int64 n_train reads as int32 pairs), so it is rejected here."""
    B, R, C, H, dh = Q.shape
    if n_train is not None:
        if (n_train.dtype != torch.int32 or not n_train.is_cuda or not n_train.is_contiguous()
                or tuple(n_train.shape) != (B,) or n_train.device != Q.device):
            raise ValueError("n_train must be a contiguous CUDA int32 tensor [B] on the device of Q")
    if col_valid is not None:
        if (col_valid.dtype not in (torch.uint8, torch.bool) or not col_valid.is_cuda
                or not col_valid.is_contiguous() or tuple(col_valid.shape) != (B, C) or col_valid.device != Q.device):
            raise ValueError("col_valid must be a contiguous CUDA uint8/bool tensor [B,C] on the device of Q")
    if LSE is not None:
        if (LSE.dtype != torch.float32 or not LSE.is_cuda or not LSE.is_contiguous()
                or tuple(LSE.shape) != tuple(lse_shape) or LSE.device != Q.device):
            raise ValueError("LSE must be a contiguous CUDA float32 tensor %s on the device of Q" % (lse_shape,))


def _on(device):
    """Make `device` the calling thread's current CUDA device for the ABI call (the library launches on it)."""
    if device.index is None or device.index == torch.cuda.current_device():
        return contextlib.nullcontext()
    return torch.cuda.device(device)


def _stream(stream, device):
    if stream is None:
        stream = torch.cuda.current_stream(device)
    return ctypes.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _workspace(shape, op, ws, device):
    need = workspace_bytes(shape, op)
    if ws is None and need:
        ws = torch.empty(need, dtype=torch.uint8, device=device)
    if ws is not None and (not ws.is_cuda or not ws.is_contiguous() or ws.device != device):
        raise ValueError("ws must be a contiguous CUDA tensor on the device of Q")
    return ws, (ws.numel() * ws.element_size() if ws is not None else 0)


def _raise(st, what):
    if st != OK:
        raise TabattnError(st, what)


def tabattn_feature_fwd(Q, K, V, col_valid=None, softmax_scale=0.0, O=None, LSE=None, ws=None, stream=None):
    """Feature-axis attention forward (tabattn.h: tabattn_feature_fwd).  Returns (O, LSE[B,R,H,C])."""
    _check_inputs(Q, K, V, O)
    B, R, C, H, dh = Q.shape
    _check_aux(Q, None, col_valid, LSE, (B, R, H, C))
    shape, keep = make_shape(Q, None, col_valid, None, softmax_scale)
    O = torch.empty_like(Q) if O is None else O
    LSE = torch.empty((B, R, H, C), dtype=torch.float32, device=Q.device) if LSE is None else LSE
    ws, nws = _workspace(shape, OP_FEATURE_FWD, ws, Q.device)
    with _on(Q.device):
        st = lib().tabattn_feature_fwd(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), _ptr(O), _ptr(LSE),
                                       _ptr(ws), nws, _stream(stream, Q.device))
    _raise(st, "tabattn_feature_fwd")
    return O, LSE


def tabattn_feature_bwd(Q, K, V, O, dO, LSE, col_valid=None, softmax_scale=0.0, dQ=None, dK=None, dV=None,
                        ws=None, stream=None):
    """Feature-axis attention backward (tabattn.h: tabattn_feature_bwd).  Returns (dQ, dK, dV)."""
    _check_inputs(Q, K, V, O, dO, dQ, dK, dV)
    B, R, C, H, dh = Q.shape
    _check_aux(Q, None, col_valid, LSE, (B, R, H, C))
    shape, keep = make_shape(Q, None, col_valid, None, softmax_scale)
    dQ = torch.empty_like(Q) if dQ is None else dQ
    dK = torch.empty_like(Q) if dK is None else dK
    dV = torch.empty_like(Q) if dV is None else dV
    ws, nws = _workspace(shape, OP_FEATURE_BWD, ws, Q.device)
    with _on(Q.device):
        st = lib().tabattn_feature_bwd(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), _ptr(O), _ptr(dO),
                                       _ptr(LSE), _ptr(dQ), _ptr(dK), _ptr(dV), _ptr(ws), nws,
                                       _stream(stream, Q.device))
    _raise(st, "tabattn_feature_bwd")
    return dQ, dK, dV


def tabattn_item_fwd(Q, K, V, n_train, col_valid=None, softmax_scale=0.0, n_train_host=None, O=None, LSE=None,
                     ws=None, stream=None):
    """Item-axis attention forward (tabattn.h: tabattn_item_fwd).  Returns (O, LSE[B,C,H,R])."""
    _check_inputs(Q, K, V, O)
    B, R, C, H, dh = Q.shape
    _check_aux(Q, n_train, col_valid, LSE, (B, C, H, R))
    shape, keep = make_shape(Q, n_train, col_valid, n_train_host, softmax_scale)
    O = torch.empty_like(Q) if O is None else O
    LSE = torch.empty((B, C, H, R), dtype=torch.float32, device=Q.device) if LSE is None else LSE
    ws, nws = _workspace(shape, OP_ITEM_FWD, ws, Q.device)
    with _on(Q.device):
        st = lib().tabattn_item_fwd(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), _ptr(O), _ptr(LSE),
                                    _ptr(ws), nws, _stream(stream, Q.device))
    _raise(st, "tabattn_item_fwd")
    return O, LSE


def tabattn_item_bwd(Q, K, V, O, dO, LSE, n_train, col_valid=None, softmax_scale=0.0, n_train_host=None,
                     dQ=None, dK=None, dV=None, ws=None, stream=None):
    """Item-axis attention backward (tabattn.h: tabattn_item_bwd).  Returns (dQ, dK, dV)."""
    _check_inputs(Q, K, V, O, dO, dQ, dK, dV)
    B, R, C, H, dh = Q.shape
    _check_aux(Q, n_train, col_valid, LSE, (B, C, H, R))
    shape, keep = make_shape(Q, n_train, col_valid, n_train_host, softmax_scale)
    dQ = torch.empty_like(Q) if dQ is None else dQ
    dK = torch.empty_like(Q) if dK is None else dK
    dV = torch.empty_like(Q) if dV is None else dV
    ws, nws = _workspace(shape, OP_ITEM_BWD, ws, Q.device)
    with _on(Q.device):
        st = lib().tabattn_item_bwd(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), _ptr(O), _ptr(dO), _ptr(LSE),
                                    _ptr(dQ), _ptr(dK), _ptr(dV), _ptr(ws), nws, _stream(stream, Q.device))
    _raise(st, "tabattn_item_bwd")
    return dQ, dK, dV


def tabattn_feature_fwd_infer(Q, K, V, row0, row1, col_valid=None, softmax_scale=0.0, O=None, ws=None, stream=None):
    """Forward-only feature attention on the table rows [row0, row1), no LSE (tabattn.h:
    tabattn_feature_fwd_infer).  Returns O; rows outside the range are left as they were."""
    _check_inputs(Q, K, V, O)
    _check_aux(Q, None, col_valid)
    shape, keep = make_shape(Q, None, col_valid, None, softmax_scale)
    O = torch.empty_like(Q) if O is None else O
    ws, nws = _workspace(shape, OP_FEATURE_FWD, ws, Q.device)
    with _on(Q.device):
        st = lib().tabattn_feature_fwd_infer(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), _ptr(O), int(row0),
                                             int(row1), _ptr(ws), nws, _stream(stream, Q.device))
    _raise(st, "tabattn_feature_fwd_infer")
    return O


def tabattn_item_fwd_infer(Q, K, V, n_train, row0, row1, col_valid=None, softmax_scale=0.0, n_train_host=None,
                           O=None, ws=None, stream=None):
    """Forward-only item attention: query rows [row0, row1) against the train rows, no LSE (tabattn.h:
    tabattn_item_fwd_infer).  Returns O; rows outside the range are left as they were."""
    _check_inputs(Q, K, V, O)
    _check_aux(Q, n_train, col_valid)
    shape, keep = make_shape(Q, n_train, col_valid, n_train_host, softmax_scale)
    O = torch.empty_like(Q) if O is None else O
    ws, nws = _workspace(shape, OP_ITEM_FWD, ws, Q.device)
    with _on(Q.device):
        st = lib().tabattn_item_fwd_infer(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), _ptr(O), int(row0),
                                          int(row1), _ptr(ws), nws, _stream(stream, Q.device))
    _raise(st, "tabattn_item_fwd_infer")
    return O
