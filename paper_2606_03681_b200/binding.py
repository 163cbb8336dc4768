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
           "tabattn_item_fwd_noalloc",
           "tabattn_feature_fwd_infer", "tabattn_item_fwd_infer", "tabattn_workspace_bytes",
           "tabattn_attn_block_fwd", "tabattn_attn_block_bwd", "tabattn_attn_block_workspace_bytes",
           "tabattn_mlp_fwd", "tabattn_mlp_bwd", "tabattn_mlp_workspace_bytes",
           "tabattn_newton_schulz", "tabattn_newton_schulz_workspace_bytes", "tabattn_status_string", "tabattn_version", "tabattn_launch_count")


class TabattnShape(ctypes.Structure):
    """Mirror of ``tabattn_shape`` (include/tabattn.h)."""
    _fields_ = [("B", ctypes.c_int32), ("R", ctypes.c_int32), ("C", ctypes.c_int32),
                ("H", ctypes.c_int32), ("dh", ctypes.c_int32),
                ("n_train", ctypes.c_void_p), ("n_train_host", ctypes.c_void_p),
                ("col_valid", ctypes.c_void_p), ("softmax_scale", ctypes.c_float)]


class TabattnAttnSaved(ctypes.Structure):
    """Mirror of ``tabattn_attn_saved``."""
    _fields_ = [(n, ctypes.c_void_p) for n in ("h", "rstd", "q", "k", "v", "o", "lse")]


class TabattnMlpSaved(ctypes.Structure):
    """Mirror of ``tabattn_mlp_saved``."""
    _fields_ = [(n, ctypes.c_void_p) for n in ("h", "rstd", "u", "a")]


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
        L.tabattn_item_fwd_noalloc.argtypes = [shp, vp, vp, vp, vp, vp, vp]
        for f in (L.tabattn_feature_fwd, L.tabattn_item_fwd, L.tabattn_feature_bwd, L.tabattn_item_bwd,
                  L.tabattn_feature_fwd_infer, L.tabattn_item_fwd_infer, L.tabattn_item_fwd_noalloc):
            f.restype = ctypes.c_int
        f32, i64 = ctypes.c_float, ctypes.c_int64
        asv, msv = ctypes.POINTER(TabattnAttnSaved), ctypes.POINTER(TabattnMlpSaved)
        L.tabattn_attn_block_fwd.argtypes = [shp, i32, f32, f32, vp, vp, vp, vp, vp, asv, vp, sz, vp]
        L.tabattn_attn_block_bwd.argtypes = [shp, i32, f32, vp, vp, vp, vp, asv, vp, vp, vp, vp, vp, vp, sz, vp]
        L.tabattn_attn_block_workspace_bytes.argtypes = [shp, i32, i32]
        L.tabattn_attn_block_workspace_bytes.restype = sz
        L.tabattn_mlp_fwd.argtypes = [i64, i32, i32, f32, f32, vp, vp, vp, vp, vp, msv, vp]
        L.tabattn_mlp_bwd.argtypes = [i64, i32, i32, f32, vp, vp, vp, vp, msv, vp, vp, vp, vp, vp, vp, sz, vp]
        L.tabattn_mlp_workspace_bytes.argtypes = [i64, i32, i32]
        L.tabattn_mlp_workspace_bytes.restype = sz
        L.tabattn_newton_schulz.argtypes = [i32, i32, i32, vp, vp, i32, vp, sz, vp]
        L.tabattn_newton_schulz_workspace_bytes.argtypes = [i32, i32, i32]
        L.tabattn_newton_schulz_workspace_bytes.restype = sz
        for f in (L.tabattn_attn_block_fwd, L.tabattn_attn_block_bwd, L.tabattn_mlp_fwd, L.tabattn_mlp_bwd,
                  L.tabattn_newton_schulz):
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


NOALLOC_MAX_BC = 65536   # TABATTN_NOALLOC_MAX_BC


def tabattn_item_fwd_noalloc(Q, K, V, n_train, col_valid=None, softmax_scale=0.0, n_train_host=None, O=None,
                             LSE=None, stream=None):
    """Item-axis attention forward with the scratch inside the library (tabattn.h: tabattn_item_fwd_noalloc): the
    C call allocates nothing.  Pass preallocated ``O`` / ``LSE`` to keep the whole call allocation-free; masked calls
    need B*C <= NOALLOC_MAX_BC; calls that overlap on the GPU race on the shared scratch."""
    _check_inputs(Q, K, V, O)
    B, R, C, H, dh = Q.shape
    _check_aux(Q, n_train, col_valid, LSE, (B, C, H, R))
    shape, keep = make_shape(Q, n_train, col_valid, n_train_host, softmax_scale)
    O = torch.empty_like(Q) if O is None else O
    LSE = torch.empty((B, C, H, R), dtype=torch.float32, device=Q.device) if LSE is None else LSE
    with _on(Q.device):
        st = lib().tabattn_item_fwd_noalloc(ctypes.byref(shape), _ptr(Q), _ptr(K), _ptr(V), _ptr(O), _ptr(LSE),
                                            _stream(stream, Q.device))
    _raise(st, "tabattn_item_fwd_noalloc")
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


# ---- sub-blocks (tabattn.h: "The sub-blocks around the attention kernels") ---------
def _check_dense(t, dtype, shape, what):
    if t.dtype != dtype or not t.is_cuda or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
        raise ValueError("%s must be a contiguous CUDA %s tensor of shape %s" % (what, dtype, tuple(shape)))


def _bytes_ws(need, ws, device):
    if ws is None and need:
        ws = torch.empty(need, dtype=torch.uint8, device=device)
    return ws, (ws.numel() * ws.element_size() if ws is not None else 0)


class AttnSaved:
    """Caller-owned activations the attention sub-block's forward leaves for its backward."""

    def __init__(self, x, H, axis):
        B, R, C, e = x.shape
        bf = dict(dtype=torch.bfloat16, device=x.device)
        self.h, self.q, self.k, self.v, self.o = (torch.empty((B, R, C, e), **bf) for _ in range(5))
        self.rstd = torch.empty((B * R * C,), dtype=torch.float32, device=x.device)
        self.lse = torch.empty((B, R, H, C) if axis == 0 else (B, C, H, R), dtype=torch.float32, device=x.device)

    def struct(self):
        return TabattnAttnSaved(*[t.data_ptr() for t in (self.h, self.rstd, self.q, self.k, self.v, self.o, self.lse)])


class MlpSaved:
    def __init__(self, x, hidden):
        cells, e = x.numel() // x.shape[-1], x.shape[-1]
        bf = dict(dtype=torch.bfloat16, device=x.device)
        self.h = torch.empty((cells, e), **bf)
        self.u = torch.empty((cells, hidden), **bf)
        self.a = torch.empty((cells, hidden), **bf)
        self.rstd = torch.empty((cells,), dtype=torch.float32, device=x.device)

    def struct(self):
        return TabattnMlpSaved(*[t.data_ptr() for t in (self.h, self.rstd, self.u, self.a)])


def _block_shape(x, H, n_train, col_valid, n_train_host):
    B, R, C, e = x.shape
    if e % H:
        raise ValueError("e must be H * dh")
    q5 = x.view(B, R, C, H, e // H)
    _check_aux(q5, n_train, col_valid)
    return make_shape(q5, n_train, col_valid, n_train_host, 0.0)


def tabattn_attn_block_fwd(axis, x, g, Wqkv, Wo, H, n_train=None, col_valid=None, alpha=1.0, eps=1e-6,
                           n_train_host=None, saved=None, y=None, ws=None, stream=None):
    """Attention sub-block forward (tabattn.h: tabattn_attn_block_fwd).  x [B,R,C,e] bf16; axis 0 feature, 1 item.
    Returns (y, saved)."""
    B, R, C, e = x.shape
    for t, shp, nm in ((x, x.shape, "x"), (g, (e,), "g"), (Wqkv, (3 * e, e), "Wqkv"), (Wo, (e, e), "Wo")):
        _check_dense(t, torch.bfloat16, shp, nm)
    shape, keep = _block_shape(x, H, n_train, col_valid, n_train_host)
    saved = AttnSaved(x, H, axis) if saved is None else saved
    y = torch.empty_like(x) if y is None else y
    sv = saved.struct()
    ws, nws = _bytes_ws(int(lib().tabattn_attn_block_workspace_bytes(ctypes.byref(shape), axis, 0)), ws, x.device)
    with _on(x.device):
        st = lib().tabattn_attn_block_fwd(ctypes.byref(shape), axis, float(alpha), float(eps), _ptr(x), _ptr(g),
                                          _ptr(Wqkv), _ptr(Wo), _ptr(y), ctypes.byref(sv), _ptr(ws), nws,
                                          _stream(stream, x.device))
    _raise(st, "tabattn_attn_block_fwd")
    return y, saved


def tabattn_attn_block_bwd(axis, x, g, Wqkv, Wo, H, saved, dy, n_train=None, col_valid=None, alpha=1.0,
                           n_train_host=None, ws=None, stream=None):
    """Attention sub-block backward.  Returns (dx bf16, dg f32 [e], dWqkv f32 [3e,e], dWo f32 [e,e])."""
    B, R, C, e = x.shape
    _check_dense(dy, torch.bfloat16, x.shape, "dy")
    shape, keep = _block_shape(x, H, n_train, col_valid, n_train_host)
    f32 = dict(dtype=torch.float32, device=x.device)
    dx, dg = torch.empty_like(x), torch.empty((e,), **f32)
    dWqkv, dWo = torch.empty((3 * e, e), **f32), torch.empty((e, e), **f32)
    sv = saved.struct()
    ws, nws = _bytes_ws(int(lib().tabattn_attn_block_workspace_bytes(ctypes.byref(shape), axis, 1)), ws, x.device)
    with _on(x.device):
        st = lib().tabattn_attn_block_bwd(ctypes.byref(shape), axis, float(alpha), _ptr(x), _ptr(g), _ptr(Wqkv),
                                          _ptr(Wo), ctypes.byref(sv), _ptr(dy), _ptr(dx), _ptr(dg), _ptr(dWqkv),
                                          _ptr(dWo), _ptr(ws), nws, _stream(stream, x.device))
    _raise(st, "tabattn_attn_block_bwd")
    return dx, dg, dWqkv, dWo


def tabattn_mlp_fwd(x, g, W1, W2, alpha=1.0, eps=1e-6, saved=None, y=None, stream=None):
    """MLP sub-block forward (tabattn.h: tabattn_mlp_fwd).  x [..., e] bf16.  Returns (y, saved)."""
    e, hidden = x.shape[-1], W1.shape[0]
    cells = x.numel() // e
    for t, shp, nm in ((x, x.shape, "x"), (g, (e,), "g"), (W1, (hidden, e), "W1"), (W2, (e, hidden), "W2")):
        _check_dense(t, torch.bfloat16, shp, nm)
    saved = MlpSaved(x, hidden) if saved is None else saved
    y = torch.empty_like(x) if y is None else y
    sv = saved.struct()
    with _on(x.device):
        st = lib().tabattn_mlp_fwd(cells, e, hidden, float(alpha), float(eps), _ptr(x), _ptr(g), _ptr(W1), _ptr(W2),
                                   _ptr(y), ctypes.byref(sv), _stream(stream, x.device))
    _raise(st, "tabattn_mlp_fwd")
    return y, saved


def tabattn_mlp_bwd(x, g, W1, W2, saved, dy, alpha=1.0, ws=None, stream=None):
    """MLP sub-block backward.  Returns (dx bf16, dg f32 [e], dW1 f32 [hidden,e], dW2 f32 [e,hidden])."""
    e, hidden = x.shape[-1], W1.shape[0]
    cells = x.numel() // e
    _check_dense(dy, torch.bfloat16, x.shape, "dy")
    f32 = dict(dtype=torch.float32, device=x.device)
    dx, dg = torch.empty_like(x), torch.empty((e,), **f32)
    dW1, dW2 = torch.empty((hidden, e), **f32), torch.empty((e, hidden), **f32)
    sv = saved.struct()
    ws, nws = _bytes_ws(int(lib().tabattn_mlp_workspace_bytes(cells, e, hidden)), ws, x.device)
    with _on(x.device):
        st = lib().tabattn_mlp_bwd(cells, e, hidden, float(alpha), _ptr(x), _ptr(g), _ptr(W1), _ptr(W2),
                                   ctypes.byref(sv), _ptr(dy), _ptr(dx), _ptr(dg), _ptr(dW1), _ptr(dW2), _ptr(ws), nws,
                                   _stream(stream, x.device))
    _raise(st, "tabattn_mlp_bwd")
    return dx, dg, dW1, dW2


def tabattn_newton_schulz(G, steps=5, X=None, ws=None, stream=None):
    """Batched Newton-Schulz orthogonalisation (tabattn.h: tabattn_newton_schulz).  G [nb,m,n] bf16, m <= n."""
    if G.dim() != 3:
        raise ValueError("G must be [nb, m, n]")
    nb, m, n = G.shape
    _check_dense(G, torch.bfloat16, G.shape, "G")
    X = torch.empty_like(G) if X is None else X
    ws, nws = _bytes_ws(int(lib().tabattn_newton_schulz_workspace_bytes(nb, m, n)), ws, G.device)
    with _on(G.device):
        st = lib().tabattn_newton_schulz(nb, m, n, _ptr(G), _ptr(X), int(steps), _ptr(ws), nws,
                                         _stream(stream, G.device))
    _raise(st, "tabattn_newton_schulz")
    return X
