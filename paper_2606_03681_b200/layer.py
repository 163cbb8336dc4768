"""One layer of the hot path = the four C-ABI calls of SURVEY.md §8(a), in training order:
feature fwd, item fwd, item bwd, feature bwd (each block applies feature-axis
attention then sample-axis attention; backward runs in reverse order).

Marshalling only: buffers are preallocated once (``LayerBuffers``) so the timed region holds
nothing but kernel launches; ``layer_fwd_bwd_host`` is the same step driven from pinned HOST
buffers (host->device copies of the eight inputs, device->host read of the results).
"""
import torch

from . import binding as _b


class LayerBuffers:
    """Outputs + workspace for one layer of shape [B,R,C,H,dh]; reusable across calls."""

    def __init__(self, B, R, C, H, dh, device="cuda"):
        shp = (B, R, C, H, dh)
        bf = dict(dtype=torch.bfloat16, device=device)
        self.shape = shp
        self.O_f = torch.empty(shp, **bf)
        self.O_i = torch.empty(shp, **bf)
        self.LSE_f = torch.empty((B, R, H, C), dtype=torch.float32, device=device)
        self.LSE_i = torch.empty((B, C, H, R), dtype=torch.float32, device=device)
        self.grads_f = tuple(torch.empty(shp, **bf) for _ in range(3))
        self.grads_i = tuple(torch.empty(shp, **bf) for _ in range(3))
        probe = torch.empty((0,), **bf)
        s = _b.TabattnShape(B, R, C, H, dh, None, None, None, 0.0)
        need = max(_b.workspace_bytes(s, op) for op in range(4))
        self.ws = torch.empty(max(need, 16), dtype=torch.uint8, device=device)
        del probe


def layer_fwd_bwd(feat, item, n_train, col_valid, buf: LayerBuffers, n_train_host=None, stream=None):
    """Enqueue feature fwd, item fwd, item bwd, feature bwd on the current stream.

    ``feat`` / ``item`` are dicts with device tensors Q, K, V, dO.  Results land in ``buf``."""
    _b.tabattn_feature_fwd(feat["Q"], feat["K"], feat["V"], col_valid, O=buf.O_f, LSE=buf.LSE_f, ws=buf.ws,
                           stream=stream)
    _b.tabattn_item_fwd(item["Q"], item["K"], item["V"], n_train, col_valid, n_train_host=n_train_host,
                        O=buf.O_i, LSE=buf.LSE_i, ws=buf.ws, stream=stream)
    _b.tabattn_item_bwd(item["Q"], item["K"], item["V"], buf.O_i, item["dO"], buf.LSE_i, n_train, col_valid,
                        n_train_host=n_train_host, dQ=buf.grads_i[0], dK=buf.grads_i[1], dV=buf.grads_i[2],
                        ws=buf.ws, stream=stream)
    _b.tabattn_feature_bwd(feat["Q"], feat["K"], feat["V"], buf.O_f, feat["dO"], buf.LSE_f, col_valid,
                           dQ=buf.grads_f[0], dK=buf.grads_f[1], dV=buf.grads_f[2], ws=buf.ws, stream=stream)
    return buf


class LayerGraph:
    """The four calls of one layer captured once into a CUDA graph and replayed with one launch.

    For launch-bound shapes: Tiny is 83 us/layer through the four ctypes calls (host-bound) and 27 us/layer as a graph
    replay on a B200; at Base and above the kernels dominate and a graph changes nothing.  The library allocates
    nothing and reads no host state at launch time besides its per-device caches, which the warm-up call fills before
    the capture, so its calls are capturable as they are (tensor maps travel as kernel parameters).  The graph holds
    the POINTERS of ``feat`` / ``item`` / ``n_train`` / ``col_valid`` / ``buf``: a replay reads whatever those tensors
    hold then and writes its results into ``buf``; keep them alive and do not reallocate them."""

    def __init__(self, feat, item, n_train, col_valid, buf: LayerBuffers, n_train_host=None):
        self.buf = buf
        self._keep = (feat, item, n_train, col_valid)
        cur = torch.cuda.current_stream()
        side = torch.cuda.Stream()
        side.wait_stream(cur)
        with torch.cuda.stream(side):
            layer_fwd_bwd(feat, item, n_train, col_valid, buf, n_train_host)   # warm-up: per-device set-up, caches
            side.synchronize()
            n0 = _b.launch_count()
            self.graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(self.graph, stream=side):
                layer_fwd_bwd(feat, item, n_train, col_valid, buf, n_train_host)
            self.kernels_per_replay = _b.launch_count() - n0
        cur.wait_stream(side)

    def replay(self):
        """Enqueue the captured layer on the current stream; results land in ``self.buf``."""
        self.graph.replay()
        return self.buf


def _slice(d, b0, b1):
    return {k: v[b0:b1] for k, v in d.items()}


class _View:
    """LayerBuffers restricted to tables [b0, b1): B is the outermost dimension of every buffer, so the
    slices are contiguous and the C ABI can be called on them directly."""

    def __init__(self, buf, b0, b1):
        self.O_f, self.O_i = buf.O_f[b0:b1], buf.O_i[b0:b1]
        self.LSE_f, self.LSE_i = buf.LSE_f[b0:b1], buf.LSE_i[b0:b1]
        self.grads_f = tuple(g[b0:b1] for g in buf.grads_f)
        self.grads_i = tuple(g[b0:b1] for g in buf.grads_i)
        self.ws = buf.ws


def layer_fwd_bwd_host(feat_host, item_host, feat_dev, item_dev, out_host, n_train, col_valid,
                       buf: LayerBuffers, n_train_host=None, groups=16):
    """The same step from pinned host buffers: H2D of the 8 inputs, the four calls, D2H of the
    8 results (O and dQ/dK/dV of both axes) into ``out_host``.  Returns (h2d_bytes, d2h_bytes).

    The tables are independent, so the step is pipelined over ``groups`` table groups on three streams
    (copy-in, the caller's current stream for the kernels, copy-out): group k+1 is uploaded and group k-1
    downloaded while group k computes -- PCIe is full duplex and the copies dominate the step
    (2 x 1.1 GB against 2.5 ms of kernels at base).  On return the current stream has been made to wait
    for the last download, so events recorded on it bracket the whole step."""
    B, R, C, H, _ = buf.shape
    # table-group boundaries must keep every sliced buffer 16-byte aligned: the f32 LSE slices start at
    # b0 * R*H*C * 4 bytes, so b0 is kept a multiple of 4 / gcd(R*H*C, 4)
    import math
    align = 4 // math.gcd(R * H * C, 4)
    groups = max(1, min(groups, B // align if B >= align else 1))
    cur = torch.cuda.current_stream()
    if getattr(buf, "_side", None) is None:
        buf._side = (torch.cuda.Stream(), torch.cuda.Stream())
    s_in, s_out = buf._side
    s_in.wait_stream(cur)     # the previous step's kernels are done with the staging buffers
    s_out.wait_stream(cur)
    h2d = d2h = 0
    cuts = sorted({min(B, (B * g // groups) // align * align) for g in range(groups)} | {B})
    bounds = [(a, b) for a, b in zip(cuts[:-1], cuts[1:]) if b > a]
    for b0, b1 in bounds:
        with torch.cuda.stream(s_in):
            for src, dst in ((feat_host, feat_dev), (item_host, item_dev)):
                for k in ("Q", "K", "V", "dO"):
                    dst[k][b0:b1].copy_(src[k][b0:b1], non_blocking=True)
                    h2d += src[k][b0:b1].numel() * src[k].element_size()
            ev_in = torch.cuda.Event()
            ev_in.record(s_in)
        cur.wait_event(ev_in)
        view = _View(buf, b0, b1)
        layer_fwd_bwd(_slice(feat_dev, b0, b1), _slice(item_dev, b0, b1), n_train[b0:b1],
                      None if col_valid is None else col_valid[b0:b1], view,
                      None if n_train_host is None else n_train_host[b0:b1])
        ev_c = torch.cuda.Event()
        ev_c.record(cur)
        with torch.cuda.stream(s_out):
            s_out.wait_event(ev_c)
            results = (view.O_f, view.O_i) + view.grads_f + view.grads_i
            for dst, src in zip(out_host, results):
                dst[b0:b1].copy_(src, non_blocking=True)
                d2h += src.numel() * src.element_size()
    cur.wait_stream(s_out)
    return h2d, d2h
