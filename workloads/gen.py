"""Seeded tensors for one attention call (Q, K, V, dO) of a config.

Two backends with the same recipe but different random streams:

* ``device=None``  -> numpy (``default_rng([seed, layer, axis, tensor])``,
  ``standard_normal(float32)`` -> bf16 RNE); returns ``uint16`` arrays.  This is
  what the CPU-only tests and the small GPU parity tests use.
* ``device="cuda"`` -> torch on the GPU (``torch.Generator(device)`` seeded from
  the same four integers, ``randn(float32).to(bfloat16)``); returns torch bf16
  tensors.  Used for the large configs; the oracle reads the same bits back
  from the device, so the choice of stream cannot affect parity.

No attention arithmetic lives here (the Ragged config's Q = bf16(X @ W)
projection, reading c17 of SURVEY.md §8(c), is input synthesis: it only makes
inputs whose scale and correlation look like a projected embedding).
"""
import numpy as np

from .bf16 import f32_to_bf16_bits, bf16_bits_to_f32
from .configs import TabShape

_AXIS = {"feature": 0, "item": 1}
_TENSOR = {"Q": 0, "K": 1, "V": 2, "dO": 3, "X": 7}


def _seed_tuple(cfg, layer, axis, tensor):
    return [int(cfg.seed), int(layer), _AXIS[axis], _TENSOR[tensor]]


def _torch_seed(cfg, layer, axis, tensor):
    s = _seed_tuple(cfg, layer, axis, tensor)
    return ((s[0] * 1000 + s[1]) * 10 + s[2]) * 10 + s[3]


def _normal_np(cfg, layer, axis, tensor, shape, scale=1.0):
    rng = np.random.default_rng(_seed_tuple(cfg, layer, axis, tensor))
    x = rng.standard_normal(size=shape, dtype=np.float32)
    if scale != 1.0:
        x *= np.float32(scale)
    return f32_to_bf16_bits(x)


def _normal_torch(cfg, layer, axis, tensor, shape, device, scale=1.0):
    import torch
    g = torch.Generator(device=device)
    g.manual_seed(_torch_seed(cfg, layer, axis, tensor))
    x = torch.randn(shape, generator=g, device=device, dtype=torch.float32)
    if scale != 1.0:
        x *= scale
    return x.to(torch.bfloat16)


def _projected_np(cfg, layer, axis, names):
    shape = (cfg.B, cfg.R, cfg.C, cfg.d)
    x = bf16_bits_to_f32(_normal_np(cfg, 0, "feature", "X", shape))
    out = {}
    for t in names:
        w = bf16_bits_to_f32(_normal_np(cfg, layer, axis, t, (cfg.d, cfg.d),
                                        scale=cfg.d ** -0.5))
        y = (x.reshape(-1, cfg.d) @ w).astype(np.float32)
        out[t] = f32_to_bf16_bits(y).reshape(cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh)
    return out


def _projected_torch(cfg, layer, axis, names, device, x_cache=None):
    import torch
    shape = (cfg.B, cfg.R, cfg.C, cfg.d)
    if x_cache is not None and "X" in x_cache:
        x = x_cache["X"]
    else:
        x = _normal_torch(cfg, 0, "feature", "X", shape, device)
        if x_cache is not None:
            x_cache["X"] = x
    out = {}
    for t in names:
        w = _normal_torch(cfg, layer, axis, t, (cfg.d, cfg.d), device, scale=cfg.d ** -0.5)
        y = (x.reshape(-1, cfg.d).float() @ w.float()).to(torch.bfloat16)
        out[t] = y.reshape(cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh).contiguous()
    return out


def make_call_inputs(cfg: TabShape, axis: str, layer: int = 0, device=None, x_cache=None):
    """Q, K, V, dO for one attention call: dict of [B,R,C,H,dh] bf16.

    numpy backend -> uint16 bit patterns; torch backend -> bf16 tensors on
    ``device``.  dO ~ N(0,1) everywhere (reading c18)."""
    shape = (cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh)
    if device is None:
        if cfg.projected:
            out = _projected_np(cfg, layer, axis, ("Q", "K", "V"))
        else:
            out = {"Q": _normal_np(cfg, layer, axis, "Q", shape, cfg.q_scale),
                   "K": _normal_np(cfg, layer, axis, "K", shape),
                   "V": _normal_np(cfg, layer, axis, "V", shape)}
        out["dO"] = _normal_np(cfg, layer, axis, "dO", shape)
        return out
    if cfg.projected:
        out = _projected_torch(cfg, layer, axis, ("Q", "K", "V"), device, x_cache)
    else:
        out = {"Q": _normal_torch(cfg, layer, axis, "Q", shape, device, cfg.q_scale),
               "K": _normal_torch(cfg, layer, axis, "K", shape, device),
               "V": _normal_torch(cfg, layer, axis, "V", shape, device)}
    out["dO"] = _normal_torch(cfg, layer, axis, "dO", shape, device)
    return out


def make_layer_inputs(cfg: TabShape, layer: int = 0, device=None, x_cache=None):
    """Inputs of one layer: {"feature": {...}, "item": {...}}."""
    return {axis: make_call_inputs(cfg, axis, layer, device, x_cache)
            for axis in ("feature", "item")}
