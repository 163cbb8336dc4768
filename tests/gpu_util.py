"""Helpers for the -m gpu parity tests: run libtabattn through its C ABI (via the ctypes binding)
and compare against the fp64 oracle element by element (SURVEY.md §8(c) "Comparison rule")."""
import numpy as np
import torch

import paper_2606_03681_b200 as tab
from oracle import ref
from workloads import bf16_bits_to_f64

from helpers import FWD_REL_L2, FWD_MAXABS_FRAC, GRAD_REL_L2, LSE_TOL, rel_l2, check_grad_hard


def to_dev(bits):
    """uint16 bf16 bit patterns -> CUDA bfloat16 tensor (bit copy)."""
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)


def to_bits(t):
    """CUDA bfloat16 tensor -> uint16 bit patterns on the host (bit copy)."""
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def to_f64(t):
    return bf16_bits_to_f64(to_bits(t))


def is_pos_zero(bits):
    return np.all(bits == 0)


def run_gpu(axis, inp, n_train=None, col_valid=None, scale=0.0):
    """inp: dict of uint16 arrays Q,K,V,dO.  Returns dict of GPU results (torch tensors)."""
    d = {k: to_dev(v) for k, v in inp.items()}
    cv = torch.from_numpy(np.ascontiguousarray(col_valid, dtype=np.uint8)).cuda() if col_valid is not None else None
    if axis == "feature":
        O, LSE = tab.tabattn_feature_fwd(d["Q"], d["K"], d["V"], cv, scale)
        dQ, dK, dV = tab.tabattn_feature_bwd(d["Q"], d["K"], d["V"], O, d["dO"], LSE, cv, scale)
    else:
        nt = torch.from_numpy(np.ascontiguousarray(n_train, dtype=np.int32)).cuda()
        O, LSE = tab.tabattn_item_fwd(d["Q"], d["K"], d["V"], nt, cv, scale, n_train_host=n_train)
        dQ, dK, dV = tab.tabattn_item_bwd(d["Q"], d["K"], d["V"], O, d["dO"], LSE, nt, cv, scale,
                                          n_train_host=n_train)
    torch.cuda.synchronize()
    return dict(O=O, LSE=LSE, dQ=dQ, dK=dK, dV=dV)


def run_oracle(axis, inp, n_train=None, col_valid=None, scale=0.0):
    if axis == "feature":
        O, LSE = ref.feature_fwd(inp["Q"], inp["K"], inp["V"], col_valid, scale)
        dQ, dK, dV = ref.feature_bwd(inp["Q"], inp["K"], inp["V"], inp["dO"], col_valid, scale)
    else:
        O, LSE = ref.item_fwd(inp["Q"], inp["K"], inp["V"], n_train, col_valid, scale)
        dQ, dK, dV = ref.item_bwd(inp["Q"], inp["K"], inp["V"], inp["dO"], n_train, col_valid, scale)
    return dict(O=O, LSE=LSE, dQ=dQ, dK=dK, dV=dV)


def valid_mask_cells(shape5, axis, n_train, col_valid):
    """Boolean [B,R,C] masks: where outputs are defined (valid columns) and where dK/dV are
    defined non-zero (valid column and, for item attention, row < n_train)."""
    B, R, C = shape5[:3]
    colv = np.ones((B, C), bool) if col_valid is None else np.asarray(col_valid).astype(bool)
    cell = np.broadcast_to(colv[:, None, :], (B, R, C)).copy()
    key = cell.copy()
    if axis == "item":
        rows = np.arange(R)[None, :, None] < np.asarray(n_train)[:, None, None]
        key &= rows
    return cell, key


def check_parity(axis, inp, gpu, orc, n_train=None, col_valid=None, what=""):
    """The bar of BASELINE.json: O rel-L2 <= 5e-3, max|dO| <= 1e-2 max|V|; dQ/dK/dV rel-L2 <= 1e-2
    over valid positions; masked positions bit-exact +0; LSE within LSE_TOL."""
    shape5 = inp["Q"].shape
    cell, key = valid_mask_cells(shape5, axis, n_train, col_valid)
    # max|V| over the positions that can influence an output (masked V may be NaN-poisoned)
    v_abs = np.abs(bf16_bits_to_f64(inp["V"]))[key]
    vmax = v_abs.max() if v_abs.size else 0.0
    out = {}
    for name, mask in (("O", cell), ("dQ", cell), ("dK", key), ("dV", key)):
        bits = to_bits(gpu[name])
        g = bf16_bits_to_f64(bits)
        r = orc[name]
        assert is_pos_zero(bits[~mask]), "%s %s: masked positions are not +0" % (what, name)
        assert np.all(r[~mask] == 0.0)
        assert np.isfinite(g).all(), "%s %s: non-finite values" % (what, name)
        e = rel_l2(g[mask], r[mask])
        out[name] = e
        tol = FWD_REL_L2 if name == "O" else GRAD_REL_L2
        assert e <= tol, "%s %s rel-L2 %.3e > %.1e" % (what, name, e, tol)
        if name == "O":
            mx = np.abs(g[mask] - r[mask]).max() if mask.any() else 0.0
            assert mx <= FWD_MAXABS_FRAC * vmax, "%s O max-abs %.3e" % (what, mx)
        else:
            # per-sequence and per-element gates: feature sequences run along C (axis 2), item along R (axis 1)
            check_grad_hard(name, g, r, 2 if axis == "feature" else 1, what)
    lse_g = gpu["LSE"].cpu().numpy().astype(np.float64)
    lse_r = orc["LSE"]
    if axis == "feature":      # [B,R,H,C]
        m = np.broadcast_to(cell[:, :, None, :], lse_r.shape)
    else:                      # [B,C,H,R]
        m = np.broadcast_to(cell.transpose(0, 2, 1)[:, :, None, :], lse_r.shape)
    assert np.all(lse_g[~m] == 0.0), "%s LSE at invalid columns must be 0" % what
    if m.any():
        err = np.abs(lse_g[m] - lse_r[m]).max()
        out["LSE"] = err
        assert err <= LSE_TOL * max(1.0, np.abs(lse_r[m]).max()), "%s LSE err %.3e" % (what, err)
    return out
