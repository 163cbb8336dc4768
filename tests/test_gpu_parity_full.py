"""GPU-vs-oracle parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(SURVEY.md §4 tier T2, §8(d) "CPU baseline beside it": the sampling rule).  Needs a B200.

The whole config runs on the GPU through the C ABI exactly as in bench.py (device-generated seeded
inputs, preallocated LayerBuffers).  The fp64 oracle then computes a seeded SAMPLE of whole
sequences from the same bits -- for item attention every table's first and last valid column (the
last one is the target column) plus one random valid column; for feature attention every table's
rows {0, n_b-1, n_b, R-1} plus random rows -- and those are compared element by element with the
BASELINE.json tolerances.  Over the FULL outputs the test checks what holds at any size: all values
finite, and every position the ABI defines as zero is bit-exact +0.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from workloads import get_config, draw_structure, make_call_inputs, bf16_bits_to_f64  # noqa: E402
from helpers import FWD_REL_L2, FWD_MAXABS_FRAC, GRAD_REL_L2, LSE_TOL, rel_l2, check_grad_hard  # noqa: E402

# (config, layer): ragged is checked on the first and the last of its 12 layers (own seeded projections each)
FULL = [("base", 0), ("feature_heavy", 0), ("long_item", 0), ("ragged", 0), ("ragged", 11)]
N_RANDOM_ROWS = 24


def _bits(t):
    import torch
    return t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def _sample_cols(cfg, col_valid, rng):
    cols = []
    for b in range(cfg.B):
        valid = np.arange(cfg.C) if col_valid is None else np.flatnonzero(col_valid[b])
        pick = {int(valid[0]), int(valid[-1]), int(rng.choice(valid))}
        cols += [(b, c) for c in sorted(pick)]
    return cols


def _sample_rows(cfg, n_train, rng):
    rows = []
    for b in range(cfg.B):
        n = int(n_train[b])
        pick = {0, n - 1, min(n, cfg.R - 1), cfg.R - 1}
        pick |= set(int(r) for r in rng.integers(0, cfg.R, size=N_RANDOM_ROWS // 4))
        rows += [(b, r) for r in sorted(pick)]
    return rows


def _check(name, g, r, tol, what):
    assert np.isfinite(g).all(), "%s %s: non-finite" % (what, name)
    e = rel_l2(g, r)
    assert e <= tol, "%s %s rel-L2 %.3e > %.1e" % (what, name, e, tol)
    return e


def _poison(torch, L, n_train_h, col_valid):
    """NaN at every position that must not influence an output (SURVEY.md §8(b) "Values at masked
    positions"): all inputs at invalid columns; item K/V at rows >= n_train[b]."""
    nan = float("nan")
    for ax in ("feature", "item"):
        if col_valid is not None:
            bad = (col_valid == 0)[:, None, :, None, None]
            for k in ("Q", "K", "V", "dO"):
                L[ax][k].masked_fill_(bad, nan)
    for b, n in enumerate(n_train_h):
        L["item"]["K"][b, int(n):] = nan
        L["item"]["V"][b, int(n):] = nan


@pytest.mark.parametrize("name,layer", FULL, ids=["%s-L%d" % f for f in FULL])
def test_full_size_sampled_parity(name, layer):
    import torch
    import paper_2606_03681_b200 as tab
    from oracle import ref

    cfg = get_config(name)
    dev = torch.device("cuda", 0)
    n_train_h, col_valid_h = draw_structure(cfg)
    n_train = torch.from_numpy(n_train_h).to(dev)
    col_valid = torch.from_numpy(col_valid_h).to(dev) if col_valid_h is not None else None
    L = {ax: make_call_inputs(cfg, ax, layer, device=dev) for ax in ("feature", "item")}
    _poison(torch, L, n_train_h, col_valid)
    buf = tab.LayerBuffers(cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh, device=dev)
    tab.layer_fwd_bwd(L["feature"], L["item"], n_train, col_valid, buf, n_train_h)
    torch.cuda.synchronize()

    rng = np.random.default_rng(9000 + cfg.seed)
    colv = np.ones((cfg.B, cfg.C), bool) if col_valid_h is None else col_valid_h.astype(bool)
    rows_lt_n = np.arange(cfg.R)[None, :] < n_train_h[:, None]          # [B,R]

    for axis, outs, lse in (("feature", (buf.O_f,) + buf.grads_f, buf.LSE_f),
                            ("item", (buf.O_i,) + buf.grads_i, buf.LSE_i)):
        inp = {k: _bits(v) for k, v in L[axis].items()}
        got = {k: _bits(t) for k, t in zip(("O", "dQ", "dK", "dV"), outs)}
        lse_g = lse.cpu().numpy().astype(np.float64)
        what = "%s/%s(full)" % (name, axis)
        # ---- properties over the full outputs ----------------------------------------------------
        for k, bits in got.items():
            assert not np.any((bits & 0x7F80) == 0x7F80), "%s %s: non-finite values" % (what, k)
            dead = np.broadcast_to(~colv[:, None, :], bits.shape[:3])
            assert np.all(bits[dead] == 0), "%s %s: invalid columns are not +0" % (what, k)
        if axis == "item":
            for k in ("dK", "dV"):
                dead = np.broadcast_to(~rows_lt_n[:, :, None], got[k].shape[:3])
                assert np.all(got[k][dead] == 0), "%s %s: rows >= n_train are not +0" % (what, k)
            assert np.all(lse_g[np.broadcast_to(~colv[:, :, None, None], lse_g.shape)] == 0.0)
        else:
            assert np.all(lse_g[np.broadcast_to(~colv[:, None, None, :], lse_g.shape)] == 0.0)
        # ---- sampled whole sequences against the oracle ------------------------------------------
        if axis == "item":
            sel = _sample_cols(cfg, col_valid_h, rng)
            O, LSE = ref.item_fwd(inp["Q"], inp["K"], inp["V"], n_train_h, col_valid_h, cols=sel)
            dQ, dK, dV = ref.item_bwd(inp["Q"], inp["K"], inp["V"], inp["dO"], n_train_h, col_valid_h, cols=sel)
            bs = np.array([b for b, _ in sel]); cs = np.array([c for _, c in sel])
            g = {k: bf16_bits_to_f64(v[bs, :, cs]) for k, v in got.items()}            # [n_sel,R,H,dh]
            lg = lse_g[bs, cs]                                                          # [n_sel,H,R]
            vmax = max(np.abs(bf16_bits_to_f64(inp["V"][b, :n_train_h[b], c])).max() for b, c in sel)
        else:
            sel = _sample_rows(cfg, n_train_h, rng)
            O, LSE = ref.feature_fwd(inp["Q"], inp["K"], inp["V"], col_valid_h, rows=sel)
            dQ, dK, dV = ref.feature_bwd(inp["Q"], inp["K"], inp["V"], inp["dO"], col_valid_h, rows=sel)
            bs = np.array([b for b, _ in sel]); rs = np.array([r for _, r in sel])
            g = {k: bf16_bits_to_f64(v[bs, rs]) for k, v in got.items()}                # [n_sel,C,H,dh]
            lg = lse_g[bs, rs]                                                          # [n_sel,H,C]
            vmax = max(np.abs(bf16_bits_to_f64(inp["V"][b, r][colv[b]])).max() for b, r in sel)
        err = {"O": _check("O", g["O"], O, FWD_REL_L2, what)}
        for k, r in (("dQ", dQ), ("dK", dK), ("dV", dV)):
            err[k] = _check(k, g[k], r, GRAD_REL_L2, what)
            check_grad_hard(k, g[k], r, 1, what)     # compact layout [n_sel, seq, H, dh]: the sequence is axis 1
        mx = np.abs(g["O"] - O).max()
        assert mx <= FWD_MAXABS_FRAC * vmax, "%s O max-abs %.3e > 1e-2 * %.3f" % (what, mx, vmax)
        lerr = np.abs(lg - LSE).max()
        assert lerr <= LSE_TOL * max(1.0, np.abs(LSE).max()), "%s LSE err %.3e" % (what, lerr)
        print("%s: %d sampled sequences  " % (what, len(sel)) + " ".join("%s=%.2e" % kv for kv in err.items())
              + " LSE=%.2e" % lerr)
        del inp, got
