"""GPU-vs-oracle parity of the sub-blocks around the attention kernels through the
C ABI: attention sub-block and MLP sub-block fwd+bwd, batched Newton-Schulz.  Needs a B200.

Tolerances: every activation between two kernels is stored as bf16 (2^-9 relative per element,
rel-L2 ~1.1e-3 per rounding); a forward output sits behind 4-5 such roundings on the branch (not on the residual
path), a gradient behind 8-10, and the attention kernels' own error (<= 5e-3 / 1e-2) enters the attention
sub-block.  Bars: forward y rel-L2 <= 5e-3 (the residual term is exact), branch-only rel-L2 <= 1e-2; dx <= 1e-2
(residual dy exact) and the parameter gradients (fp32, summed over all cells) <= 1.5e-2; Newton-Schulz against the
oracle with the same bf16 storage points <= 2e-2, against exact fp64 <= 5e-2."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from workloads import f32_to_bf16_bits, bf16_bits_to_f64, TabShape, draw_structure  # noqa: E402
from helpers import rel_l2  # noqa: E402

Y_TOL, BRANCH_TOL, DX_TOL, DW_TOL = 5e-3, 1e-2, 1e-2, 1.5e-2


def _bits(rng, shape, scale=1.0, shift=0.0):
    return f32_to_bf16_bits((rng.standard_normal(shape) * scale + shift).astype(np.float32))


def _dev(bits):
    import gpu_util as gu
    return gu.to_dev(bits)


def _f64(t):
    import gpu_util as gu
    return gu.to_f64(t)


MLP_CASES = [
    # cells, e, hidden, alpha
    (300, 64, 128, 1.0),          # ragged last tile (300 = 2 * 128 + 44)
    (1000, 192, 768, 0.95 ** 2),  # the baseline width
    (777, 256, 768, 1.0),         # the record width
    (20000, 256, 768, 1.0),       # 157 row tiles: every persistent GEMM CTA walks several (148 CTAs per column tile)
]


@pytest.mark.parametrize("case", MLP_CASES, ids=["e64", "e192", "e256", "e256_multi_tile"])
def test_mlp_block_parity(case):
    import torch
    import paper_2606_03681_b200 as tab
    from oracle import block_ref as br
    cells, e, hid, alpha = case
    rng = np.random.default_rng(100 + e)
    x, g, dy = _bits(rng, (cells, e)), _bits(rng, (e,), 0.1, 1.0), _bits(rng, (cells, e))
    W1, W2 = _bits(rng, (hid, e), e ** -0.5), _bits(rng, (e, hid), hid ** -0.5)
    dx_, dg_, dW1_, dW2_ = br.mlp_bwd(x, g, W1, W2, dy, alpha)
    y_ = br.mlp_fwd(x, g, W1, W2, alpha)
    tx, tg, t1, t2, tdy = (_dev(a) for a in (x, g, W1, W2, dy))
    y, saved = tab.tabattn_mlp_fwd(tx, tg, t1, t2, alpha)
    dx, dg, dW1, dW2 = tab.tabattn_mlp_bwd(tx, tg, t1, t2, saved, tdy, alpha)
    torch.cuda.synchronize()
    xs = alpha * bf16_bits_to_f64(x)
    yg = _f64(y)
    assert np.isfinite(yg).all()
    assert rel_l2(yg, y_) <= Y_TOL
    assert rel_l2(yg - xs, y_ - xs) <= BRANCH_TOL + 4e-3   # (the bf16 rounding of y itself is relative to |y|, not |branch|)
    assert rel_l2(_f64(dx), dx_) <= DX_TOL
    for got, want, nm in ((dg, dg_, "dg"), (dW1, dW1_, "dW1"), (dW2, dW2_, "dW2")):
        gv = got.double().cpu().numpy()
        assert np.isfinite(gv).all()
        assert rel_l2(gv, want) <= DW_TOL, "%s rel-L2 %.3e" % (nm, rel_l2(gv, want))
    # bitwise reproducible (fixed-order reductions, no atomics)
    y2, saved2 = tab.tabattn_mlp_fwd(tx, tg, t1, t2, alpha)
    r2 = tab.tabattn_mlp_bwd(tx, tg, t1, t2, saved2, tdy, alpha)
    torch.cuda.synchronize()
    assert torch.equal(y, y2) and all(torch.equal(a, b) for a, b in zip((dx, dg, dW1, dW2), r2))


ATTN_CASES = [
    # name, B, R, C, H, dh, n_train, mask, alpha
    ("e64", 2, 70, 5, 2, 32, 40, "none", 1.0),
    ("e192_masked", 2, 150, 12, 6, 32, 100, "prefix", 0.95),
    ("e256", 1, 300, 6, 4, 64, 200, "none", 0.95 ** 4),
    ("e128", 1, 130, 3, 4, 32, 90, "none", 1.0),   # dWqkv in one launch, one 128-row tile per gradient tensor
]


@pytest.mark.parametrize("axis", [0, 1], ids=["feature", "item"])
@pytest.mark.parametrize("case", ATTN_CASES, ids=[c[0] for c in ATTN_CASES])
def test_attention_block_parity(case, axis):
    import torch
    import paper_2606_03681_b200 as tab
    from oracle import block_ref as br
    name, B, R, C, H, dh, n, mask, alpha = case
    e = H * dh
    vf = None if mask == "none" else (max(1, (C - 1) // 3), C - 1)
    cfg = TabShape(name, 60 + len(name), B=B, R=R, C=C, H=H, dh=dh, n_train=n, mask=mask, valid_features=vf)
    n_train, col_valid = draw_structure(cfg)
    rng = np.random.default_rng(200 + e + axis)
    x, g, dy = _bits(rng, (B, R, C, e)), _bits(rng, (e,), 0.1, 1.0), _bits(rng, (B, R, C, e))
    Wqkv, Wo = _bits(rng, (3 * e, e), e ** -0.5), _bits(rng, (e, e), e ** -0.5)
    ax = "feature" if axis == 0 else "item"
    y_ = br.attn_block_fwd(ax, x, g, Wqkv, Wo, H, n_train, col_valid, alpha)
    dx_, dg_, dWqkv_, dWo_ = br.attn_block_bwd(ax, x, g, Wqkv, Wo, dy, H, n_train, col_valid, alpha)
    tx, tg, tq, to, tdy = (_dev(a) for a in (x, g, Wqkv, Wo, dy))
    nt = torch.from_numpy(n_train).cuda()
    cv = torch.from_numpy(np.ascontiguousarray(col_valid, dtype=np.uint8)).cuda() if col_valid is not None else None
    y, saved = tab.tabattn_attn_block_fwd(axis, tx, tg, tq, to, H, nt, cv, alpha, n_train_host=n_train)
    dx, dg, dWqkv, dWo = tab.tabattn_attn_block_bwd(axis, tx, tg, tq, to, H, saved, tdy, nt, cv, alpha,
                                                    n_train_host=n_train)
    torch.cuda.synchronize()
    xs = alpha * bf16_bits_to_f64(x)
    yg, dxg = _f64(y), _f64(dx)
    assert np.isfinite(yg).all() and np.isfinite(dxg).all()
    assert rel_l2(yg, y_) <= Y_TOL
    assert rel_l2(yg - xs, y_ - xs) <= BRANCH_TOL + 4e-3
    assert rel_l2(dxg, dx_) <= DX_TOL
    if col_valid is not None:
        # invalid columns: only the residual path (y = alpha x, dx = alpha dy, each rounded to bf16 once)
        bad = np.broadcast_to(~np.asarray(col_valid).astype(bool)[:, None, :], (B, R, C))
        assert np.abs(yg[bad] - xs[bad]).max() <= 2.0 ** -8 * np.abs(xs).max()
        assert np.abs(dxg[bad] - alpha * bf16_bits_to_f64(dy)[bad]).max() <= 2.0 ** -8 * np.abs(bf16_bits_to_f64(dy)).max()
    for got, want, nm in ((dg, dg_, "dg"), (dWqkv, dWqkv_, "dWqkv"), (dWo, dWo_, "dWo")):
        gv = got.double().cpu().numpy()
        assert np.isfinite(gv).all()
        assert rel_l2(gv, want) <= DW_TOL, "%s rel-L2 %.3e" % (nm, rel_l2(gv, want))


NS_CASES = [(3, 192, 192), (2, 256, 256), (4, 64, 200), (1, 192, 576)]


@pytest.mark.parametrize("case", NS_CASES, ids=["%dx%dx%d" % c for c in NS_CASES])
def test_newton_schulz_parity(case):
    import torch
    import paper_2606_03681_b200 as tab
    from oracle import block_ref as br
    nb, m, n = case
    rng = np.random.default_rng(300 + m + n)
    G = _bits(rng, (nb, m, n), 0.02)       # gradient-like scale; the iteration normalises it
    rt = lambda z: bf16_bits_to_f64(f32_to_bf16_bits(z.astype(np.float32)))
    X_same = br.newton_schulz(G, 5, round_fn=rt)     # the algorithm with Muon's bf16 storage of the iterates
    X_exact = br.newton_schulz(G, 5)
    X = tab.tabattn_newton_schulz(_dev(G), 5)
    torch.cuda.synchronize()
    Xg = _f64(X)
    assert np.isfinite(Xg).all()
    assert rel_l2(Xg, X_same) <= 2e-2, "vs bf16-storage oracle %.3e" % rel_l2(Xg, X_same)
    assert rel_l2(Xg, X_exact) <= 5e-2, "vs exact oracle %.3e" % rel_l2(Xg, X_exact)
    # what the method is for: the result is close to orthogonal (singular values in the quintic's band)
    S = np.linalg.svd(Xg[0], compute_uv=False)
    assert S.max() < 1.25 and np.median(S) > 0.5
    # zero steps = the Frobenius-normalised input
    X0 = _f64(tab.tabattn_newton_schulz(_dev(G), 0))
    assert rel_l2(X0, br.newton_schulz(G, 0)) <= 3e-3


# ---- at the size bench.py times (the long_item table: 688,128 cells, e = 256, hidden = 768) -------------------------
def _full_inputs(torch, dev, B, R, C, e, hid, seed):
    g = torch.Generator(device=dev)
    g.manual_seed(seed)
    rnd = lambda *s, scale=1.0: (torch.randn(*s, generator=g, device=dev, dtype=torch.float32) * scale).to(torch.bfloat16)
    x, dy = rnd(B, R, C, e), rnd(B, R, C, e)
    gain = (1 + 0.1 * torch.randn(e, generator=g, device=dev)).to(torch.bfloat16)
    return x, dy, gain, rnd(3 * e, e, scale=e ** -0.5), rnd(e, e, scale=e ** -0.5), rnd(hid, e, scale=e ** -0.5), \
        rnd(e, hid, scale=hid ** -0.5)


def _np_bits(t):
    import gpu_util as gu
    return gu.to_bits(t)


def test_mlp_block_full_size():
    """All 688,128 cells: y and dx on a seeded sample of cells (the block is per-cell), the parameter gradients
    (sums over ALL cells) against the oracle's full reduction."""
    import torch
    import paper_2606_03681_b200 as tab
    from oracle import block_ref as br
    dev = torch.device("cuda", 0)
    B, R, C, e, hid, alpha = 8, 4096, 21, 256, 768, 0.95
    x, dy, gain, _, _, W1, W2 = _full_inputs(torch, dev, B, R, C, e, hid, 77)
    y, saved = tab.tabattn_mlp_fwd(x, gain, W1, W2, alpha)
    dx, dg, dW1, dW2 = tab.tabattn_mlp_bwd(x, gain, W1, W2, saved, dy, alpha)
    torch.cuda.synchronize()
    for t in (y, dx, dg, dW1, dW2):
        assert bool(torch.isfinite(t.float()).all())
    xb, dyb = _np_bits(x).reshape(-1, e), _np_bits(dy).reshape(-1, e)
    gb, w1, w2 = _np_bits(gain), _np_bits(W1), _np_bits(W2)
    dx_, dg_, dW1_, dW2_ = br.mlp_bwd(xb, gb, w1, w2, dyb, alpha)       # the full reduction (numpy fp64 matmuls)
    y_ = br.mlp_fwd(xb, gb, w1, w2, alpha)
    assert rel_l2(_f64(y).reshape(-1, e), y_) <= Y_TOL
    assert rel_l2(_f64(dx).reshape(-1, e), dx_) <= DX_TOL
    # per-cell gate on a sample (a wrong tile would hide in the global norm): first / last cells and random ones
    rng = np.random.default_rng(5)
    idx = np.unique(np.concatenate([[0, 127, 128, xb.shape[0] - 1], rng.integers(0, xb.shape[0], 4096)]))
    err = np.linalg.norm(_f64(y).reshape(-1, e)[idx] - y_[idx], axis=1) / np.linalg.norm(y_[idx], axis=1)
    assert err.max() <= 4 * Y_TOL
    for got, want, nm in ((dg, dg_, "dg"), (dW1, dW1_, "dW1"), (dW2, dW2_, "dW2")):
        assert rel_l2(got.double().cpu().numpy(), want) <= DW_TOL, nm


@pytest.mark.parametrize("axis", [0, 1], ids=["feature", "item"])
def test_attention_block_full_size(axis):
    """The long_item table through the attention sub-block.  Feature axis: everything, including the parameter
    gradients, against the oracle on the whole tensor.  Item axis (43 TFLOP in fp64): y and dx of a seeded sample
    of whole (b, c) sequences -- the block is per-sequence -- and finiteness of everything."""
    import torch
    import paper_2606_03681_b200 as tab
    from oracle import block_ref as br
    dev = torch.device("cuda", 0)
    B, R, C, H, dh, n, alpha = 8, 4096, 21, 4, 64, 3072, 0.95
    e = H * dh
    x, dy, gain, Wqkv, Wo, _, _ = _full_inputs(torch, dev, B, R, C, e, 768, 78 + axis)
    n_train = np.full(B, n, np.int32)
    nt = torch.from_numpy(n_train).to(dev)
    y, saved = tab.tabattn_attn_block_fwd(axis, x, gain, Wqkv, Wo, H, nt, None, alpha, n_train_host=n_train)
    dx, dg, dWqkv, dWo = tab.tabattn_attn_block_bwd(axis, x, gain, Wqkv, Wo, H, saved, dy, nt, None, alpha,
                                                    n_train_host=n_train)
    torch.cuda.synchronize()
    for t in (y, dx, dg, dWqkv, dWo):
        assert bool(torch.isfinite(t.float()).all())
    xb, dyb = _np_bits(x), _np_bits(dy)
    gb, wq, wo = _np_bits(gain), _np_bits(Wqkv), _np_bits(Wo)
    if axis == 0:
        y_ = br.attn_block_fwd("feature", xb, gb, wq, wo, H, n_train, None, alpha)
        dx_, dg_, dWqkv_, dWo_ = br.attn_block_bwd("feature", xb, gb, wq, wo, dyb, H, n_train, None, alpha)
        assert rel_l2(_f64(y), y_) <= Y_TOL and rel_l2(_f64(dx), dx_) <= DX_TOL
        for got, want, nm in ((dg, dg_, "dg"), (dWqkv, dWqkv_, "dWqkv"), (dWo, dWo_, "dWo")):
            assert rel_l2(got.double().cpu().numpy(), want) <= DW_TOL, nm
    else:
        rng = np.random.default_rng(6)
        yg, dxg = _f64(y), _f64(dx)
        for b, c in [(0, 0), (B - 1, C - 1), (int(rng.integers(B)), int(rng.integers(C)))]:
            sl = (slice(b, b + 1), slice(None), slice(c, c + 1))
            y_ = br.attn_block_fwd("item", xb[sl], gb, wq, wo, H, n_train[b:b + 1], None, alpha)
            dx_ = br.attn_block_bwd("item", xb[sl], gb, wq, wo, dyb[sl], H, n_train[b:b + 1], None, alpha)[0]
            assert rel_l2(yg[sl], y_) <= Y_TOL, (b, c)
            assert rel_l2(dxg[sl], dx_) <= DX_TOL, (b, c)
