"""Pins of the sub-block oracle (oracle/block_ref.py) against things other than
itself: torch-CPU fp64 autograd on an independently written formulation (library rms_norm / linear / gelu /
scaled_dot_product_attention), central finite differences, closed forms, and the SVD identity of Newton-Schulz."""
import numpy as np
import pytest
import torch
import torch.nn.functional as F

from oracle import block_ref as br


def _r(rng, *s, scale=1.0):
    return rng.standard_normal(s) * scale


def _t(a, grad=True):
    return torch.tensor(a, dtype=torch.float64, requires_grad=grad)


# ---- MLP ------------------------------------------------------------------------------------------------
def _torch_mlp(x, g, W1, W2, alpha, eps):
    xs = alpha * x
    h = F.rms_norm(xs, (xs.shape[-1],), g, eps)
    return xs + F.linear(F.gelu(F.linear(h, W1)), W2)


@pytest.mark.parametrize("alpha", [1.0, 0.95 ** 3])
def test_mlp_matches_torch_autograd(alpha):
    rng = np.random.default_rng(1)
    M, e, hid, eps = 37, 16, 40, 1e-6
    x, g, W1, W2, dy = _r(rng, M, e), 1 + 0.1 * _r(rng, e), _r(rng, hid, e, scale=e ** -0.5), \
        _r(rng, e, hid, scale=hid ** -0.5), _r(rng, M, e)
    tx, tg, t1, t2 = _t(x), _t(g), _t(W1), _t(W2)
    ty = _torch_mlp(tx, tg, t1, t2, alpha, eps)
    ty.backward(_t(dy, False))
    np.testing.assert_allclose(br.mlp_fwd(x, g, W1, W2, alpha, eps), ty.detach().numpy(), atol=1e-12)
    dx, dg, dW1, dW2 = br.mlp_bwd(x, g, W1, W2, dy, alpha, eps)
    for got, want in ((dx, tx.grad), (dg, tg.grad), (dW1, t1.grad), (dW2, t2.grad)):
        np.testing.assert_allclose(got, want.numpy(), atol=1e-11)


def test_mlp_finite_differences_and_closed_forms():
    rng = np.random.default_rng(2)
    M, e, hid = 5, 8, 12
    x, g, W1, W2, dy = _r(rng, M, e), 1 + 0.1 * _r(rng, e), _r(rng, hid, e, scale=0.4), _r(rng, e, hid, scale=0.3), \
        _r(rng, M, e)
    dx, dg, dW1, dW2 = br.mlp_bwd(x, g, W1, W2, dy, 0.9, 1e-6)
    L = lambda x_, g_, a_, b_: float((br.mlp_fwd(x_, g_, a_, b_, 0.9, 1e-6) * dy).sum())
    hstep = 1e-6
    for arr, grad, idx in ((x, dx, (2, 3)), (g, dg, (5,)), (W1, dW1, (7, 1)), (W2, dW2, (4, 9))):
        ap, am = arr.copy(), arr.copy()
        ap[idx] += hstep
        am[idx] -= hstep
        args_p = [ap if a is arr else a for a in (x, g, W1, W2)]
        args_m = [am if a is arr else a for a in (x, g, W1, W2)]
        fd = (L(*args_p) - L(*args_m)) / (2 * hstep)
        assert fd == pytest.approx(grad[idx], abs=1e-7 * max(1.0, abs(grad[idx])))
    # W2 = 0: the block is the (scaled) identity; its input gradient is alpha dy
    y = br.mlp_fwd(x, g, W1, np.zeros_like(W2), 0.9)
    np.testing.assert_allclose(y, 0.9 * x, atol=1e-15)
    dx0 = br.mlp_bwd(x, g, W1, np.zeros_like(W2), dy, 0.9)[0]
    np.testing.assert_allclose(dx0, 0.9 * dy, atol=1e-15)
    # RMSNorm: unit gain -> rows of h have mean square 1 (eps -> 0); scale invariance in x
    h, _ = br.rmsnorm_fwd(x, np.ones(e), 0.0)
    np.testing.assert_allclose((h * h).mean(-1), 1.0, atol=1e-14)
    np.testing.assert_allclose(br.rmsnorm_fwd(7.0 * x, g, 0.0)[0], br.rmsnorm_fwd(x, g, 0.0)[0], atol=1e-13)
    # GELU closed values: gelu(0) = 0, gelu'(0) = 1/2, gelu(x) - gelu(-x) = x
    assert br.gelu(np.array(0.0)) == 0.0 and br.gelu_grad(np.array(0.0)) == 0.5
    z = np.linspace(-4, 4, 9)
    np.testing.assert_allclose(br.gelu(z) - br.gelu(-z), z, atol=1e-15)


# ---- attention sub-block -----------------------------------------------------------------------------------
def _torch_attn_block(axis, x, g, Wqkv, Wo, H, n_train, col_valid, alpha, eps):
    B, R, C, e = x.shape
    dh = e // H
    xs = alpha * x
    h = F.rms_norm(xs, (e,), g, eps)
    q, k, v = F.linear(h, Wqkv).split(e, dim=-1)
    out = torch.zeros_like(xs)
    for b in range(B):
        cols = [c for c in range(C) if col_valid is None or col_valid[b][c]]
        if not cols:
            continue
        sel = lambda t: t[b][:, cols].reshape(R, len(cols), H, dh)
        qb, kb, vb = sel(q), sel(k), sel(v)
        if axis == "feature":   # sequences along the columns: [R, H, Cv, dh]
            ob = F.scaled_dot_product_attention(qb.permute(0, 2, 1, 3), kb.permute(0, 2, 1, 3), vb.permute(0, 2, 1, 3))
            ob = ob.permute(0, 2, 1, 3)
        else:                   # sequences along the rows, keys = train rows: [Cv, H, R, dh]
            n = int(n_train[b])
            ob = F.scaled_dot_product_attention(qb.permute(1, 2, 0, 3), kb[:n].permute(1, 2, 0, 3),
                                                vb[:n].permute(1, 2, 0, 3))
            ob = ob.permute(2, 0, 1, 3)
        ob = ob.reshape(R, len(cols), e)
        full = torch.zeros(R, C, e, dtype=xs.dtype)
        full[:, cols] = ob
        out[b] = full
    return xs + F.linear(out, Wo)


@pytest.mark.parametrize("axis", ["feature", "item"])
@pytest.mark.parametrize("masked", [False, True])
def test_attn_block_matches_torch_autograd(axis, masked):
    rng = np.random.default_rng(3)
    B, R, C, H, dh, eps, alpha = 2, 9, 5, 2, 4, 1e-6, 0.95
    e = H * dh
    x, g, dy = _r(rng, B, R, C, e), 1 + 0.1 * _r(rng, e), _r(rng, B, R, C, e)
    Wqkv, Wo = _r(rng, 3 * e, e, scale=e ** -0.5), _r(rng, e, e, scale=e ** -0.5)
    nt = np.array([6, 9], np.int32)
    cv = np.array([[1, 0, 1, 1, 1], [1, 1, 0, 0, 1]], np.uint8) if masked else None
    tx, tg, tq, to = _t(x), _t(g), _t(Wqkv), _t(Wo)
    ty = _torch_attn_block(axis, tx, tg, tq, to, H, nt, cv, alpha, eps)
    ty.backward(_t(dy, False))
    y = br.attn_block_fwd(axis, x, g, Wqkv, Wo, H, nt, cv, alpha, eps)
    np.testing.assert_allclose(y, ty.detach().numpy(), atol=1e-12)
    dx, dg, dWqkv, dWo = br.attn_block_bwd(axis, x, g, Wqkv, Wo, dy, H, nt, cv, alpha, eps)
    for got, want in ((dx, tx.grad), (dg, tg.grad), (dWqkv, tq.grad), (dWo, to.grad)):
        np.testing.assert_allclose(got, want.numpy(), atol=1e-11)
    if masked:
        # invalid columns pass through the residual only: y = alpha x, dx = alpha dy there
        bad = ~cv.astype(bool)
        np.testing.assert_allclose(y[bad[:, None, :].repeat(R, 1)], alpha * x[bad[:, None, :].repeat(R, 1)], atol=1e-15)
        np.testing.assert_allclose(dx[bad[:, None, :].repeat(R, 1)], alpha * dy[bad[:, None, :].repeat(R, 1)], atol=1e-15)


def test_attn_block_zero_out_projection_is_identity():
    rng = np.random.default_rng(4)
    x = _r(rng, 1, 4, 3, 8)
    y = br.attn_block_fwd("item", x, np.ones(8), _r(rng, 24, 8), np.zeros((8, 8)), 2, np.array([3], np.int32), None, 0.5)
    np.testing.assert_allclose(y, 0.5 * x, atol=1e-15)


# ---- Newton-Schulz -------------------------------------------------------------------------------------------
def _poly(s, steps):
    a, b, c = br.NS_COEFFS
    for _ in range(steps):
        s = a * s + b * s ** 3 + c * s ** 5
    return s


@pytest.mark.parametrize("shape", [(3, 8, 8), (2, 6, 14)])
def test_newton_schulz_svd_identity(shape):
    """X_k = U p^k(S / (||G||_F + eps)) V^T: the iteration acts on the singular values only."""
    rng = np.random.default_rng(5)
    G = _r(rng, *shape)
    X = br.newton_schulz(G, steps=5)
    for i in range(shape[0]):
        U, S, Vt = np.linalg.svd(G[i], full_matrices=False)
        s0 = S / (np.sqrt((G[i] ** 2).sum()) + 1e-7)
        np.testing.assert_allclose(X[i], (U * _poly(s0, 5)) @ Vt, atol=1e-11)
    # zero steps: the normalised input; batch entries are independent
    np.testing.assert_allclose(br.newton_schulz(G, steps=0)[1], G[1] / (np.linalg.norm(G[1]) + 1e-7), atol=1e-15)
    np.testing.assert_array_equal(br.newton_schulz(G[1:2], steps=3)[0], br.newton_schulz(G, steps=3)[1])


def test_newton_schulz_orthogonalises():
    """After 5 steps the singular values of a well-conditioned matrix sit in the band the quintic converges to
    (about [0.68, 1.13]); an orthogonal input scaled to Frobenius norm 1 keeps its singular vectors."""
    rng = np.random.default_rng(6)
    G = _r(rng, 1, 16, 16) + 4 * np.eye(16)
    S = np.linalg.svd(br.newton_schulz(G, 5)[0], compute_uv=False)
    assert S.min() > 0.6 and S.max() < 1.2
    Q, _ = np.linalg.qr(_r(rng, 8, 8))
    X = br.newton_schulz(Q[None], 5)[0]
    s = _poly(np.array([1 / np.sqrt(8)]), 5)[0]
    np.testing.assert_allclose(X, s * Q, atol=1e-9)


def test_newton_schulz_round_fn_is_applied():
    from workloads import f32_to_bf16_bits, bf16_bits_to_f64
    rt = lambda z: bf16_bits_to_f64(f32_to_bf16_bits(z.astype(np.float32)))
    rng = np.random.default_rng(7)
    G = _r(rng, 1, 8, 16)
    Xr, Xe = br.newton_schulz(G, 5, round_fn=rt), br.newton_schulz(G, 5)
    assert np.array_equal(Xr, rt(Xr)) and not np.array_equal(Xr, Xe)
    assert np.linalg.norm(Xr - Xe) / np.linalg.norm(Xe) < 3e-2
