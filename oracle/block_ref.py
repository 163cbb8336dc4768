"""fp64 oracle of the sub-blocks around the attention kernels.

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / ``--impl reference`` leg may import this module.  It shares nothing with
paper_2606_03681_b200/ and never imports it.

Plain numpy float64, written out in the order of the definitions; the only primitives are
``numpy`` matmul, ``scipy.special.erf`` and the attention oracle (oracle/ref.py, itself pinned).
Passages: PAPER.md:L69 (Fig. 3: attention, norm, attention, norm, MLP, norm per block), L91 (the
norms move ahead of attention and MLP: pre-norm), L99 (block input scaled by 0.95^i), L105 / L294
(RMSNorm), L277 (explicit Q, K, V), L81 / L342 (MLP hidden 768), L85-87, L95, L286 (Muon, batched
Newton-Schulz).  Readings where the paper is silent (b1-b6): no biases; gain-only
RMSNorm  xs / sqrt(mean(xs^2) + eps) * g;  exact (erf) GELU;  weights [out][in];  the decay alpha
multiplies the sub-block's input, and the residual carries the scaled input;  Newton-Schulz as
published for Muon (quintic, coefficients 3.4445, -4.7750, 2.0315, Frobenius pre-normalisation).

    attention sub-block:  xs = alpha x;  h = rmsnorm(xs) g;  [q|k|v] = h Wqkv^T;  o = attn(q,k,v);
                          y = xs + o Wo^T
    MLP sub-block:        xs = alpha x;  h = rmsnorm(xs) g;  u = h W1^T;  a = gelu(u);  y = xs + a W2^T

The backward functions recompute everything from the inputs (they take no saved activations).
Pinned in tests/test_oracle_blocks.py against torch-CPU fp64 autograd on an independently written
formulation (F.rms_norm, F.linear, F.gelu, F.scaled_dot_product_attention), central finite
differences, closed forms, and -- for Newton-Schulz -- the SVD identity X_k = U p^k(S) V^T.
"""
import numpy as np
from scipy.special import erf

from . import ref

NS_COEFFS = (3.4445, -4.7750, 2.0315)


def widen(a):
    """uint16 bf16 bit patterns -> float64 (exact); float64 passes through."""
    a = np.asarray(a)
    if a.dtype == np.uint16:
        return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    return a.astype(np.float64)


# ---- RMSNorm -----------------------------------------------------------------------------------------
def rmsnorm_fwd(xs, g, eps):
    rstd = 1.0 / np.sqrt((xs * xs).mean(axis=-1, keepdims=True) + eps)
    return xs * rstd * g, rstd


def rmsnorm_bwd(xs, g, rstd, dh):
    """d/dxs of h = xs rstd g  given dh; also dg."""
    xh = xs * rstd
    t = dh * g
    c = (t * xh).mean(axis=-1, keepdims=True)
    return rstd * (t - xh * c), (dh * xh).reshape(-1, xs.shape[-1]).sum(axis=0)


def gelu(u):
    return 0.5 * u * (1.0 + erf(u / np.sqrt(2.0)))


def gelu_grad(u):
    return 0.5 * (1.0 + erf(u / np.sqrt(2.0))) + u * np.exp(-0.5 * u * u) / np.sqrt(2.0 * np.pi)


# ---- MLP sub-block -------------------------------------------------------------------------------------
def mlp_fwd(x, g, W1, W2, alpha=1.0, eps=1e-6):
    x, g, W1, W2 = widen(x), widen(g), widen(W1), widen(W2)
    xs = alpha * x
    h, _ = rmsnorm_fwd(xs, g, eps)
    u = h @ W1.T
    a = gelu(u)
    return xs + a @ W2.T


def mlp_bwd(x, g, W1, W2, dy, alpha=1.0, eps=1e-6):
    """Returns dx [cells,e], dg [e], dW1 [hidden,e], dW2 [e,hidden]."""
    x, g, W1, W2, dy = widen(x), widen(g), widen(W1), widen(W2), widen(dy)
    xs = alpha * x
    h, rstd = rmsnorm_fwd(xs, g, eps)
    u = h @ W1.T
    a = gelu(u)
    da = dy @ W2
    dW2 = dy.T @ a
    du = da * gelu_grad(u)
    dW1 = du.T @ h
    dh = du @ W1
    dxs_norm, dg = rmsnorm_bwd(xs, g, rstd, dh)
    return alpha * (dy + dxs_norm), dg, dW1, dW2


# ---- attention sub-block ---------------------------------------------------------------------------------
def _attention_fwd(axis, q, k, v, n_train, col_valid):
    return (ref.feature_fwd(q, k, v, col_valid) if axis == "feature" else ref.item_fwd(q, k, v, n_train, col_valid))[0]


def _attention_bwd(axis, q, k, v, do, n_train, col_valid):
    if axis == "feature":
        return ref.feature_bwd(q, k, v, do, col_valid)
    return ref.item_bwd(q, k, v, do, n_train, col_valid)


def attn_block_fwd(axis, x, g, Wqkv, Wo, H, n_train=None, col_valid=None, alpha=1.0, eps=1e-6):
    """x [B,R,C,e] -> y [B,R,C,e]; axis 'feature' or 'item'."""
    x, g, Wqkv, Wo = widen(x), widen(g), widen(Wqkv), widen(Wo)
    B, R, C, e = x.shape
    dh_ = e // H
    xs = alpha * x
    h, _ = rmsnorm_fwd(xs, g, eps)
    qkv = h @ Wqkv.T
    q, k, v = (np.ascontiguousarray(qkv[..., i * e:(i + 1) * e]).reshape(B, R, C, H, dh_) for i in range(3))
    o = _attention_fwd(axis, q, k, v, n_train, col_valid).reshape(B, R, C, e)
    return xs + o @ Wo.T


def attn_block_bwd(axis, x, g, Wqkv, Wo, dy, H, n_train=None, col_valid=None, alpha=1.0, eps=1e-6):
    """Returns dx [B,R,C,e], dg [e], dWqkv [3e,e], dWo [e,e]."""
    x, g, Wqkv, Wo, dy = widen(x), widen(g), widen(Wqkv), widen(Wo), widen(dy)
    B, R, C, e = x.shape
    dh_ = e // H
    xs = alpha * x
    h, rstd = rmsnorm_fwd(xs, g, eps)
    qkv = h @ Wqkv.T
    q, k, v = (np.ascontiguousarray(qkv[..., i * e:(i + 1) * e]).reshape(B, R, C, H, dh_) for i in range(3))
    o = _attention_fwd(axis, q, k, v, n_train, col_valid).reshape(B, R, C, e)
    do = dy @ Wo
    dWo = dy.reshape(-1, e).T @ o.reshape(-1, e)
    dq, dk, dv = _attention_bwd(axis, q, k, v, np.ascontiguousarray(do).reshape(B, R, C, H, dh_), n_train, col_valid)
    dqkv = np.concatenate([t.reshape(B, R, C, e) for t in (dq, dk, dv)], axis=-1)
    dWqkv = dqkv.reshape(-1, 3 * e).T @ h.reshape(-1, e)
    dh = dqkv @ Wqkv
    dxs_norm, dg = rmsnorm_bwd(xs, g, rstd, dh)
    return alpha * (dy + dxs_norm), dg, dWqkv, dWo


# ---- batched Newton-Schulz (Muon) --------------------------------------------------------------------------
def newton_schulz(G, steps=5, eps=1e-7, round_fn=None):
    """G [nb,m,n] (m <= n).  X = G / (||G||_F + eps); steps x: A = X X^T; B = b A + c A A; X = a X + B X.
    ``round_fn`` (optional) is applied to X0, A, B and every new X: it models the bf16 storage of the
    iterates that Muon prescribes (the caller passes a bf16 round-trip); None = exact fp64."""
    a, b, c = NS_COEFFS
    rf = round_fn if round_fn is not None else (lambda z: z)
    G = widen(G)
    out = np.empty_like(G)
    for i in range(G.shape[0]):
        X = rf(G[i] / (np.sqrt((G[i] * G[i]).sum()) + eps))
        for _ in range(steps):
            A = rf(X @ X.T)
            Bm = rf(b * A + c * (A @ A))
            X = rf(a * X + Bm @ X)
        out[i] = X
    return out
