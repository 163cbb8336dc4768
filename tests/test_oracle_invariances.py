"""Pins of the oracle's structure rules: train-only keys, column mask, independence
("Train-only rule", "Column mask", "Sequence independence", "Library special case")."""
import math

import numpy as np
import pytest

from oracle import ref


def _rand(rng, *shape):
    return rng.standard_normal(shape)


def _np_sdpa(q, k, v, scale):
    """Independent fp64 numpy softmax(q k^T * scale) v and logsumexp; q [Lq,dh], k,v [Lk,dh]."""
    s = (q @ k.T) * scale
    m = s.max(axis=1, keepdims=True)
    e = np.exp(s - m)
    z = e.sum(axis=1, keepdims=True)
    return (e / z) @ v, (m + np.log(z))[:, 0]


def test_matches_numpy_sdpa_feature_and_item():
    rng = np.random.default_rng(11)
    B, R, C, H, dh = 2, 10, 7, 3, 8
    Q, K, V = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    nt = np.array([6, 10], np.int32)
    scale = 1 / math.sqrt(dh)
    O, L = ref.feature_fwd(Q, K, V)
    Oi, Li = ref.item_fwd(Q, K, V, nt)
    for b in range(B):
        for h in range(H):
            for r in range(R):
                o, l = _np_sdpa(Q[b, r, :, h], K[b, r, :, h], V[b, r, :, h], scale)
                np.testing.assert_allclose(O[b, r, :, h], o, atol=1e-12)
                np.testing.assert_allclose(L[b, r, h], l, atol=1e-12)
            for c in range(C):
                o, l = _np_sdpa(Q[b, :, c, h], K[b, :nt[b], c, h], V[b, :nt[b], c, h], scale)
                np.testing.assert_allclose(Oi[b, :, c, h], o, atol=1e-12)
                np.testing.assert_allclose(Li[b, c, h], l, atol=1e-12)


def test_matches_torch_cpu_fp64_sdpa():
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(12)
    B, R, C, H, dh = 1, 9, 4, 2, 8
    Q, K, V = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    nt = np.array([5], np.int32)
    O, _ = ref.item_fwd(Q, K, V, nt)
    # item: sequences over rows, batch = (C,H)
    q = torch.from_numpy(Q[0]).permute(1, 2, 0, 3)          # [C,H,R,dh]
    k = torch.from_numpy(K[0, :5]).permute(1, 2, 0, 3)
    v = torch.from_numpy(V[0, :5]).permute(1, 2, 0, 3)
    o = torch.nn.functional.scaled_dot_product_attention(q, k, v).permute(2, 0, 1, 3).numpy()
    np.testing.assert_allclose(O[0], o, atol=1e-12)


def test_full_train_reduces_to_self_attention():
    """n_b = R: item attention is ordinary full self-attention over rows (pin v)."""
    rng = np.random.default_rng(13)
    B, R, C, H, dh = 1, 6, 2, 2, 4
    Q, K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(4))
    nt = np.array([R], np.int32)
    O, L = ref.item_fwd(Q, K, V, nt)
    # feature attention on the transposed table computes the same thing
    T = lambda x: np.ascontiguousarray(x.transpose(0, 2, 1, 3, 4))
    Of, Lf = ref.feature_fwd(T(Q), T(K), T(V))
    np.testing.assert_allclose(O, T(Of), atol=1e-14)
    np.testing.assert_allclose(L, Lf, atol=1e-14)     # [B,C,H,R] both
    gi = ref.item_bwd(Q, K, V, G, nt)
    gf = ref.feature_bwd(T(Q), T(K), T(V), T(G))
    for a, b in zip(gi, gf):
        np.testing.assert_allclose(a, T(b), atol=1e-13)


def test_train_only_rule_permutations():
    rng = np.random.default_rng(14)
    B, R, C, H, dh = 1, 9, 2, 2, 4
    n = 5
    Q, K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(4))
    nt = np.array([n], np.int32)
    O, L = ref.item_fwd(Q, K, V, nt)
    dq, dk, dv = ref.item_bwd(Q, K, V, G, nt)
    # (i) permute train rows together: test-row outputs unchanged, train-row outputs permute along
    perm = np.concatenate([rng.permutation(n), np.arange(n, R)])
    P = lambda x: x[:, perm]
    O2, L2 = ref.item_fwd(P(Q), P(K), P(V), nt)
    np.testing.assert_allclose(O2, P(O), atol=1e-14)
    np.testing.assert_allclose(L2, L[..., perm], atol=1e-14)
    g2 = ref.item_bwd(P(Q), P(K), P(V), P(G), nt)
    for a, b in zip(g2, (dq, dk, dv)):
        np.testing.assert_allclose(a, P(b), atol=1e-13)
    # (ii) permute test rows: outputs equivariant, dK/dV unchanged
    perm = np.concatenate([np.arange(n), n + rng.permutation(R - n)])
    O3, _ = ref.item_fwd(P(Q), P(K), P(V), nt)
    np.testing.assert_allclose(O3, P(O), atol=1e-14)
    g3 = ref.item_bwd(P(Q), P(K), P(V), P(G), nt)
    np.testing.assert_allclose(g3[0], P(dq), atol=1e-13)
    np.testing.assert_allclose(g3[1], dk, atol=1e-13)
    np.testing.assert_allclose(g3[2], dv, atol=1e-13)


def test_test_rows_are_never_keys():
    rng = np.random.default_rng(15)
    B, R, C, H, dh = 2, 8, 3, 2, 4
    Q, K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(4))
    nt = np.array([5, 3], np.int32)
    base = ref.item_fwd(Q, K, V, nt) + ref.item_bwd(Q, K, V, G, nt)
    K2, V2 = K.copy(), V.copy()
    for b in range(B):
        K2[b, nt[b]:] = np.nan           # (iii)/(iv): K,V of test rows must not matter, even NaN
        V2[b, nt[b]:] = np.inf
    other = ref.item_fwd(Q, K2, V2, nt) + ref.item_bwd(Q, K2, V2, G, nt)
    for a, b in zip(base, other):
        assert np.array_equal(a, b)
    # changing Q / dO of one test row t changes only O_t, LSE_t, dQ_t (+ its additive share of dK,dV)
    t = 6
    Q3, G3 = Q.copy(), G.copy()
    Q3[0, t] += 1.0
    G3[0, t] -= 2.0
    O3, L3 = ref.item_fwd(Q3, K, V, nt)
    dq3, dk3, dv3 = ref.item_bwd(Q3, K, V, G3, nt)
    keep = [r for r in range(R) if r != t]
    assert np.array_equal(O3[0, keep], base[0][0, keep]) and np.array_equal(O3[1], base[0][1])
    assert np.array_equal(L3[0][..., keep], base[1][0][..., keep])
    assert np.array_equal(dq3[0, keep], base[2][0, keep])
    assert not np.array_equal(O3[0, t], base[0][0, t])
    # additive contribution: dK(all rows) - dK(without row t's dO and with old Q) == contribution of row t alone
    G_only = np.zeros_like(G)
    G_only[0, t] = G3[0, t]
    _, dk_only, dv_only = ref.item_bwd(Q3, K, V, G_only, nt)
    G_rest = G.copy()
    G_rest[0, t] = 0
    _, dk_rest, dv_rest = ref.item_bwd(Q, K, V, G_rest, nt)
    np.testing.assert_allclose(dk3, dk_rest + dk_only, atol=1e-13)
    np.testing.assert_allclose(dv3, dv_rest + dv_only, atol=1e-13)


@pytest.mark.parametrize("axis", ["feature", "item"])
def test_mask_equals_physical_compaction(axis):
    rng = np.random.default_rng(16)
    B, R, C, H, dh = 2, 6, 6, 2, 4
    Q, K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(4))
    valid = np.array([[1, 0, 1, 1, 0, 1], [0, 1, 1, 0, 0, 1]], np.uint8)
    nt = np.array([4, 6], np.int32)
    # NaN-poison the invalid columns: must not leak
    Qp, Kp, Vp, Gp = (x.copy() for x in (Q, K, V, G))
    for b in range(B):
        for x in (Qp, Kp, Vp, Gp):
            x[b][:, valid[b] == 0] = np.nan
    if axis == "feature":
        full = ref.feature_fwd(Qp, Kp, Vp, valid) + ref.feature_bwd(Qp, Kp, Vp, Gp, valid)
    else:
        full = ref.item_fwd(Qp, Kp, Vp, nt, valid) + ref.item_bwd(Qp, Kp, Vp, Gp, nt, valid)
    assert all(np.isfinite(x).all() for x in full)
    for b in range(B):
        cols = np.flatnonzero(valid[b])
        inval = np.flatnonzero(valid[b] == 0)
        sl = lambda x: np.ascontiguousarray(x[b:b + 1][:, :, cols])
        if axis == "feature":
            comp = ref.feature_fwd(sl(Q), sl(K), sl(V)) + ref.feature_bwd(sl(Q), sl(K), sl(V), sl(G))
            lse_full = full[1][b][:, :, cols]
            lse_inv = full[1][b][:, :, inval]
        else:
            comp = ref.item_fwd(sl(Q), sl(K), sl(V), nt[b:b + 1]) + ref.item_bwd(sl(Q), sl(K), sl(V), sl(G), nt[b:b + 1])
            lse_full = full[1][b][cols]
            lse_inv = full[1][b][inval]
        assert np.array_equal(lse_full, comp[1][0])
        assert np.all(lse_inv == 0)
        for i in (0, 2, 3, 4):
            assert np.array_equal(full[i][b][:, cols], comp[i][0])
            assert np.all(full[i][b][:, inval] == 0)


def test_all_valid_mask_equals_no_mask_and_empty_table():
    rng = np.random.default_rng(17)
    B, R, C, H, dh = 2, 4, 3, 1, 4
    Q, K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(4))
    nt = np.array([2, 4], np.int32)
    ones = np.ones((B, C), np.uint8)
    for a, b in zip(ref.feature_fwd(Q, K, V, ones), ref.feature_fwd(Q, K, V)):
        assert np.array_equal(a, b)
    for a, b in zip(ref.item_bwd(Q, K, V, G, nt, ones), ref.item_bwd(Q, K, V, G, nt)):
        assert np.array_equal(a, b)
    none = ones.copy()
    none[1] = 0                           # table 1 has no valid column (reading c9): all zeros
    O, L = ref.feature_fwd(Q, K, V, none)
    assert np.all(O[1] == 0) and np.all(L[1] == 0)
    O, L = ref.item_fwd(Q, K, V, nt, none)
    assert np.all(O[1] == 0) and np.all(L[1] == 0)


def test_selection_equals_slice_of_full_result():
    rng = np.random.default_rng(18)
    B, R, C, H, dh = 2, 5, 4, 2, 4
    Q, K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(4))
    nt = np.array([3, 5], np.int32)
    O, L = ref.item_fwd(Q, K, V, nt)
    dq, dk, dv = ref.item_bwd(Q, K, V, G, nt)
    sel = [[1, 2], [0, 3]]
    Os, Ls = ref.item_fwd(Q, K, V, nt, cols=sel)
    gs = ref.item_bwd(Q, K, V, G, nt, cols=sel)
    for n, (b, c) in enumerate(sel):
        assert np.array_equal(Os[n], O[b, :, c]) and np.array_equal(Ls[n], L[b, c])
        for a, f in zip(gs, (dq, dk, dv)):
            assert np.array_equal(a[n], f[b, :, c])
    # a single (b, c) computed alone from a physically sliced table equals its slice, bit for bit
    one = ref.item_fwd(np.ascontiguousarray(Q[1:2, :, 2:3]), np.ascontiguousarray(K[1:2, :, 2:3]),
                       np.ascontiguousarray(V[1:2, :, 2:3]), nt[1:2])
    assert np.array_equal(one[0][0, :, 0], O[1, :, 2])
    Of, Lf = ref.feature_fwd(Q, K, V)
    Osel, Lsel = ref.feature_fwd(Q, K, V, rows=[[1, 4], [0, 0]])
    assert np.array_equal(Osel[0], Of[1, 4]) and np.array_equal(Lsel[1], Lf[0, 0])


def test_bad_arguments_raise():
    Q = np.zeros((1, 2, 2, 1, 4))
    with pytest.raises(ValueError):
        ref.item_fwd(Q, Q, Q, np.array([0], np.int32))       # n_train = 0 is an error (reading c8)
    with pytest.raises(ValueError):
        ref.item_fwd(Q, Q, Q, np.array([3], np.int32))
    with pytest.raises(TypeError):
        ref.feature_fwd(Q.astype(np.float32), Q.astype(np.float32), Q.astype(np.float32))
