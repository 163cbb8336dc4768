"""Pins of the fp64 oracle against closed forms (SURVEY.md §8(c) "What pins each part")."""
import json
import math
import os

import numpy as np
import pytest

from oracle import ref

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rand(rng, *shape):
    return rng.standard_normal(shape)


def test_golden_two_key_closed_form():
    g = json.load(open(os.path.join(GOLD, "two_key_closed_form.json")))
    # feature attention: B=R=H=1, C=2 keys; only query column 0 has q=1, make column 1's q arbitrary
    q = np.array([g["q"][0], -0.3]).reshape(1, 1, 2, 1, 1)
    k = np.array(g["k"]).reshape(1, 1, 2, 1, 1)
    v = np.array(g["v"]).reshape(1, 1, 2, 1, 1)
    dO = np.array([g["dO"][0], 0.0]).reshape(1, 1, 2, 1, 1)   # zero upstream on the other query
    O, LSE = ref.feature_fwd(q, k, v, scale=g["scale"])
    assert O[0, 0, 0, 0, 0] == pytest.approx(g["O"][0], abs=1e-14)
    assert LSE[0, 0, 0, 0] == pytest.approx(g["LSE"][0], abs=1e-14)
    dq, dk, dv = ref.feature_bwd(q, k, v, dO, scale=g["scale"])
    assert dq[0, 0, 0, 0, 0] == pytest.approx(g["dq"][0], abs=1e-14)
    np.testing.assert_allclose(dk[0, 0, :, 0, 0], g["dk"], atol=1e-14)
    np.testing.assert_allclose(dv[0, 0, :, 0, 0], g["dv"], atol=1e-14)
    # item attention: the same numbers with the two keys as train rows 0,1 and the query as test row 2
    q = np.array([0.7, -0.3, g["q"][0]]).reshape(1, 3, 1, 1, 1)
    k = np.array(g["k"] + [123.0]).reshape(1, 3, 1, 1, 1)
    v = np.array(g["v"] + [-55.0]).reshape(1, 3, 1, 1, 1)
    dO = np.array([0.0, 0.0, g["dO"][0]]).reshape(1, 3, 1, 1, 1)
    nt = np.array([2], np.int32)
    O, LSE = ref.item_fwd(q, k, v, nt, scale=g["scale"])
    assert O[0, 2, 0, 0, 0] == pytest.approx(g["O"][0], abs=1e-14)
    assert LSE[0, 0, 0, 2] == pytest.approx(g["LSE"][0], abs=1e-14)
    dq, dk, dv = ref.item_bwd(q, k, v, dO, nt, scale=g["scale"])
    assert dq[0, 2, 0, 0, 0] == pytest.approx(g["dq"][0], abs=1e-14)
    np.testing.assert_allclose(dk[0, :, 0, 0, 0], g["dk"] + [0.0], atol=1e-14)
    np.testing.assert_allclose(dv[0, :, 0, 0, 0], g["dv"] + [0.0], atol=1e-14)


def test_softmax_weights_via_identity_values():
    """V = identity rows -> O_i = p_i: weights sum to 1, lie in (0,1]."""
    rng = np.random.default_rng(1)
    B, R, C, H, dh = 2, 3, 5, 2, 8
    Q, K = _rand(rng, B, R, C, H, dh), _rand(rng, B, R, C, H, dh)
    V = np.zeros((B, R, C, H, dh))
    for c in range(C):
        V[:, :, c, :, c] = 1.0
    O, _ = ref.feature_fwd(Q, K, V)
    P = O[..., :C]
    assert np.all(P > 0) and np.all(P <= 1)
    np.testing.assert_allclose(P.sum(-1), 1.0, atol=1e-15)
    assert np.all(O[..., C:] == 0)


def test_output_in_value_hull():
    rng = np.random.default_rng(2)
    B, R, C, H, dh = 2, 9, 3, 2, 4
    Q, K, V = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    nt = np.array([5, 9], np.int32)
    O, _ = ref.item_fwd(Q, K, V, nt)
    for b in range(B):
        lo = V[b, :nt[b]].min(axis=0)
        hi = V[b, :nt[b]].max(axis=0)
        assert np.all(O[b] >= lo[None] - 1e-14) and np.all(O[b] <= hi[None] + 1e-14)


@pytest.mark.parametrize("axis", ["feature", "item"])
def test_identical_keys_give_mean_of_values(axis):
    rng = np.random.default_rng(3)
    B, R, C, H, dh = 2, 7, 4, 2, 4
    Q, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    scale = 1.0 / math.sqrt(dh)
    if axis == "feature":
        kvec = _rand(rng, B, R, 1, H, dh)
        K = np.broadcast_to(kvec, Q.shape).copy()
        O, LSE = ref.feature_fwd(Q, K, V)
        np.testing.assert_allclose(O, np.broadcast_to(V.mean(axis=2, keepdims=True), O.shape), atol=1e-14)
        s = scale * np.einsum("brchk,brhk->brhc", Q, kvec[:, :, 0])
        np.testing.assert_allclose(LSE, s + math.log(C), atol=1e-13)
        dq, dk, dv = ref.feature_bwd(Q, K, V, G)
        np.testing.assert_allclose(dq, 0.0, atol=1e-14)
        np.testing.assert_allclose(dv, np.broadcast_to(G.sum(axis=2, keepdims=True) / C, dv.shape), atol=1e-14)
    else:
        nt = np.array([3, 7], np.int32)
        kvec = _rand(rng, B, 1, C, H, dh)
        K = np.broadcast_to(kvec, Q.shape).copy()
        O, LSE = ref.item_fwd(Q, K, V, nt)
        for b in range(B):
            mean = V[b, :nt[b]].mean(axis=0)
            np.testing.assert_allclose(O[b], np.broadcast_to(mean[None], O[b].shape), atol=1e-14)
            s = scale * np.einsum("rchk,chk->chr", Q[b], kvec[b, 0])
            np.testing.assert_allclose(LSE[b], s + math.log(nt[b]), atol=1e-13)
        dq, dk, dv = ref.item_bwd(Q, K, V, G, nt)
        np.testing.assert_allclose(dq, 0.0, atol=1e-14)
        for b in range(B):
            np.testing.assert_allclose(dv[b, :nt[b]], np.broadcast_to(G[b].sum(axis=0, keepdims=True) / nt[b],
                                                                       dv[b, :nt[b]].shape), atol=1e-13)
            assert np.all(dv[b, nt[b]:] == 0) and np.all(dk[b, nt[b]:] == 0)


@pytest.mark.parametrize("axis", ["feature", "item"])
def test_zero_query_gives_uniform_mean(axis):
    rng = np.random.default_rng(4)
    B, R, C, H, dh = 1, 6, 5, 2, 4
    K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    Q = np.zeros_like(K)
    if axis == "feature":
        O, LSE = ref.feature_fwd(Q, K, V)
        np.testing.assert_allclose(O, np.broadcast_to(V.mean(axis=2, keepdims=True), O.shape), atol=1e-14)
        np.testing.assert_allclose(LSE, math.log(C), atol=1e-14)
        _, dk, _ = ref.feature_bwd(Q, K, V, G)
    else:
        nt = np.array([4], np.int32)
        O, LSE = ref.item_fwd(Q, K, V, nt)
        np.testing.assert_allclose(O[0], np.broadcast_to(V[0, :4].mean(axis=0)[None], O[0].shape), atol=1e-14)
        np.testing.assert_allclose(LSE, math.log(4), atol=1e-14)
        _, dk, _ = ref.item_bwd(Q, K, V, G, nt)
    np.testing.assert_allclose(dk, 0.0, atol=1e-15)


def test_single_key_item():
    """n_train = 1: O_i = V_0, LSE_i = s_i0, dV_0 = sum_i dO_i, dQ = dK = 0."""
    rng = np.random.default_rng(5)
    B, R, C, H, dh = 2, 5, 3, 2, 4
    Q, K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(4))
    nt = np.ones(B, np.int32)
    O, LSE = ref.item_fwd(Q, K, V, nt)
    np.testing.assert_allclose(O, np.broadcast_to(V[:, :1], O.shape), atol=1e-15)
    s = np.einsum("brchk,bchk->bchr", Q, K[:, 0]) / math.sqrt(dh)
    np.testing.assert_allclose(LSE, s, atol=1e-14)
    dq, dk, dv = ref.item_bwd(Q, K, V, G, nt)
    np.testing.assert_allclose(dq, 0.0, atol=1e-15)
    np.testing.assert_allclose(dk, 0.0, atol=1e-15)
    np.testing.assert_allclose(dv[:, 0], G.sum(axis=1), atol=1e-14)
    assert np.all(dv[:, 1:] == 0)


def test_single_valid_column_feature():
    rng = np.random.default_rng(6)
    B, R, C, H, dh = 2, 4, 5, 2, 4
    Q, K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(4))
    valid = np.zeros((B, C), np.uint8)
    valid[0, 2] = 1
    valid[1, 4] = 1
    O, LSE = ref.feature_fwd(Q, K, V, valid)
    dq, dk, dv = ref.feature_bwd(Q, K, V, G, valid)
    for b, c in ((0, 2), (1, 4)):
        np.testing.assert_allclose(O[b, :, c], V[b, :, c], atol=1e-15)
        np.testing.assert_allclose(dv[b, :, c], G[b, :, c], atol=1e-15)
        others = [x for x in range(C) if x != c]
        assert np.all(O[b][:, others] == 0) and np.all(LSE[b][:, :, others] == 0)
        assert np.all(dv[b][:, others] == 0)
    np.testing.assert_allclose(dq, 0.0, atol=1e-15)
    np.testing.assert_allclose(dk, 0.0, atol=1e-15)


def test_dominant_key():
    rng = np.random.default_rng(7)
    B, R, C, H, dh = 1, 6, 2, 1, 8
    Q, K, V = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    nt = np.array([4], np.int32)
    qhat = _rand(rng, dh)
    qhat /= np.linalg.norm(qhat)
    Q[:] = 20.0 * qhat
    K[:] = 0.1 * K
    K[0, 2] = 50.0 * qhat            # key row 2 dominates: s = 1000/sqrt(8) ~ 353
    O, _ = ref.item_fwd(Q, K, V, nt)
    np.testing.assert_allclose(O, np.broadcast_to(V[:, 2:3], O.shape), atol=1e-12)


def test_key_shift_invariance():
    """Adding one vector to every key shifts each row of S by a constant."""
    rng = np.random.default_rng(8)
    B, R, C, H, dh = 1, 5, 3, 2, 4
    Q, K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(4))
    nt = np.array([3], np.int32)
    shift = _rand(rng, 1, 1, C, H, dh)
    O0, L0 = ref.item_fwd(Q, K, V, nt)
    O1, L1 = ref.item_fwd(Q, K + shift, V, nt)
    np.testing.assert_allclose(O1, O0, atol=1e-13)
    dL = np.einsum("brchk,bchk->bchr", Q, shift[:, 0]) / math.sqrt(dh)
    np.testing.assert_allclose(L1 - L0, dL, atol=1e-13)
    g0 = ref.item_bwd(Q, K, V, G, nt)
    g1 = ref.item_bwd(Q, K + shift, V, G, nt)
    np.testing.assert_allclose(g1[0], g0[0], atol=1e-13)   # dQ unchanged (sum_j dS_ij = 0)
    np.testing.assert_allclose(g1[2], g0[2], atol=1e-13)   # dV unchanged


def test_scale_argument_and_default():
    rng = np.random.default_rng(9)
    B, R, C, H, dh = 1, 3, 4, 1, 16
    Q, K, V = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    O0, L0 = ref.feature_fwd(Q, K, V)                    # default 1/sqrt(dh) = 0.25
    O1, L1 = ref.feature_fwd(Q, K, V, scale=0.25)
    O2, L2 = ref.feature_fwd(Q * 0.25, K, V, scale=1.0)
    assert np.array_equal(O0, O1) and np.array_equal(L0, L1)
    np.testing.assert_allclose(O2, O0, atol=1e-14)


def test_bf16_entry_equals_double_entry_on_widened_bits():
    from workloads import f32_to_bf16_bits, bf16_bits_to_f64
    rng = np.random.default_rng(10)
    shape = (2, 5, 3, 2, 4)
    bits = [f32_to_bf16_bits(rng.standard_normal(shape).astype(np.float32)) for _ in range(4)]
    dbl = [bf16_bits_to_f64(b) for b in bits]
    nt = np.array([2, 5], np.int32)
    for a, b in zip(ref.item_fwd(*bits[:3], nt), ref.item_fwd(*dbl[:3], nt)):
        assert np.array_equal(a, b)
    for a, b in zip(ref.feature_bwd(*bits), ref.feature_bwd(*dbl)):
        assert np.array_equal(a, b)
