"""Pins of the evaluation-path oracle (oracle/eval_ref.py): the forward restricted to a
query-row range.  Checked against things other than itself: the independently written C oracle's full forward
(oracle/tabattn_ref.c), the hand-derived golden fixture, closed forms and the invariances the row range and the
train-only key rule imply."""
import json
import os

import numpy as np
import pytest

from oracle import eval_ref, ref

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rand(rng, *shape):
    return rng.standard_normal(shape)


def _mask(rng, B, C):
    m = (rng.random((B, C)) < 0.6).astype(np.uint8)
    m[:, C - 1] = 1
    return m


@pytest.mark.parametrize("masked", [False, True])
def test_item_infer_equals_slice_of_full_forward(masked):
    rng = np.random.default_rng(11)
    B, R, C, H, dh = 2, 37, 5, 2, 8
    Q, K, V = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    nt = np.array([20, 37], np.int32)
    cv = _mask(rng, B, C) if masked else None
    full, _ = ref.item_fwd(Q, K, V, nt, cv)
    for row0, row1 in ((0, R), (20, 37), (5, 6), (30, 33)):
        O = eval_ref.item_fwd_infer(Q, K, V, nt, row0, row1, cv)
        np.testing.assert_allclose(O, full[:, row0:row1], atol=1e-12, rtol=0)


@pytest.mark.parametrize("masked", [False, True])
def test_feature_infer_equals_slice_of_full_forward(masked):
    rng = np.random.default_rng(12)
    B, R, C, H, dh = 2, 9, 7, 2, 4
    Q, K, V = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    cv = _mask(rng, B, C) if masked else None
    full, _ = ref.feature_fwd(Q, K, V, cv)
    for row0, row1 in ((0, R), (3, 8), (8, 9)):
        O = eval_ref.feature_fwd_infer(Q, K, V, row0, row1, cv)
        np.testing.assert_allclose(O, full[:, row0:row1], atol=1e-12, rtol=0)


def test_golden_two_key_closed_form_on_a_test_row():
    g = json.load(open(os.path.join(GOLD, "two_key_closed_form.json")))
    # two train rows as keys, the query as test row 2 (the only row of the range)
    q = np.array([0.7, -0.3, g["q"][0]]).reshape(1, 3, 1, 1, 1)
    k = np.array(g["k"] + [123.0]).reshape(1, 3, 1, 1, 1)
    v = np.array(g["v"] + [-55.0]).reshape(1, 3, 1, 1, 1)
    O = eval_ref.item_fwd_infer(q, k, v, np.array([2], np.int32), 2, 3, scale=g["scale"])
    assert O.shape == (1, 1, 1, 1, 1)
    assert O[0, 0, 0, 0, 0] == pytest.approx(g["O"][0], abs=1e-14)
    # feature axis: the two keys as two columns of one row
    q = np.array([g["q"][0], -0.3]).reshape(1, 1, 2, 1, 1)
    k = np.array(g["k"]).reshape(1, 1, 2, 1, 1)
    v = np.array(g["v"]).reshape(1, 1, 2, 1, 1)
    O = eval_ref.feature_fwd_infer(q, k, v, 0, 1, scale=g["scale"])
    assert O[0, 0, 0, 0, 0] == pytest.approx(g["O"][0], abs=1e-14)


def test_single_key_and_identical_keys():
    rng = np.random.default_rng(13)
    B, R, C, H, dh = 1, 12, 3, 2, 4
    Q, K, V = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    # n_train = 1: every query returns V_0
    O = eval_ref.item_fwd_infer(Q, K, V, np.array([1], np.int32), 4, 12)
    np.testing.assert_allclose(O, np.broadcast_to(V[:, 0:1], O.shape), atol=1e-14)
    # identical keys among the train rows: O = arithmetic mean of the train V
    n = 7
    K2 = K.copy()
    K2[:, :n] = K[:, 0:1]
    O = eval_ref.item_fwd_infer(Q, K2, V, np.array([n], np.int32), 7, 12)
    np.testing.assert_allclose(O, np.broadcast_to(V[:, :n].mean(axis=1, keepdims=True), O.shape), atol=1e-13)


def test_row_range_and_train_only_invariances():
    rng = np.random.default_rng(14)
    B, R, C, H, dh = 2, 20, 3, 1, 4
    Q, K, V = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    nt = np.array([12, 15], np.int32)
    base = eval_ref.item_fwd_infer(Q, K, V, nt, 15, 20)
    # queries outside the range never matter
    Q2 = Q.copy()
    Q2[:, :15] = rng.standard_normal(Q2[:, :15].shape)
    np.testing.assert_array_equal(eval_ref.item_fwd_infer(Q2, K, V, nt, 15, 20), base)
    # K, V of the rows that are not train rows never matter, even NaN
    K2, V2 = K.copy(), V.copy()
    for b in range(B):
        K2[b, nt[b]:] = np.nan
        V2[b, nt[b]:] = np.nan
    np.testing.assert_array_equal(eval_ref.item_fwd_infer(Q, K2, V2, nt, 15, 20), base)
    # permuting the train rows (K and V together) leaves the test-row outputs unchanged
    K3, V3 = K.copy(), V.copy()
    for b in range(B):
        perm = rng.permutation(nt[b])
        K3[b, :nt[b]] = K[b, perm]
        V3[b, :nt[b]] = V[b, perm]
    np.testing.assert_allclose(eval_ref.item_fwd_infer(Q, K3, V3, nt, 15, 20), base, atol=1e-13)
    # chunks of the range tile it exactly (train-row K/V reused across test chunks)
    parts = [eval_ref.item_fwd_infer(Q, K, V, nt, a, b) for a, b in ((15, 17), (17, 18), (18, 20))]
    np.testing.assert_allclose(np.concatenate(parts, axis=1), base, atol=1e-14, rtol=0)


def test_invalid_columns_and_bf16_bits():
    rng = np.random.default_rng(15)
    B, R, C, H, dh = 1, 6, 4, 1, 2
    Q, K, V = (_rand(rng, B, R, C, H, dh) for _ in range(3))
    cv = np.array([[1, 0, 1, 1]], np.uint8)
    O = eval_ref.item_fwd_infer(Q, K, V, np.array([3], np.int32), 3, 6, cv)
    assert np.all(O[:, :, 1] == 0)
    Kp = K.copy()
    Kp[:, :, 1] = np.nan
    Of = eval_ref.feature_fwd_infer(Q, Kp, V, 0, 6, cv)
    assert np.all(Of[:, :, 1] == 0) and np.isfinite(Of).all()
    # uint16 inputs are widened exactly: 0x3F80 = 1.0, 0xC000 = -2.0
    bits = np.full((1, 2, 1, 1, 1), 0x3F80, np.uint16)
    vb = np.array([0x3F80, 0xC000], np.uint16).reshape(1, 2, 1, 1, 1)
    O = eval_ref.item_fwd_infer(bits, bits, vb, np.array([2], np.int32), 0, 1, scale=1.0)
    assert O[0, 0, 0, 0, 0] == pytest.approx(-0.5, abs=1e-15)
