"""Oracle vs scalar-loop brute force and vs central finite differences
("Brute force on tiny tables", "Gradients")."""
import numpy as np
import pytest

from oracle import brute, ref
from workloads import bf16_bits_to_f64, get_config, make_call_inputs, draw_structure


def _rand(rng, *shape):
    return rng.standard_normal(shape)


@pytest.mark.parametrize("masked", [False, True])
def test_bruteforce_tiny(masked):
    rng = np.random.default_rng(21)
    B, R, C, H, dh = 2, 8, 4, 2, 4
    Q, K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(4))
    valid = np.array([[1, 0, 1, 1], [1, 1, 1, 0]], np.uint8) if masked else None
    nt = np.array([5, 8], np.int32)
    Ob, Lb, gb = brute.feature(Q, K, V, G, valid)
    O, L = ref.feature_fwd(Q, K, V, valid)
    g = ref.feature_bwd(Q, K, V, G, valid)
    np.testing.assert_allclose(O, Ob, atol=1e-13)
    np.testing.assert_allclose(L, Lb, atol=1e-13)
    for a, b in zip(g, gb):
        np.testing.assert_allclose(a, b, atol=1e-13)
    Ob, Lb, gb = brute.item(Q, K, V, nt, G, valid)
    O, L = ref.item_fwd(Q, K, V, nt, valid)
    g = ref.item_bwd(Q, K, V, G, nt, valid)
    np.testing.assert_allclose(O, Ob, atol=1e-13)
    np.testing.assert_allclose(L, Lb, atol=1e-13)
    for a, b in zip(g, gb):
        np.testing.assert_allclose(a, b, atol=1e-13)


def _fd_check(fwd, bwd, tensors, G, coords, h=1e-5, tol=1e-7):
    """L = sum(O * G); compare analytic dL/dx with central differences at `coords`."""
    grads = bwd(*tensors, G)
    for ti, name in enumerate("QKV"):
        for idx in coords[ti]:
            plus = [t.copy() for t in tensors]
            minus = [t.copy() for t in tensors]
            plus[ti][idx] += h
            minus[ti][idx] -= h
            fd = ((fwd(*plus)[0] * G).sum() - (fwd(*minus)[0] * G).sum()) / (2 * h)
            an = grads[ti][idx]
            assert abs(fd - an) <= tol * max(1.0, abs(an)), (name, idx, fd, an)


def _all_coords(shape):
    return [tuple(i) for i in np.ndindex(*shape)]


@pytest.mark.parametrize("masked", [False, True])
def test_finite_differences_all_coordinates_tiny(masked):
    rng = np.random.default_rng(22)
    B, R, C, H, dh = 1, 4, 3, 2, 2
    Q, K, V, G = (_rand(rng, B, R, C, H, dh) for _ in range(4))
    valid = np.array([[1, 0, 1]], np.uint8) if masked else None
    nt = np.array([3], np.int32)
    coords = [_all_coords(Q.shape)] * 3
    _fd_check(lambda q, k, v: ref.feature_fwd(q, k, v, valid),
              lambda q, k, v, g: ref.feature_bwd(q, k, v, g, valid), [Q, K, V], G, coords)
    _fd_check(lambda q, k, v: ref.item_fwd(q, k, v, nt, valid),
              lambda q, k, v, g: ref.item_bwd(q, k, v, g, nt, valid), [Q, K, V], G, coords)


def test_finite_differences_random_coordinates_on_tiny_config():
    cfg = get_config("tiny")
    nt, _ = draw_structure(cfg)
    rng = np.random.default_rng(23)
    for axis in ("feature", "item"):
        x = make_call_inputs(cfg, axis)
        Q, K, V, G = (bf16_bits_to_f64(x[k]) for k in ("Q", "K", "V", "dO"))
        coords = [[tuple(rng.integers(0, s) for s in Q.shape) for _ in range(64)] for _ in range(3)]
        if axis == "feature":
            _fd_check(ref.feature_fwd, ref.feature_bwd, [Q, K, V], G, coords)
        else:
            _fd_check(lambda q, k, v: ref.item_fwd(q, k, v, nt),
                      lambda q, k, v, g: ref.item_bwd(q, k, v, g, nt), [Q, K, V], G, coords)


def test_gradient_structure():
    """dV linear in dO; scaling dO by a scales all grads by a; zero dO on train rows
    (last layer: only test-row O feeds the loss) is handled."""
    rng = np.random.default_rng(24)
    B, R, C, H, dh = 1, 7, 2, 2, 4
    Q, K, V, G1, G2 = (_rand(rng, B, R, C, H, dh) for _ in range(5))
    nt = np.array([4], np.int32)
    g1 = ref.item_bwd(Q, K, V, G1, nt)
    g2 = ref.item_bwd(Q, K, V, G2, nt)
    g12 = ref.item_bwd(Q, K, V, G1 + G2, nt)
    ga = ref.item_bwd(Q, K, V, -2.5 * G1, nt)
    for a, b, c, d in zip(g1, g2, g12, ga):
        np.testing.assert_allclose(c, a + b, atol=1e-13)
        np.testing.assert_allclose(d, -2.5 * a, atol=1e-13)
    G0 = G1.copy()
    G0[:, :4] = 0
    dq, dk, dv = ref.item_bwd(Q, K, V, G0, nt)
    assert np.all(dq[:, :4] == 0) and np.any(dk[:, :4] != 0) and np.any(dv[:, :4] != 0)
