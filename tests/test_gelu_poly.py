"""DESIGN.md reading b4: the GELU of the GEMM epilogues (csrc/gemm_tc.cu: erf_half2, gelu_pair, gelu_grad_pair).

The device code cannot run without a GPU, but its arithmetic is nine fp32 constants, a clamp and a fixed Horner
sequence; this test reads the constants out of the CUDA source, replays the sequence in numpy float32 and checks the
error bounds DESIGN.md states against math.erf in fp64: |erf error| <= 4.2e-5, |gelu error| <= 8.8e-5 (absolute) and
the same for the derivative, on [-6, 6]; odd symmetry; saturation beyond the clamp."""
import math
import os
import re

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "..", "paper_2606_03681_b200", "csrc", "gemm_tc.cu")


def _coefficients():
    text = open(SRC).read()
    body = text[text.index("uint64_t erf_half2("):text.index("// gelu(x) = x/2")]
    c = [np.float32(x) for x in re.findall(r"pk2\((-?\d\.\d+e[+-]\d+)f\)", body)]
    assert len(c) == 9, c                      # c8 ... c0 in Horner order
    assert "fminf(fmaxf(a, -3.f), 3.f)" in body and "0.70710678118654752f" in body
    return c


def _erf_half(x):
    c = _coefficients()
    z = (np.asarray(x, np.float32) * np.float32(0.70710678118654752)).astype(np.float32)
    z = np.clip(z, np.float32(-3), np.float32(3))
    s = (z * z).astype(np.float32)
    p = (c[0] * s + c[1]).astype(np.float32)
    for ck in c[2:]:
        p = (p * s + ck).astype(np.float32)
    return (z * p).astype(np.float32)


X = np.linspace(-6, 6, 200001).astype(np.float32)
ERF = np.array([math.erf(float(v) / math.sqrt(2.0)) for v in X])


def test_erf_polynomial_error_bound():
    got = _erf_half(X).astype(np.float64)
    assert np.abs(got - ERF).max() <= 4.2e-5
    assert np.array_equal(_erf_half(-X), -_erf_half(X))                    # odd, exactly
    far = _erf_half(np.array([4.5, 10.0, 1e30, -1e30], np.float32))
    assert np.all(np.abs(np.abs(far) - 1.0) <= 4.2e-5) and far[3] < 0      # saturates at the clamp


def test_gelu_and_derivative_error_bounds():
    x = X.astype(np.float64)
    er = _erf_half(X).astype(np.float64)
    gelu = 0.5 * x + 0.5 * x * er
    assert np.abs(gelu - 0.5 * x * (1.0 + ERF)).max() <= 8.8e-5
    gauss = x * np.exp(-0.5 * x * x) / math.sqrt(2.0 * math.pi)
    grad = 0.5 + 0.5 * er + gauss
    assert np.abs(grad - (0.5 * (1.0 + ERF) + gauss)).max() <= 2.5e-5
    # where it matters for a bf16 result: relative error below a quarter of the bf16 rounding step for |gelu| >= 0.05
    ref = 0.5 * x * (1.0 + ERF)
    big = np.abs(ref) >= 0.05
    assert (np.abs(gelu - ref)[big] / np.abs(ref)[big]).max() <= 2.0 ** -9 / 2
