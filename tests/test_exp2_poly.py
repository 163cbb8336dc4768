"""DESIGN.md reading r4: the FMA-pipe exponential of the item kernels (csrc/common.cuh: exp2_poly2).

The kernel code cannot run without a GPU, but its arithmetic is four fp32 constants and a fixed sequence of fp32
operations; this test reads the constants out of the CUDA source and replays the sequence in numpy float32
(round-to-nearest, like the device's FADD2/FFMA2 up to the fused rounding of the fma), and checks the error
bound DESIGN.md states (2.0e-4 relative), exactness of the range split, and the clamp at -126."""
import os
import re

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "..", "paper_2606_03681_b200", "csrc", "common.cuh")


def _coefficients():
    text = open(SRC).read()
    body = text[text.index("void exp2_poly2("):text.index("// 2^x for a pair")]
    c = [np.float32(x) for x in re.findall(r"f2pack\((\d\.\d+)f,", body)]
    assert len(c) == 4, c          # c3, c2, c1, c0 in Horner order
    assert "-126.f" in body and "12582912.f" in body
    return c


def _exp2_poly(x):
    c3, c2, c1, c0 = _coefficients()
    x = np.maximum(np.asarray(x, np.float32), np.float32(-126.0))
    magic = np.float32(12582912.0)
    t = (x + magic).astype(np.float32)
    n = (t - magic).astype(np.float32)
    f = (x - n).astype(np.float32)
    p = (c3 * f + c2).astype(np.float32)
    p = (p * f + c1).astype(np.float32)
    p = (p * f + c0).astype(np.float32)
    bits = p.view(np.int32) + (t.view(np.int32) << 23)          # wraps like the device's 32-bit add
    return bits.astype(np.int32).view(np.float32), n, f


def test_range_split_is_exact_and_centred():
    x = np.random.default_rng(0).uniform(-126, 9, size=200001).astype(np.float32)
    _, n, f = _exp2_poly(x)
    assert np.all(n == np.rint(x))                 # round to nearest (ties to even), exact
    assert np.all(np.abs(f) <= 0.5) and np.all((n + f).astype(np.float32) == x)


def test_relative_error_bound():
    x = np.linspace(-125.5, 8.5, 400001, dtype=np.float32)
    y, _, _ = _exp2_poly(x)
    ref = np.exp2(x.astype(np.float64))
    rel = np.abs(y.astype(np.float64) / ref - 1.0)
    assert rel.max() <= 2.1e-4, rel.max()          # DESIGN.md r4: 2.0e-4, an eighth of the bf16 step 2^-9
    assert rel.max() < 2.0 ** -9 / 8 * 1.1


def test_clamp_and_masked_scores():
    y, _, _ = _exp2_poly(np.array([-np.inf, -1e30, -127.0, -126.0], np.float32))
    assert np.all(np.isfinite(y)) and np.all(y >= 0)
    assert np.all(y <= np.float32(2.0 ** -126) * np.float32(1.001))    # masked score -> ~2^-126, never garbage
    one, _, _ = _exp2_poly(np.array([0.0], np.float32))
    assert abs(float(one[0]) - 1.0) <= 2.1e-4
