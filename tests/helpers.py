"""Shared test helpers (comparison rules of SURVEY.md §8(c); no attention arithmetic)."""
import numpy as np

from workloads import f32_to_bf16_bits, bf16_bits_to_f64

# BASELINE.json north_star tolerances (bf16 in, fp32 accumulate)
FWD_REL_L2 = 5e-3
FWD_MAXABS_FRAC = 1e-2      # max|O_gpu - O_ref| <= 1e-2 * max|V|
GRAD_REL_L2 = 1e-2
LSE_TOL = 1e-3              # max|dLSE| <= 1e-3 * max(1, max|LSE|)  (reading c11, reported)


def rel_l2(a, b):
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    den = np.linalg.norm(b.ravel())
    num = np.linalg.norm((a - b).ravel())
    return num / den if den > 0 else num


def rand_bf16(rng, shape, scale=1.0):
    return f32_to_bf16_bits((rng.standard_normal(shape) * scale).astype(np.float32))


def to_f64(bits):
    return bf16_bits_to_f64(bits)
