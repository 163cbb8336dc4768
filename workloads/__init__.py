"""Seeded synthetic workloads for libtabattn (input generation only).

This package is the ONLY code shared by the CPU oracle (``oracle/``) and the
CUDA path (``paper_2606_03681_b200/``).  It holds no attention arithmetic:
only shapes (BASELINE.json ``configs``), seeded draws of ``n_train`` / column
masks / tensors, and the bf16 <-> float bit conversions needed to hand the
same bits to both sides.  The recipe is stated in DESIGN.md ("Input recipe").
"""
from .bf16 import f32_to_bf16_bits, bf16_bits_to_f32, bf16_bits_to_f64
from .configs import (TabShape, CONFIGS, CONFIG_NAMES, get_config, fig6_shape,
                      draw_structure)
from .gen import make_call_inputs, make_layer_inputs

__all__ = [
    "f32_to_bf16_bits", "bf16_bits_to_f32", "bf16_bits_to_f64",
    "TabShape", "CONFIGS", "CONFIG_NAMES", "get_config", "fig6_shape",
    "draw_structure", "make_call_inputs", "make_layer_inputs",
]
