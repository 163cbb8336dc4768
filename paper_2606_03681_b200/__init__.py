"""paper_2606_03681_b200 -- libtabattn: B200 (sm_100a) dual-axis attention, forward and backward.

The data-parallel hot path of the nanoTabPFN (TabPFN-v2-style) pretraining step that
arxiv/paper_2606_03681 speedruns (Fig. 3, L91, L277, L294): feature-axis and
item-axis scaled-dot-product attention over a [B,R,C,H,dh] cell tensor.  The product is the
C-ABI library declared in include/tabattn.h (csrc/); this package is its ctypes binding.
"""
from . import binding
from .binding import (TabattnError, TabattnShape, EXPORTS, LIB_PATH, lib, make_shape, status_string, version, launch_count,
                      workspace_bytes, tabattn_feature_fwd, tabattn_feature_bwd, tabattn_item_fwd,
                      tabattn_item_bwd, tabattn_feature_fwd_infer, tabattn_item_fwd_infer, tabattn_item_fwd_noalloc,
                      NOALLOC_MAX_BC, OP_FEATURE_FWD, OP_FEATURE_BWD, OP_ITEM_FWD, OP_ITEM_BWD,
                      OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_WORKSPACE, ERR_CUDA)
from .binding import (tabattn_attn_block_fwd, tabattn_attn_block_bwd, tabattn_mlp_fwd, tabattn_mlp_bwd,
                      tabattn_newton_schulz, AttnSaved, MlpSaved)
from .layer import LayerBuffers, LayerGraph, layer_fwd_bwd, layer_fwd_bwd_host

__all__ = [
    "TabattnError", "TabattnShape", "EXPORTS", "LIB_PATH", "lib", "make_shape", "status_string", "version", "launch_count",
    "workspace_bytes", "tabattn_feature_fwd", "tabattn_feature_bwd", "tabattn_item_fwd", "tabattn_item_bwd",
    "tabattn_feature_fwd_infer", "tabattn_item_fwd_infer", "tabattn_item_fwd_noalloc", "NOALLOC_MAX_BC",
    "tabattn_attn_block_fwd", "tabattn_attn_block_bwd",
    "tabattn_mlp_fwd", "tabattn_mlp_bwd", "tabattn_newton_schulz", "AttnSaved", "MlpSaved", "LayerBuffers", "LayerGraph", "layer_fwd_bwd", "layer_fwd_bwd_host",
]
