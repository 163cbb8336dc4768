"""Timeline of the feature backward kernel on one CTA (developer tool; needs a B200 and a trace build).

    TABATTN_TRACE=1 python -m paper_2606_03681_b200.build --force
    python -m paper_2606_03681_b200.trace_feature_bwd [base|long_item|feature_heavy|ragged]
    python -m paper_2606_03681_b200.build --force          # back to the shipped library

Prints, for tiles 6..39 of CTA 0, the clock64() stamps (relative to the first one) of the events named in
csrc/feature_tc_bwd.cu (TR(...)): one row per tile, columns = TMA issue, S / dP MMA issue, accumulation warp, and the
softmax warpgroup's S-ready, pass A, dP-ready, pass B, turn, P/dS stored, accumulators ready, drained.
"""
import ctypes
import sys

import torch

import paper_2606_03681_b200 as tab
from workloads import get_config, draw_structure, make_call_inputs

NAMES = ["tma", "Siss", "dPiss", "accW", "accC", "sFull", "passA", "dpFull", "passB", "turn", "pdsArr", "accFull", "drained"]


def main():
    cfg = get_config(sys.argv[1] if len(sys.argv) > 1 else "base")
    if not hasattr(tab.lib(), "tabattn_debug_set_trace"):
        raise SystemExit("libtabattn.so was built without TABATTN_TRACE=1")
    dev = torch.device("cuda", 0)
    _, cv_h = draw_structure(cfg)
    cv = torch.from_numpy(cv_h).to(dev) if cv_h is not None else None
    f = make_call_inputs(cfg, "feature", 0, device=dev)
    O, LSE = tab.tabattn_feature_fwd(f["Q"], f["K"], f["V"], cv)
    for _ in range(3):
        tab.tabattn_feature_bwd(f["Q"], f["K"], f["V"], O, f["dO"], LSE, cv)
    trace = torch.zeros(64 * 16, dtype=torch.int64, device=dev)
    torch.cuda.synchronize()
    tab.lib().tabattn_debug_set_trace(ctypes.c_void_p(trace.data_ptr()))
    tab.tabattn_feature_bwd(f["Q"], f["K"], f["V"], O, f["dO"], LSE, cv)
    torch.cuda.synchronize()
    t = trace.cpu().numpy().reshape(64, 16)
    t0 = t[t > 0].min()
    print("tile " + " ".join("%7s" % n for n in NAMES))
    for i in range(6, 40):
        print("%4d " % i + " ".join("%7d" % (t[i, e] - t0 if t[i, e] else -1) for e in range(len(NAMES))))


if __name__ == "__main__":
    main()
