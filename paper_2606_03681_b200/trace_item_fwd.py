"""Timeline of the item forward kernel's first softmax warpgroup on one CTA (developer tool; needs a B200 and a trace
build).

    TABATTN_TRACE=1 python -m paper_2606_03681_b200.build --force
    python -m paper_2606_03681_b200.trace_item_fwd [base|long_item|feature_heavy|ragged]
    python -m paper_2606_03681_b200.build --force          # back to the shipped library

Prints, for key-tile steps 4..47 of CTA 0, the clock64() stamps (relative to the first one) of the first thread of each
softmax warpgroup at the events named in csrc/item_tc_fwd.cu (TR(...)): S ready, S loaded from TMEM (buffer released),
row maximum done, exponentials done, P buffer free (previous PV finished), P stored; then warpgroup 0's two epilogue
stamps (last PV done, O stored; only on an item's last step) and the step-to-step difference of the first column.
"""
import ctypes
import sys

import torch

import paper_2606_03681_b200 as tab
from workloads import get_config, draw_structure, make_call_inputs

EV = ["sFull", "sLoaded", "maxDone", "expDone", "pFree", "pStored", "-"]
NAMES = [e + "0" for e in EV] + [e + "1" for e in EV] + ["lastPV", "oStored"]

def main():
    cfg = get_config(sys.argv[1] if len(sys.argv) > 1 else "base")
    if not hasattr(tab.lib(), "tabattn_debug_set_trace_item_fwd"):
        raise SystemExit("libtabattn.so was built without TABATTN_TRACE=1")
    dev = torch.device("cuda", 0)
    nt_h, cv_h = draw_structure(cfg)
    nt = torch.from_numpy(nt_h).to(dev)
    cv = torch.from_numpy(cv_h).to(dev) if cv_h is not None else None
    f = make_call_inputs(cfg, "item", 0, device=dev)
    for _ in range(3):
        tab.tabattn_item_fwd(f["Q"], f["K"], f["V"], nt, cv)
    trace = torch.zeros(64 * 16, dtype=torch.int64, device=dev)
    torch.cuda.synchronize()
    tab.lib().tabattn_debug_set_trace_item_fwd(ctypes.c_void_p(trace.data_ptr()))
    tab.tabattn_item_fwd(f["Q"], f["K"], f["V"], nt, cv)
    torch.cuda.synchronize()
    t = trace.cpu().numpy().reshape(64, 16)
    t0 = t[t > 0].min()
    print("step " + " ".join("%8s" % n for n in NAMES) + "     step")
    for i in range(4, 48):
        print("%4d " % i + " ".join("%8d" % (t[i, e] - t0 if t[i, e] else -1) for e in range(len(NAMES)))
              + " %8d" % (t[i, 0] - t[i - 1, 0]))


if __name__ == "__main__":
    main()
