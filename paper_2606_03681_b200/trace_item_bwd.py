"""Timeline of the item backward kernels' score warpgroups on one CTA (developer tool; needs a B200 and a trace build).

    TABATTN_TRACE=1 python -m paper_2606_03681_b200.build --force
    python -m paper_2606_03681_b200.trace_item_bwd [base|long_item|feature_heavy|ragged]
    python -m paper_2606_03681_b200.build --force          # back to the shipped library

Prints, for the first 32 chunk steps of each TMEM set of CTA 0 in the dQ pass and then in the dK/dV pass, the
clock64() stamps (relative to the pass's first one) of the events named in csrc/item_tc_bwd.cu (TR(...)): S / dP
ready, loaded (set released), arithmetic done, P / dS columns free, P / dS stored -- for the warpgroups (set 0, columns
0-31) and (set 1, columns 0-31) -- then, for set 0's chunks, the S / dP issue warp (chunk landed, set free, issued)
the two stamps of warpgroup (0, 0) at the start of an item (item decoded, row statistics read; on the item's first
chunk only), a second stamp right after the first (the cost of a stamp), and the step-to-step difference of the first column.
"""
import ctypes
import sys

import torch

import paper_2606_03681_b200 as tab
from workloads import get_config, draw_structure, make_call_inputs

EV = ["ready", "loaded", "math", "free", "stored"]
NAMES = [e + w for w in ("00", "10") for e in EV] + ["landed", "setFree", "sIssued", "decoded", "stats", "calib"]


def main():
    cfg = get_config(sys.argv[1] if len(sys.argv) > 1 else "base")
    if not hasattr(tab.lib(), "tabattn_debug_set_trace_item_bwd"):
        raise SystemExit("libtabattn.so was built without TABATTN_TRACE=1")
    dev = torch.device("cuda", 0)
    nt_h, cv_h = draw_structure(cfg)
    nt = torch.from_numpy(nt_h).to(dev)
    cv = torch.from_numpy(cv_h).to(dev) if cv_h is not None else None
    f = make_call_inputs(cfg, "item", 0, device=dev)
    O, LSE = tab.tabattn_item_fwd(f["Q"], f["K"], f["V"], nt, cv)
    for _ in range(3):
        tab.tabattn_item_bwd(f["Q"], f["K"], f["V"], O, f["dO"], LSE, nt, cv)
    trace = torch.zeros(64 * 16, dtype=torch.int64, device=dev)
    torch.cuda.synchronize()
    tab.lib().tabattn_debug_set_trace_item_bwd(ctypes.c_void_p(trace.data_ptr()))
    tab.tabattn_item_bwd(f["Q"], f["K"], f["V"], O, f["dO"], LSE, nt, cv)
    torch.cuda.synchronize()
    t = trace.cpu().numpy().reshape(64, 16)
    for name, lo in (("dQ pass", 0), ("dK/dV pass", 32)):
        blk = t[lo:lo + 32]
        t0 = blk[blk > 0].min()
        print(name)
        print("step " + " ".join("%8s" % n for n in NAMES) + "     step")
        for i in range(2, 30):
            print("%4d " % i + " ".join("%8d" % (blk[i, e] - t0 if blk[i, e] else -1) for e in range(len(NAMES)))
                  + " %8d" % (blk[i, 0] - blk[i - 1, 0]))


if __name__ == "__main__":
    main()
