"""Timeline of the GEMM core on one CTA (developer tool; needs a B200 and a trace build).

    TABATTN_TRACE=1 python -m paper_2606_03681_b200.build --force
    python -m paper_2606_03681_b200.trace_gemm [qkv|up|gg]
    python -m paper_2606_03681_b200.build --force          # back to the shipped library

`qkv`: the QKV projection of the attention sub-block (688,128 cells, e = 256: K = 256, N = 768 into three tensors);
`up`: the MLP up-projection (K = 256, N = 768, two outputs); `gg`: du = (dy W2) o gelu'(u) of the MLP backward
(K = 256, N = 768, auxiliary tile u).  Prints, for row tiles 2..41 of CTA 0, the clock64() stamps
(relative to the first) of the events named in csrc/gemm_tc.cu (TR(...)): producer (loads start, last load issued), MMA
warp (first k-block landed, MMAs issued), first epilogue warp (accumulator complete, its staging part written, all
warps done, store issued, staging read; a second group of four for the second output of `up`), and the tile-to-tile
difference of the first column.
"""
import ctypes
import sys

import torch

import paper_2606_03681_b200 as tab

NAMES = ["loads", "loaded", "kb0", "mmaIss", "accFull", "stg0", "all0", "store0", "read0", "stg1", "all1", "store1", "read1"]


def main():
    which = sys.argv[1] if len(sys.argv) > 1 else "qkv"
    if not hasattr(tab.lib(), "tabattn_debug_set_trace_gemm"):
        raise SystemExit("libtabattn.so was built without TABATTN_TRACE=1")
    dev = torch.device("cuda", 0)
    g = torch.Generator(device=dev)
    g.manual_seed(7)
    B, R, C, H, dh, hid = 8, 4096, 21, 4, 64, 768
    e, cells = H * dh, B * R * C
    bf = torch.bfloat16
    x = torch.randn((B, R, C, e), generator=g, device=dev, dtype=torch.float32).to(bf)
    gain = torch.ones(e, device=dev, dtype=bf)
    if which == "qkv":
        wqkv = (torch.randn((3 * e, e), generator=g, device=dev) * e ** -0.5).to(bf)
        wo = (torch.randn((e, e), generator=g, device=dev) * e ** -0.5).to(bf)
        nt = torch.full((B,), 3072, dtype=torch.int32, device=dev)
        run = lambda: tab.tabattn_attn_block_fwd(0, x, gain, wqkv, wo, H, nt, None, 1.0)
    else:
        w1 = (torch.randn((hid, e), generator=g, device=dev) * e ** -0.5).to(bf)
        w2 = (torch.randn((e, hid), generator=g, device=dev) * hid ** -0.5).to(bf)
        if which == "up":
            run = lambda: tab.tabattn_mlp_fwd(x.view(cells, e), gain, w1, w2, 1.0)
        else:
            _, saved = tab.tabattn_mlp_fwd(x.view(cells, e), gain, w1, w2, 1.0)
            dy = torch.randn((cells, e), generator=g, device=dev, dtype=torch.float32).to(bf)
            run = lambda: tab.tabattn_mlp_bwd(x.view(cells, e), gain, w1, w2, saved, dy, 1.0)
    for _ in range(3):
        run()
    trace = torch.zeros(64 * 16, dtype=torch.int64, device=dev)
    torch.cuda.synchronize()
    tab.lib().tabattn_debug_set_trace_gemm(ctypes.c_void_p(trace.data_ptr()))
    run()
    torch.cuda.synchronize()
    t = trace.cpu().numpy().reshape(64, 16)
    t0 = t[t > 0].min()
    n = len(NAMES) if which == "up" else 9
    print("tile " + " ".join("%8s" % s for s in NAMES[:n]) + "     step")
    for i in range(2, 42):
        print("%4d " % i + " ".join("%8d" % (t[i, k] - t0 if t[i, k] else -1) for k in range(n))
              + " %8d" % (t[i, 0] - t[i - 1, 0]))


if __name__ == "__main__":
    main()
