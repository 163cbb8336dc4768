"""LayerGraph (paper_2606_03681_b200/layer.py): the four C-ABI calls of a layer captured in a CUDA graph give, on
replay, bit for bit what the direct calls give -- on an unmasked and on a masked shape (whose a0 prep kernels are part
of the graph), also after the inputs were overwritten in place (the graph holds pointers, not values)."""
import numpy as np
import pytest
import torch

from workloads import TabShape, draw_structure, get_config, make_call_inputs

pytestmark = pytest.mark.gpu

CASES = [get_config("tiny"),
         TabShape("graph_masked", 57, B=3, R=260, C=11, H=6, dh=32, n_train=200, mask="prefix",
                  valid_features=(3, 10), ragged_n_train=(100, 250))]


def _results(buf):
    return [buf.O_f, buf.LSE_f, buf.O_i, buf.LSE_i] + list(buf.grads_f) + list(buf.grads_i)


def _same(a, b):
    if a.dtype == torch.bfloat16:
        return torch.equal(a.view(torch.int16), b.view(torch.int16))
    return torch.equal(a, b)


@pytest.mark.parametrize("cfg", CASES, ids=lambda c: c.name)
def test_graph_replay_equals_direct_calls(cfg):
    import paper_2606_03681_b200 as tab
    dev = torch.device("cuda", 0)
    nt_h, cv_h = draw_structure(cfg)
    nt = torch.from_numpy(np.ascontiguousarray(nt_h, dtype=np.int32)).to(dev)
    cv = torch.from_numpy(np.ascontiguousarray(cv_h, dtype=np.uint8)).to(dev) if cv_h is not None else None
    feat = make_call_inputs(cfg, "feature", 0, device=dev)
    item = make_call_inputs(cfg, "item", 0, device=dev)
    shape = (cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh)
    ref_buf = tab.LayerBuffers(*shape, device=dev)
    g_buf = tab.LayerBuffers(*shape, device=dev)
    graph = tab.LayerGraph(feat, item, nt, cv, g_buf, n_train_host=nt_h)
    assert graph.kernels_per_replay >= 5          # feature fwd/bwd, item fwd, dQ pass, dK/dV pass (+ prep kernels)
    for round_ in range(2):
        if round_ == 1:                            # new values behind the same pointers
            for d in (feat, item):
                for k in d:
                    d[k].copy_(torch.flip(d[k], dims=(1,)))
        for t in _results(g_buf):
            t.view(torch.int16 if t.dtype == torch.bfloat16 else torch.int32).fill_(-1)      # NaN patterns
        n0 = tab.launch_count()
        graph.replay()
        torch.cuda.synchronize()
        assert tab.launch_count() == n0            # a replay makes no host-side launches
        tab.layer_fwd_bwd(feat, item, nt, cv, ref_buf, n_train_host=nt_h)
        torch.cuda.synchronize()
        for i, (a, b) in enumerate(zip(_results(g_buf), _results(ref_buf))):
            assert torch.isfinite(b.float()).all(), "direct result %d not finite" % i
            assert _same(a, b), "round %d: result %d differs between graph replay and direct calls" % (round_, i)


def test_mlp_block_and_newton_schulz_replay_equal_direct_calls():
    """The GEMM kernels are launched with programmatic dependent launch; a captured chain of them (MLP sub-block forward
    and backward, Newton-Schulz) must replay to the bits of the direct calls."""
    import paper_2606_03681_b200 as tab
    dev = torch.device("cuda", 0)
    g = torch.Generator(device=dev)
    g.manual_seed(5)
    cells, e, hid = 1500, 256, 768
    bf = torch.bfloat16
    x = torch.randn((cells, e), generator=g, device=dev).to(bf)
    dy = torch.randn((cells, e), generator=g, device=dev).to(bf)
    gain = (1.0 + 0.1 * torch.randn((e,), generator=g, device=dev)).to(bf)
    w1 = (torch.randn((hid, e), generator=g, device=dev) * e ** -0.5).to(bf)
    w2 = (torch.randn((e, hid), generator=g, device=dev) * hid ** -0.5).to(bf)
    G = (torch.randn((6, 128, 256), generator=g, device=dev) * 0.02).to(bf)

    def run():
        y, saved = tab.tabattn_mlp_fwd(x, gain, w1, w2, 0.9)
        grads = tab.tabattn_mlp_bwd(x, gain, w1, w2, saved, dy, 0.9)
        X = tab.tabattn_newton_schulz(G, 5)
        return (y,) + tuple(grads) + (X,)

    want = run()
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            got = run()
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(2):
        for t in got:
            t.zero_()
        graph.replay()
        torch.cuda.synchronize()
        for i, (a, b) in enumerate(zip(got, want)):
            assert _same(a, b), "result %d differs between graph replay and direct calls" % i
