"""GPU-vs-oracle parity through the C ABI (SURVEY.md §4 tiers T1-T3).  Needs a B200."""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from workloads import (get_config, fig6_shape, draw_structure, make_call_inputs, TabShape,  # noqa: E402
                       f32_to_bf16_bits)


def _gu():
    import gpu_util
    return gpu_util


def _run_case(cfg, axis, n_train=None, col_valid=None, poison=False, what=None):
    gu = _gu()
    nt_draw, cv_draw = draw_structure(cfg)
    n_train = nt_draw if n_train is None else np.asarray(n_train, np.int32)
    col_valid = cv_draw if col_valid is None else col_valid
    inp = make_call_inputs(cfg, axis)
    orc = gu.run_oracle(axis, inp, n_train, col_valid)
    if poison:
        # NaN at every position that must not influence any output (SURVEY.md §8(b) "Values at masked positions")
        nan = np.uint16(0x7FC0)
        inp = {k: v.copy() for k, v in inp.items()}
        if col_valid is not None:
            bad = ~np.asarray(col_valid).astype(bool)
            for k in ("Q", "K", "V", "dO"):
                inp[k][np.broadcast_to(bad[:, None, :], inp[k].shape[:3])] = nan
        if axis == "item":
            for b in range(cfg.B):
                inp["K"][b, n_train[b]:] = nan
                inp["V"][b, n_train[b]:] = nan
    gpu = gu.run_gpu(axis, inp, n_train, col_valid)
    return gu.check_parity(axis, inp, gpu, orc, n_train, col_valid, what or "%s/%s" % (cfg.name, axis))


# ---- T1: full tensors on the small shapes --------------------------------------------------------
@pytest.mark.parametrize("axis", ["feature", "item"])
def test_tiny_config(axis):
    _run_case(get_config("tiny"), axis)


@pytest.mark.parametrize("axis", ["feature", "item"])
def test_fig6_shape(axis):
    # 16 thinking + 80 train + 20 test rows; non-multiple-of-anything
    _run_case(fig6_shape(), axis)


EDGE = [
    # name, B, R, C, H, dh, n_train
    ("one_key", 2, 33, 3, 2, 32, 1),          # single key: O = V_0
    ("no_test_rows", 1, 130, 2, 1, 64, 130),  # n_train = R: plain self-attention, ragged q/k tiles
    ("one_row", 3, 1, 5, 2, 16, 1),
    ("one_col", 2, 70, 1, 3, 32, 40),         # feature attention over a single column
    ("tile_edges", 1, 257, 4, 2, 32, 129),    # one past the 128/256 tile boundaries
    ("tile_exact", 1, 256, 3, 2, 64, 128),
    ("wide_C", 1, 9, 128, 1, 32, 5),          # largest feature-axis length
    ("c17", 2, 40, 17, 2, 32, 30),
    ("c33_dh64", 1, 24, 33, 2, 64, 17),
    # more work items than SMs (several items per persistent CTA), key-block rotation of the dK/dV pass with
    # a non-power-of-two block count, last 64-key chunk split 32 + 12 / 14 + 0 between the column halves
    ("multi_item_dh32", 3, 700, 5, 2, 32, 300),
    ("multi_item_dh64", 4, 520, 5, 2, 64, 270),
    ("dh16_multi_chunk", 2, 300, 3, 2, 16, 200),
    # B*C = 8960 > 8192 cells: the backward kernels read n_train / col_valid from global memory instead of
    # their shared-memory copy (item_tc_common.cuh: Meta)
    ("meta_global_path", 70, 16, 128, 1, 16, 9),
    # many heads (the old prep kernel's per-head scratch overflowed at H >= 34)
    ("many_heads_dh16", 1, 140, 2, 40, 16, 70),
    ("many_heads_dh64", 1, 70, 2, 35, 64, 33),
]


@pytest.mark.parametrize("axis", ["feature", "item"])
@pytest.mark.parametrize("case", EDGE, ids=[e[0] for e in EDGE])
def test_edge_shapes(case, axis):
    name, B, R, C, H, dh, n = case
    cfg = TabShape(name, 100 + EDGE.index(case), B=B, R=R, C=C, H=H, dh=dh, n_train=n)
    _run_case(cfg, axis)


@pytest.mark.parametrize("axis", ["feature", "item"])
def test_ragged_n_train_and_masks_with_nan_poison(axis):
    cfg = TabShape("mini_ragged", 41, B=4, R=300, C=13, H=2, dh=32, n_train=100, mask="prefix",
                   ragged_n_train=(1, 300), valid_features=(1, 12))
    _run_case(cfg, axis, poison=True)
    cfg = TabShape("mini_subset", 42, B=3, R=150, C=37, H=2, dh=32, n_train=97, mask="subset",
                   valid_features=(3, 36), q_scale=4.0)
    _run_case(cfg, axis, poison=True)


@pytest.mark.parametrize("axis", ["feature", "item"])
def test_table_with_no_valid_column(axis):
    cfg = TabShape("dead_table", 43, B=2, R=64, C=5, H=2, dh=32, n_train=40)
    cv = np.ones((2, 5), np.uint8)
    cv[1, :] = 0
    _run_case(cfg, axis, col_valid=cv, poison=True)


@pytest.mark.parametrize("axis", ["feature", "item"])
def test_all_valid_mask_equals_null_mask(axis):
    gu = _gu()
    cfg = TabShape("allvalid", 44, B=2, R=96, C=7, H=2, dh=32, n_train=50)
    nt, _ = draw_structure(cfg)
    inp = make_call_inputs(cfg, axis)
    a = gu.run_gpu(axis, inp, nt, None)
    b = gu.run_gpu(axis, inp, nt, np.ones((2, 7), np.uint8))
    for k in ("O", "dQ", "dK", "dV"):
        assert np.array_equal(gu.to_bits(a[k]), gu.to_bits(b[k]))


@pytest.mark.parametrize("axis", ["feature", "item"])
def test_run_to_run_bitwise_determinism(axis):
    gu = _gu()
    cfg = get_config("base").scaled(B=2, R=512, n_train=300)
    nt, cv = draw_structure(cfg)
    inp = make_call_inputs(cfg, axis)
    a = gu.run_gpu(axis, inp, nt, cv)
    b = gu.run_gpu(axis, inp, nt, cv)
    for k in ("O", "dQ", "dK", "dV"):
        assert np.array_equal(gu.to_bits(a[k]), gu.to_bits(b[k])), k
    assert np.array_equal(a["LSE"].cpu().numpy(), b["LSE"].cpu().numpy())


def test_zero_dO_on_train_rows_item():
    # only test-row outputs feed the loss -> dO = 0 on train rows at the last layer
    gu = _gu()
    cfg = TabShape("dO_test_only", 45, B=2, R=200, C=4, H=2, dh=32, n_train=150)
    nt, cv = draw_structure(cfg)
    inp = make_call_inputs(cfg, "item")
    inp["dO"][:, :150] = 0
    orc = gu.run_oracle("item", inp, nt, cv)
    gpu = gu.run_gpu("item", inp, nt, cv)
    gu.check_parity("item", inp, gpu, orc, nt, cv, "dO_test_only")
    assert gu.is_pos_zero(gu.to_bits(gpu["dQ"])[:, :150] & np.uint16(0x7FFF))


def test_custom_softmax_scale():
    gu = _gu()
    cfg = TabShape("scale", 46, B=1, R=80, C=6, H=2, dh=32, n_train=60)
    nt, cv = draw_structure(cfg)
    for axis in ("feature", "item"):
        inp = make_call_inputs(cfg, axis)
        orc = gu.run_oracle(axis, inp, nt, cv, scale=0.31)
        gpu = gu.run_gpu(axis, inp, nt, cv, scale=0.31)
        gu.check_parity(axis, inp, gpu, orc, nt, cv, "scale/" + axis)


# ---- T2: scaled-down copies of the big configs (several tiles + ragged tails), full tensors -------
SCALED = [
    ("base", dict(B=2, R=384, n_train=288)),
    ("feature_heavy", dict(B=2, R=40, n_train=30)),
    ("long_item", dict(B=1, R=640, C=3, n_train=480)),
    ("ragged", dict(B=3, R=400, ragged_n_train=(100, 300))),
]


@pytest.mark.parametrize("axis", ["feature", "item"])
@pytest.mark.parametrize("name,kw", SCALED, ids=[s[0] for s in SCALED])
def test_scaled_configs(name, kw, axis):
    _run_case(get_config(name).scaled(**kw), axis, poison=True)


# ---- the pipelined host path (layer_fwd_bwd_host) must give the device path's bits -------------------
def test_host_pipeline_matches_device_path():
    import torch
    import paper_2606_03681_b200 as tab
    cfg = get_config("ragged").scaled(B=5, R=200, ragged_n_train=(40, 150))
    nt_h, cv_h = draw_structure(cfg)
    dev = torch.device("cuda", 0)
    nt = torch.from_numpy(nt_h).to(dev)
    cv = torch.from_numpy(cv_h).to(dev) if cv_h is not None else None
    L = {ax: make_call_inputs(cfg, ax, 0, device=dev) for ax in ("feature", "item")}
    ref_buf = tab.LayerBuffers(cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh, device=dev)
    tab.layer_fwd_bwd(L["feature"], L["item"], nt, cv, ref_buf, nt_h)
    torch.cuda.synchronize()
    want = [t.clone() for t in (ref_buf.O_f, ref_buf.O_i) + ref_buf.grads_f + ref_buf.grads_i]
    host = {ax: {k: torch.empty(v.shape, dtype=v.dtype, pin_memory=True).copy_(v) for k, v in L[ax].items()}
            for ax in L}
    stage = {ax: {k: torch.zeros_like(v) for k, v in L[ax].items()} for ax in L}
    out_host = [torch.zeros(want[0].shape, dtype=torch.bfloat16, pin_memory=True) for _ in range(8)]
    buf = tab.LayerBuffers(cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh, device=dev)
    for groups in (1, 3, 4):          # 5 tables: uneven groups too
        for t in out_host:
            t.zero_()
        h2d, d2h = tab.layer_fwd_bwd_host(host["feature"], host["item"], stage["feature"], stage["item"],
                                          out_host, nt, cv, buf, nt_h, groups=groups)
        torch.cuda.synchronize()
        assert h2d == 8 * want[0].numel() * 2 and d2h == 8 * want[0].numel() * 2
        for got, w in zip(out_host, want):
            assert torch.equal(got.view(torch.int16), w.cpu().view(torch.int16)), "groups=%d" % groups


# ---- the library only enqueues on the caller's stream: the four calls can be captured in a CUDA graph ----
def test_layer_is_graph_capturable():
    import torch
    import paper_2606_03681_b200 as tab
    cfg = get_config("base").scaled(B=2, R=300, n_train=200)
    nt_h, cv_h = draw_structure(cfg)
    dev = torch.device("cuda", 0)
    nt = torch.from_numpy(nt_h).to(dev)
    cv = torch.from_numpy(cv_h).to(dev) if cv_h is not None else None
    L = {ax: make_call_inputs(cfg, ax, 0, device=dev) for ax in ("feature", "item")}
    buf = tab.LayerBuffers(cfg.B, cfg.R, cfg.C, cfg.H, cfg.dh, device=dev)
    tab.layer_fwd_bwd(L["feature"], L["item"], nt, cv, buf, nt_h)      # eager (also warms up lazy init)
    torch.cuda.synchronize()
    outs = (buf.O_f, buf.O_i) + buf.grads_f + buf.grads_i
    want = [t.clone() for t in outs]
    for t in outs:
        t.zero_()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            tab.layer_fwd_bwd(L["feature"], L["item"], nt, cv, buf, nt_h)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    for rep in range(2):
        for t in outs:
            t.zero_()
        graph.replay()
        torch.cuda.synchronize()
        for got, w in zip(outs, want):
            assert torch.equal(got.view(torch.int16), w.view(torch.int16)), "replay %d" % rep


# ---- out-of-bounds writes: guard bands (compute-sanitizer is closed on this pool, profiles/r02_sanitizer.md) --------
GUARD = 4096   # bytes of sentinel before and after every output buffer


def _guarded(torch, nbytes):
    """A uint8 buffer [guard | payload | guard] filled with 0xA5; returns (whole, payload view)."""
    whole = torch.full((nbytes + 2 * GUARD,), 0xA5, dtype=torch.uint8, device="cuda")
    return whole, whole[GUARD:GUARD + nbytes]


def _guards_intact(whole):
    return bool((whole[:GUARD] == 0xA5).all()) and bool((whole[-GUARD:] == 0xA5).all())


@pytest.mark.parametrize("axis", ["feature", "item"])
@pytest.mark.parametrize("shape", [("tiny", 2, 64, 6, 2, 16, 48), ("edges", 1, 257, 4, 2, 32, 129),
                                   ("odd64", 2, 131, 23, 2, 64, 77), ("masked", 3, 75, 19, 3, 32, 50)],
                         ids=lambda s: s[0])
def test_no_write_outside_the_output_buffers(shape, axis):
    """Every output and the workspace sit between sentinel bands; the bands must survive fwd + bwd (a write past
    the tensor -- a tile tail, a clipped TMA box, a zero-fill loop -- would land in them)."""
    import torch
    import paper_2606_03681_b200 as tab
    gu = _gu()
    name, B, R, C, H, dh, n = shape
    cfg = TabShape(name, 91, B=B, R=R, C=C, H=H, dh=dh, n_train=n, mask="subset" if name == "masked" else "none",
                   valid_features=(3, C - 1) if name == "masked" else None)
    n_train, col_valid = draw_structure(cfg)
    inp = {k: gu.to_dev(v) for k, v in make_call_inputs(cfg, axis).items()}
    cv = torch.from_numpy(np.ascontiguousarray(col_valid, dtype=np.uint8)).cuda() if col_valid is not None else None
    nt = torch.from_numpy(n_train).cuda()
    cells_b = B * R * C * H * dh * 2
    lse_shape = (B, R, H, C) if axis == "feature" else (B, C, H, R)
    bufs = {k: _guarded(torch, cells_b) for k in ("O", "dQ", "dK", "dV")}
    bufs["LSE"] = _guarded(torch, B * R * C * H * 4)
    shp, _keep = tab.make_shape(inp["Q"], nt, cv)
    need = max(tab.workspace_bytes(shp, op) for op in range(4))
    bufs["ws"] = _guarded(torch, max(need, 16))
    t5 = lambda k: bufs[k][1].view(torch.bfloat16).view(B, R, C, H, dh)
    LSE = bufs["LSE"][1].view(torch.float32).view(lse_shape)
    ws = bufs["ws"][1]
    if axis == "feature":
        tab.tabattn_feature_fwd(inp["Q"], inp["K"], inp["V"], cv, O=t5("O"), LSE=LSE, ws=ws)
        tab.tabattn_feature_bwd(inp["Q"], inp["K"], inp["V"], t5("O"), inp["dO"], LSE, cv, dQ=t5("dQ"), dK=t5("dK"),
                                dV=t5("dV"), ws=ws)
    else:
        tab.tabattn_item_fwd(inp["Q"], inp["K"], inp["V"], nt, cv, O=t5("O"), LSE=LSE, ws=ws)
        tab.tabattn_item_bwd(inp["Q"], inp["K"], inp["V"], t5("O"), inp["dO"], LSE, nt, cv, dQ=t5("dQ"), dK=t5("dK"),
                             dV=t5("dV"), ws=ws)
    torch.cuda.synchronize()
    for k, (whole, payload) in bufs.items():
        assert _guards_intact(whole), "%s/%s: a kernel wrote outside %s" % (name, axis, k)
        if k in ("O", "dQ", "dK", "dV"):
            assert not bool((payload == 0xA5).all()), "%s was not written" % k
