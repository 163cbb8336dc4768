"""GPU-vs-oracle parity of the forward-only evaluation path (tabattn_*_fwd_infer) through
the C ABI.  Needs a B200.  The oracle is oracle/eval_ref.py (numpy fp64, the definition restricted to a row
range); tolerances are the forward ones of BASELINE.json (O rel-L2 <= 5e-3, max-abs <= 1e-2 max|V|)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from workloads import TabShape, draw_structure, make_call_inputs, bf16_bits_to_f64  # noqa: E402
from helpers import FWD_REL_L2, FWD_MAXABS_FRAC, rel_l2  # noqa: E402

SENTINEL = np.uint16(0x4A4A)   # bf16 pattern the output buffer is pre-filled with: rows outside the range keep it


def _check(axis, cfg, row0, row1, poison=True):
    import torch
    import gpu_util as gu
    import paper_2606_03681_b200 as tab
    from oracle import eval_ref
    n_train, col_valid = draw_structure(cfg)
    inp = make_call_inputs(cfg, axis)
    Q, K, V = inp["Q"], inp["K"], inp["V"]
    if axis == "item":
        ref = eval_ref.item_fwd_infer(Q, K, V, n_train, row0, row1, col_valid)
    else:
        ref = eval_ref.feature_fwd_infer(Q, K, V, row0, row1, col_valid)
    if poison:
        nan = np.uint16(0x7FC0)
        Q, K, V = Q.copy(), K.copy(), V.copy()
        if col_valid is not None:
            bad = ~np.asarray(col_valid).astype(bool)
            for t in (Q, K, V):
                t[np.broadcast_to(bad[:, None, :], t.shape[:3])] = nan
        if axis == "item":
            for b in range(cfg.B):
                K[b, n_train[b]:] = nan
                V[b, n_train[b]:] = nan
    d = [gu.to_dev(x) for x in (Q, K, V)]
    cv = torch.from_numpy(np.ascontiguousarray(col_valid, dtype=np.uint8)).cuda() if col_valid is not None else None
    O = torch.full(d[0].shape, 0, dtype=torch.int16, device="cuda").fill_(int(SENTINEL)).view(torch.bfloat16)
    if axis == "item":
        nt = torch.from_numpy(n_train).cuda()
        tab.tabattn_item_fwd_infer(d[0], d[1], d[2], nt, row0, row1, cv, n_train_host=n_train, O=O)
        full, _ = tab.tabattn_item_fwd(d[0], d[1], d[2], nt, cv, n_train_host=n_train)
    else:
        tab.tabattn_feature_fwd_infer(d[0], d[1], d[2], row0, row1, cv, O=O)
        full, _ = tab.tabattn_feature_fwd(d[0], d[1], d[2], cv)
    torch.cuda.synchronize()
    bits = gu.to_bits(O)
    # rows outside the range are not touched
    assert np.all(bits[:, :row0] == SENTINEL) and np.all(bits[:, row1:] == SENTINEL)
    # on the range: bit-identical to the training forward (tabattn.h), +0 at invalid columns, parity with the oracle
    got = bits[:, row0:row1]
    assert np.array_equal(got, gu.to_bits(full)[:, row0:row1])
    colv = np.ones((cfg.B, cfg.C), bool) if col_valid is None else np.asarray(col_valid).astype(bool)
    mask = np.broadcast_to(colv[:, None, :], got.shape[:3])
    assert np.all(got[~mask] == 0) and np.all(ref[~mask] == 0.0)
    g = bf16_bits_to_f64(got)
    assert np.isfinite(g).all()
    e = rel_l2(g[mask], ref[mask])
    assert e <= FWD_REL_L2, "%s O rel-L2 %.3e" % (cfg.name, e)
    vmax = np.abs(bf16_bits_to_f64(inp["V"])).max()
    assert np.abs(g[mask] - ref[mask]).max() <= FWD_MAXABS_FRAC * vmax
    return e


CASES = [
    # name, B, R, C, H, dh, n_train, mask, (row0, row1)
    ("test_chunk_dh64", 2, 300, 5, 2, 64, 200, "none", (200, 300)),
    ("test_chunk_dh32_masked", 3, 260, 12, 3, 32, 130, "prefix", (130, 260)),
    ("one_row", 1, 140, 3, 2, 32, 100, "none", (139, 140)),
    ("inner_chunk_unaligned", 2, 700, 4, 2, 16, 333, "none", (401, 659)),   # spans three 256-row items
    ("whole_range", 2, 130, 21, 4, 64, 90, "none", (0, 130)),
    ("wide_masked", 2, 40, 101, 2, 32, 30, "subset", (7, 33)),
]


@pytest.mark.parametrize("axis", ["feature", "item"])
@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_infer_parity(case, axis):
    name, B, R, C, H, dh, n, mask, (row0, row1) = case
    vf = None if mask == "none" else (max(1, (C - 1) // 3), C - 1)
    cfg = TabShape(name, 40 + len(name), B=B, R=R, C=C, H=H, dh=dh, n_train=n, mask=mask, valid_features=vf)
    _check(axis, cfg, row0, row1)


@pytest.mark.parametrize("axis", ["feature", "item"])
def test_eval_shape_last_block_test_rows(axis):
    """The evaluation shape (Table 5): 24 thinking + 800 train + 200 test rows, 100 features +
    target, (256, 4 heads); the last block needs the 200 test rows only."""
    cfg = TabShape("eval_1000x100", 5, B=1, R=1024, C=101, H=4, dh=64, n_train=824)
    _check(axis, cfg, 824, 1024, poison=True)


def test_infer_argument_checks():
    import torch
    import paper_2606_03681_b200 as tab
    q = torch.zeros((1, 8, 2, 1, 16), dtype=torch.bfloat16, device="cuda")
    nt = torch.tensor([4], dtype=torch.int32, device="cuda")
    for r0, r1 in ((-1, 4), (4, 4), (5, 3), (0, 9)):
        with pytest.raises(tab.TabattnError) as e:
            tab.tabattn_item_fwd_infer(q, q.clone(), q.clone(), nt, r0, r1)
        assert e.value.status == tab.ERR_INVALID_ARG
        with pytest.raises(tab.TabattnError) as e:
            tab.tabattn_feature_fwd_infer(q, q.clone(), q.clone(), r0, r1)
        assert e.value.status == tab.ERR_INVALID_ARG
