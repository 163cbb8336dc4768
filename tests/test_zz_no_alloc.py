"""tabattn_item_fwd_noalloc (include/tabattn.h): the item forward whose scratch -- the a0 column list of a masked
call -- is a `static __device__` array inside the library, for callers that cannot allocate.  Checked against the
existing path (tabattn_item_fwd with a caller workspace) on two calls in a row with DIFFERENT masks, so that what the
first call left in the shared array would show in the second.  Named test_zz_* so that pytest collects it last.
"""
import numpy as np
import pytest
import torch

from helpers import FWD_REL_L2, LSE_TOL, rel_l2
from workloads import TabShape, draw_structure, make_call_inputs

pytestmark = pytest.mark.gpu


def _case(cfg):
    import gpu_util
    n_train, col_valid = draw_structure(cfg)
    inp = make_call_inputs(cfg, "item")
    d = [gpu_util.to_dev(inp[k]) for k in ("Q", "K", "V")]
    nt = torch.from_numpy(np.ascontiguousarray(n_train, dtype=np.int32)).cuda()
    cv = torch.from_numpy(np.ascontiguousarray(col_valid, dtype=np.uint8)).cuda()
    return d, nt, cv, n_train, col_valid


def _compare(tag, got, want, col_valid):
    import gpu_util
    O, LSE = got
    O_ref, LSE_ref = want
    o, o_ref = gpu_util.to_f64(O), gpu_util.to_f64(O_ref)
    err = rel_l2(o, o_ref)
    assert np.isfinite(o).all() and err <= FWD_REL_L2, "%s: O rel-L2 %.3e" % (tag, err)
    lse, lse_ref = LSE.cpu().numpy().astype(np.float64), LSE_ref.cpu().numpy().astype(np.float64)
    assert np.isfinite(lse).all() and np.abs(lse - lse_ref).max() <= LSE_TOL, "%s: LSE" % tag
    # same kernels on the same inputs, no atomics: the two paths agree bit for bit
    assert torch.equal(O.view(torch.int16), O_ref.view(torch.int16)), "%s: O bits differ" % tag
    assert torch.equal(LSE, LSE_ref), "%s: LSE bits differ" % tag
    # invalid columns are +0 in both
    inv = np.broadcast_to((np.asarray(col_valid) == 0)[:, None, :, None, None], o.shape)
    if inv.any():
        assert gpu_util.is_pos_zero(gpu_util.to_bits(O)[inv]), "%s: invalid columns are not +0" % tag


def test_noalloc_matches_workspace_path_twice():
    import paper_2606_03681_b200 as tab
    cases = [TabShape("noalloc_prefix", 91, B=3, R=300, C=11, H=6, dh=32, n_train=200, mask="prefix",
                      valid_features=(3, 10), ragged_n_train=(130, 260)),
             TabShape("noalloc_subset", 92, B=2, R=200, C=21, H=2, dh=64, n_train=150, mask="subset",
                      valid_features=(4, 20))]
    for cfg in cases:          # two calls in a row through the shared scratch, different masks and shapes
        (Q, K, V), nt, cv, n_train, col_valid = _case(cfg)
        B, R, C, H, dh = Q.shape
        O = torch.full_like(Q, float("nan"))
        LSE = torch.full((B, C, H, R), float("nan"), dtype=torch.float32, device=Q.device)
        got = tab.tabattn_item_fwd_noalloc(Q, K, V, nt, cv, n_train_host=n_train, O=O, LSE=LSE)
        torch.cuda.synchronize()
        want = tab.tabattn_item_fwd(Q, K, V, nt, cv, n_train_host=n_train)
        torch.cuda.synchronize()
        _compare(cfg.name, got, want, col_valid)
    # and the first case again, after the second one overwrote the scratch
    cfg = cases[0]
    (Q, K, V), nt, cv, n_train, col_valid = _case(cfg)
    got = tab.tabattn_item_fwd_noalloc(Q, K, V, nt, cv, n_train_host=n_train)
    want = tab.tabattn_item_fwd(Q, K, V, nt, cv, n_train_host=n_train)
    torch.cuda.synchronize()
    _compare(cfg.name + "/again", got, want, col_valid)


def test_noalloc_unmasked_and_limit():
    import paper_2606_03681_b200 as tab
    # unmasked: no scratch at all, same results
    cfg = TabShape("noalloc_plain", 93, B=1, R=384, C=3, H=2, dh=64, n_train=300)
    import gpu_util
    n_train, _ = draw_structure(cfg)
    inp = make_call_inputs(cfg, "item")
    Q, K, V = (gpu_util.to_dev(inp[k]) for k in ("Q", "K", "V"))
    nt = torch.from_numpy(np.ascontiguousarray(n_train, dtype=np.int32)).cuda()
    O, LSE = tab.tabattn_item_fwd_noalloc(Q, K, V, nt, None, n_train_host=n_train)
    O_ref, LSE_ref = tab.tabattn_item_fwd(Q, K, V, nt, None, n_train_host=n_train)
    torch.cuda.synchronize()
    assert rel_l2(gpu_util.to_f64(O), gpu_util.to_f64(O_ref)) <= FWD_REL_L2
    assert (LSE - LSE_ref).abs().max().item() <= LSE_TOL
    # a masked call with more column pairs than the built-in scratch holds is refused, nothing is launched
    B, C = 600, 128
    assert B * C > tab.NOALLOC_MAX_BC
    Q = torch.zeros((B, 1, C, 1, 16), dtype=torch.bfloat16, device="cuda")
    nt = torch.ones(B, dtype=torch.int32, device="cuda")
    cv = torch.ones((B, C), dtype=torch.uint8, device="cuda")
    n0 = tab.launch_count()
    with pytest.raises(tab.TabattnError) as e:
        tab.tabattn_item_fwd_noalloc(Q, Q.clone(), Q.clone(), nt, cv)
    assert e.value.status == tab.ERR_WORKSPACE and tab.launch_count() == n0
    # the same shape without a mask needs no scratch and runs
    tab.tabattn_item_fwd_noalloc(Q, Q.clone(), Q.clone(), nt, None)
    torch.cuda.synchronize()
