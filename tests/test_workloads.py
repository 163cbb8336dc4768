"""Seeded input recipe: shapes, structure draws, bf16 conversion."""
import numpy as np

from workloads import (CONFIGS, get_config, draw_structure, make_call_inputs, fig6_shape,
                       f32_to_bf16_bits, bf16_bits_to_f32)


def test_config_table_matches_baseline_json():
    shapes = {c.name: (c.B, c.R, c.C, c.H, c.dh, c.n_train) for c in CONFIGS}
    assert shapes["tiny"] == (2, 64, 6, 2, 16, 48)
    assert shapes["base"] == (32, 1024, 11, 6, 32, 768)
    assert shapes["feature_heavy"][:5] == (16, 512, 101, 6, 32) and shapes["feature_heavy"][5] == 384
    assert shapes["long_item"] == (8, 4096, 21, 4, 64, 3072)
    assert shapes["ragged"][:5] == (16, 2048, 51, 6, 32)
    assert get_config("ragged").layers == 12
    f = fig6_shape()
    assert (f.R, f.n_train, f.C, f.d, f.H) == (116, 96, 23, 256, 4)


def test_structure_draws():
    nt, valid = draw_structure(get_config("base"))
    assert valid is None and np.all(nt == 768) and nt.dtype == np.int32
    cfg = get_config("feature_heavy")
    nt, valid = draw_structure(cfg)
    assert valid.shape == (16, 101) and valid.dtype == np.uint8
    assert np.all(valid[:, 100] == 1)
    nfeat = valid[:, :100].sum(axis=1)
    assert nfeat.min() >= 20 and nfeat.max() <= 100
    # arbitrary subset, not a prefix
    assert any(not np.all(valid[b, :nfeat[b]] == 1) for b in range(16))
    cfg = get_config("ragged")
    nt, valid = draw_structure(cfg)
    assert nt.min() >= 512 and nt.max() <= 1536 and len(set(nt.tolist())) > 1
    nfeat = valid[:, :50].sum(axis=1)
    assert nfeat.min() >= 10 and nfeat.max() <= 50 and np.all(valid[:, 50] == 1)
    for b in range(cfg.B):
        assert np.all(valid[b, :nfeat[b]] == 1) and np.all(valid[b, nfeat[b]:50] == 0)
    # seeded: same draw twice
    nt2, valid2 = draw_structure(cfg)
    assert np.array_equal(nt, nt2) and np.array_equal(valid, valid2)


def test_tensors_seeded_and_distinct():
    cfg = get_config("tiny")
    a = make_call_inputs(cfg, "feature")
    b = make_call_inputs(cfg, "feature")
    c = make_call_inputs(cfg, "item")
    for k in ("Q", "K", "V", "dO"):
        assert a[k].dtype == np.uint16 and a[k].shape == (2, 64, 6, 2, 16)
        assert np.array_equal(a[k], b[k])
        assert not np.array_equal(a[k], c[k])
    x = bf16_bits_to_f32(a["Q"])
    assert abs(x.mean()) < 0.05 and abs(x.std() - 1) < 0.05


def test_feature_heavy_q_is_sharpened_and_ragged_is_projected():
    cfg = get_config("feature_heavy").scaled(B=2, R=8)
    x = make_call_inputs(cfg, "feature")
    assert abs(bf16_bits_to_f32(x["Q"]).std() - 4) < 0.2
    assert abs(bf16_bits_to_f32(x["K"]).std() - 1) < 0.1
    cfg = get_config("ragged").scaled(B=1, R=16, C=5)
    x = make_call_inputs(cfg, "item", layer=3)
    y = make_call_inputs(cfg, "item", layer=4)
    assert abs(bf16_bits_to_f32(x["Q"]).std() - 1) < 0.2     # X~N(0,1), W~N(0,1/d) -> unit variance
    assert not np.array_equal(x["Q"], y["Q"])


def test_bf16_round_to_nearest_even():
    f = np.array([1.0, 1.00390625, 1.01171875, -2.5, 0.0, np.inf], np.float32)
    # 1.00390625 = 1 + 2^-8 is a tie between 1.0 (even mantissa) and 1.0078125 -> rounds to 1.0
    # 1.01171875 = 1 + 3*2^-8 is a tie between 1.0078125 (odd) and 1.015625 (even) -> 1.015625
    bits = f32_to_bf16_bits(f)
    back = bf16_bits_to_f32(bits)
    assert back.tolist() == [1.0, 1.0, 1.015625, -2.5, 0.0, np.inf]
    assert np.isnan(bf16_bits_to_f32(f32_to_bf16_bits(np.array([np.nan], np.float32))))[0]
    torch = __import__("pytest").importorskip("torch")
    x = np.random.default_rng(0).standard_normal(4096).astype(np.float32)
    t = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(f32_to_bf16_bits(x), t)
