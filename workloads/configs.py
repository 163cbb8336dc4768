"""The five BASELINE.json configs as shapes + seeded structure draws.

Source of every number here: /root/repo/BASELINE.json ``configs`` (restated in
SURVEY.md §8(d)); the readings c15/c16/c19 of SURVEY.md §8(c) fix what the json
leaves open.  These stand in for the paper's workloads: TabICL-prior tables of
1000 rows x <=20 features, subsampled TabArena evaluation tables
of <=1000 rows x <=100 features, batch>1 with unequal tables
(PAPER.md:L322).  The real data are not used anywhere.
"""
from dataclasses import dataclass, replace
from typing import Optional, Tuple

import numpy as np


@dataclass(frozen=True)
class TabShape:
    name: str
    seed: int          # = config index (SURVEY.md §8(d) "Seeding")
    B: int             # tables
    R: int             # rows (thinking + train + test)
    C: int             # columns (features + target)
    H: int             # heads
    dh: int            # head dim
    n_train: int       # default train-row count (ragged: ignored, drawn per table)
    mask: str = "none"        # "none" | "subset" (Feature-heavy, c15) | "prefix" (Ragged, c16)
    q_scale: float = 1.0      # Feature-heavy multiplies Q by 4 before bf16 rounding
    layers: int = 1           # Ragged: 12 layers chained
    ragged_n_train: Optional[Tuple[int, int]] = None   # inclusive range for per-table n_train
    valid_features: Optional[Tuple[int, int]] = None   # inclusive range of valid feature count
    projected: bool = False   # Ragged: Q,K,V = bf16(X @ W), c17

    @property
    def d(self) -> int:
        return self.H * self.dh

    @property
    def cells(self) -> int:
        return self.B * self.R * self.C

    def scaled(self, **kw) -> "TabShape":
        """A smaller copy of this shape (same structure rules) for CPU-sized tests."""
        return replace(self, **kw)


CONFIGS = (
    TabShape("tiny", 0, B=2, R=64, C=6, H=2, dh=16, n_train=48),
    TabShape("base", 1, B=32, R=1024, C=11, H=6, dh=32, n_train=768),
    TabShape("feature_heavy", 2, B=16, R=512, C=101, H=6, dh=32, n_train=384,
             mask="subset", q_scale=4.0, valid_features=(20, 100)),
    TabShape("long_item", 3, B=8, R=4096, C=21, H=4, dh=64, n_train=3072),
    TabShape("ragged", 4, B=16, R=2048, C=51, H=6, dh=32, n_train=1024,
             mask="prefix", layers=12, ragged_n_train=(512, 1536),
             valid_features=(10, 50), projected=True),
)
CONFIG_NAMES = tuple(c.name for c in CONFIGS)


def get_config(name_or_index) -> TabShape:
    if isinstance(name_or_index, int):
        return CONFIGS[name_or_index]
    for c in CONFIGS:
        if c.name == name_or_index:
            return c
    raise KeyError(name_or_index)


def fig6_shape() -> TabShape:
    """The one odd shape the paper prints: Fig. 6 has
    16 thinking + 80 train + 20 test = 116 rows, n_train = 96; task jm1 has 22
    features -> C = 23; Record-6 width (256, 4 heads)."""
    return TabShape("fig6", 6, B=1, R=116, C=23, H=4, dh=64, n_train=96)


def draw_structure(cfg: TabShape):
    """Seeded draw of (n_train int32[B], col_valid uint8[B,C] or None).

    Order of draws with ``numpy.random.default_rng(cfg.seed)``:
    n_train (ragged only), then valid-feature counts, then (subset masks) one
    ``permutation(C-1)`` per table.  The target column C-1 is always valid.
    """
    rng = np.random.default_rng(cfg.seed)
    if cfg.ragged_n_train is not None:
        lo, hi = cfg.ragged_n_train
        lo, hi = min(lo, cfg.R), min(hi, cfg.R)
        n_train = rng.integers(lo, hi + 1, size=cfg.B).astype(np.int32)
    else:
        n_train = np.full(cfg.B, min(cfg.n_train, cfg.R), dtype=np.int32)
    if cfg.mask == "none":
        return n_train, None
    nfeat = cfg.C - 1
    lo, hi = cfg.valid_features
    lo, hi = min(lo, nfeat), min(hi, nfeat)
    counts = rng.integers(lo, hi + 1, size=cfg.B)
    valid = np.zeros((cfg.B, cfg.C), dtype=np.uint8)
    valid[:, cfg.C - 1] = 1
    for b in range(cfg.B):
        if cfg.mask == "subset":
            cols = rng.permutation(nfeat)[: counts[b]]
            valid[b, cols] = 1
        elif cfg.mask == "prefix":
            valid[b, : counts[b]] = 1
        else:
            raise ValueError(cfg.mask)
    return n_train, valid
