"""fp64 oracle of the forward-only evaluation path.

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / ``--impl reference`` leg may import this module.  It shares nothing with
paper_2606_03681_b200/ and never imports it.

What is computed (PAPER.md:L65 evaluation tables of <= 1000 rows x <= 100 features, 800 train /
200 test rows per fold; "the test-row outputs are sliced out"; PAPER.md:L294 thinking
rows "count as part of the train portion"): the attention output O for the query rows [row0, row1)
of every table only, with no log-sum-exp saved.  It is the plain definition (SURVEY.md §8(c) steps
1-4) written out in numpy float64, one (table, sequence, head) at a time, with a library matmul as
the only primitive: scores, row maximum, exponentials, row sums, weights, weighted values.

  item:     for every valid column c and head h, query rows i in [row0, row1) attend to the key
            rows j in [0, n_train[b]) of the same column (train and test queries alike).
  feature:  for every row r in [row0, row1) and head h, the valid columns attend to one another.

Invalid columns give O = 0.  Pinned (tests/test_oracle_eval.py) against the independently written
C oracle's full forward (equal to its slice), the closed-form golden fixture, the single-key and
identical-key closed forms, and the row-range / train-only invariances.
"""
import numpy as np


def _widen(a):
    """uint16 bf16 bit patterns -> float64 (exact); float64 passes through."""
    a = np.asarray(a)
    if a.dtype == np.uint16:
        return (a.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
    if a.dtype != np.float64:
        raise TypeError("oracle inputs must be uint16 (bf16 bits) or float64")
    return a


def _softmax_av(q, k, v, scale):
    """softmax(q k^T scale) v for one sequence: q [Lq,dh], k,v [Lk,dh] -> [Lq,dh]."""
    s = (q @ k.T) * scale                       # step 1
    m = s.max(axis=1, keepdims=True)            # step 2
    e = np.exp(s - m)
    p = e / e.sum(axis=1, keepdims=True)
    return p @ v                                # step 3


def item_fwd_infer(Q, K, V, n_train, row0, row1, col_valid=None, scale=0.0):
    """O for query rows [row0,row1): returns float64 [B, row1-row0, C, H, dh]."""
    Q, K, V = _widen(Q), _widen(K), _widen(V)
    B, R, C, H, dh = Q.shape
    if not (0 <= row0 < row1 <= R):
        raise ValueError("row range")
    sc = scale if scale > 0 else 1.0 / np.sqrt(dh)
    O = np.zeros((B, row1 - row0, C, H, dh))
    for b in range(B):
        n = int(n_train[b])
        if not (1 <= n <= R):
            raise ValueError("n_train")
        for c in range(C):
            if col_valid is not None and not col_valid[b][c]:
                continue                        # step 4: invalid column -> zeros
            for h in range(H):
                O[b, :, c, h, :] = _softmax_av(Q[b, row0:row1, c, h, :], K[b, :n, c, h, :], V[b, :n, c, h, :], sc)
    return O


def feature_fwd_infer(Q, K, V, row0, row1, col_valid=None, scale=0.0):
    """O for table rows [row0,row1): returns float64 [B, row1-row0, C, H, dh]."""
    Q, K, V = _widen(Q), _widen(K), _widen(V)
    B, R, C, H, dh = Q.shape
    if not (0 <= row0 < row1 <= R):
        raise ValueError("row range")
    sc = scale if scale > 0 else 1.0 / np.sqrt(dh)
    O = np.zeros((B, row1 - row0, C, H, dh))
    for b in range(B):
        cols = np.arange(C) if col_valid is None else np.flatnonzero(np.asarray(col_valid[b]))
        if cols.size == 0:
            continue
        for r in range(row0, row1):
            for h in range(H):
                O[b, r - row0, cols, h, :] = _softmax_av(Q[b, r, cols, h, :], K[b, r, cols, h, :],
                                                         V[b, r, cols, h, :], sc)
    return O
