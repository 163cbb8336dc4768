"""Scalar-loop brute force for tiny tables.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A second, deliberately different statement of SURVEY.md §8(c) used only to pin
oracle/tabattn_ref.c: every index is a Python loop over the 5-D arrays, the
softmax is the raw ``exp(s)/sum exp(s)`` (no max subtraction: inputs are tiny),
``LSE = log(sum exp(s))``, and the gradients go through the FULL softmax
Jacobian  dS_ij = sum_k dP_ik * p_ik * (delta_kj - p_ij)  instead of the
``p * (dP - D)`` shortcut the oracle and every flash-style kernel use.
Sizes: B<=2, R<=8, C<=4, H<=2, dh<=4.
"""
import math

import numpy as np


def _keys_feature(b, C, col_valid):
    return [c for c in range(C) if col_valid is None or col_valid[b][c]]


def _attend(qs, ks, vs, gs, scale):
    """qs: list of query vectors; ks, vs: lists of key/value vectors; gs: list of
    upstream-gradient vectors or None.  Returns per-query (o, lse) and, when gs is
    given, (dq list, dk list, dv list)."""
    dh = len(qs[0])
    nq, nk = len(qs), len(ks)
    P = [[0.0] * nk for _ in range(nq)]
    outs, lses = [], []
    for i in range(nq):
        e = []
        for j in range(nk):
            s = 0.0
            for t in range(dh):
                s += qs[i][t] * ks[j][t]
            e.append(math.exp(scale * s))
        z = sum(e)
        o = [0.0] * dh
        for j in range(nk):
            P[i][j] = e[j] / z
            for t in range(dh):
                o[t] += P[i][j] * vs[j][t]
        outs.append(o)
        lses.append(math.log(z))
    if gs is None:
        return outs, lses, None
    dq = [[0.0] * dh for _ in range(nq)]
    dk = [[0.0] * dh for _ in range(nk)]
    dv = [[0.0] * dh for _ in range(nk)]
    for i in range(nq):
        dP = [sum(gs[i][t] * vs[k][t] for t in range(dh)) for k in range(nk)]
        for j in range(nk):
            for t in range(dh):
                dv[j][t] += P[i][j] * gs[i][t]
            dS = 0.0
            for k in range(nk):
                dS += dP[k] * P[i][k] * ((1.0 if k == j else 0.0) - P[i][j])
            for t in range(dh):
                dq[i][t] += scale * dS * ks[j][t]
                dk[j][t] += scale * dS * qs[i][t]
    return outs, lses, (dq, dk, dv)


def feature(Q, K, V, dO=None, col_valid=None, scale=None):
    """Returns O [B,R,C,H,dh], LSE [B,R,H,C] and (dQ,dK,dV) or None."""
    B, R, C, H, dh = Q.shape
    scale = 1.0 / math.sqrt(dh) if scale is None else scale
    O = np.zeros(Q.shape)
    LSE = np.zeros((B, R, H, C))
    grads = None if dO is None else tuple(np.zeros(Q.shape) for _ in range(3))
    for b in range(B):
        cols = _keys_feature(b, C, col_valid)
        if not cols:
            continue
        for r in range(R):
            for h in range(H):
                qs = [[float(Q[b, r, c, h, t]) for t in range(dh)] for c in cols]
                ks = [[float(K[b, r, c, h, t]) for t in range(dh)] for c in cols]
                vs = [[float(V[b, r, c, h, t]) for t in range(dh)] for c in cols]
                gs = None if dO is None else [[float(dO[b, r, c, h, t]) for t in range(dh)] for c in cols]
                o, lse, g = _attend(qs, ks, vs, gs, scale)
                for n, c in enumerate(cols):
                    O[b, r, c, h, :] = o[n]
                    LSE[b, r, h, c] = lse[n]
                    if g is not None:
                        for x in range(3):
                            grads[x][b, r, c, h, :] = g[x][n]
    return O, LSE, grads


def item(Q, K, V, n_train, dO=None, col_valid=None, scale=None):
    """Returns O [B,R,C,H,dh], LSE [B,C,H,R] and (dQ,dK,dV) or None.
    Keys are rows 0..n_train[b]-1 for every query row."""
    B, R, C, H, dh = Q.shape
    scale = 1.0 / math.sqrt(dh) if scale is None else scale
    O = np.zeros(Q.shape)
    LSE = np.zeros((B, C, H, R))
    grads = None if dO is None else tuple(np.zeros(Q.shape) for _ in range(3))
    for b in range(B):
        n = int(n_train[b])
        for c in range(C):
            if col_valid is not None and not col_valid[b][c]:
                continue
            for h in range(H):
                qs = [[float(Q[b, r, c, h, t]) for t in range(dh)] for r in range(R)]
                ks = [[float(K[b, r, c, h, t]) for t in range(dh)] for r in range(n)]
                vs = [[float(V[b, r, c, h, t]) for t in range(dh)] for r in range(n)]
                gs = None if dO is None else [[float(dO[b, r, c, h, t]) for t in range(dh)] for r in range(R)]
                o, lse, g = _attend(qs, ks, vs, gs, scale)
                for r in range(R):
                    O[b, r, c, h, :] = o[r]
                    LSE[b, c, h, r] = lse[r]
                    if g is not None:
                        grads[0][b, r, c, h, :] = g[0][r]
                if g is not None:
                    for r in range(n):
                        grads[1][b, r, c, h, :] = g[1][r]
                        grads[2][b, r, c, h, :] = g[2][r]
    return O, LSE, grads
