"""Scalar-loop twin of model.py / step.py: the same definitions written with Python floats and `math`,
no numpy linear algebra, no vectorised indexing.  TEST INFRASTRUCTURE ONLY; tiny shapes only
(L<=2, d<=32, V<=64, S<=24).  It exists so that a slip in an einsum / reshape / broadcast / concatenate
of model.py (a transposed operand, a wrong head-group index, a RoPE pair off by one, K/V rows spliced
at the wrong offset) shows up as a disagreement.
"""
from __future__ import annotations

import math

from . import weights as W


def _mat(wts, tid):
    a = wts.f32(tid)
    return [[float(v) for v in row] for row in a]


def _rmsnorm(x, eps):
    ms = sum(v * v for v in x) / len(x)
    r = 1.0 / math.sqrt(ms + eps)
    return [v * r for v in x]


def _matvec(w, x):            # w: [out][in]
    return [sum(wi[j] * x[j] for j in range(len(x))) for wi in w]


def _rope(vec, pos, dh, theta):
    out = list(vec)
    half = dh // 2
    for h0 in range(0, len(vec), dh):
        for i in range(half):
            ang = pos * theta ** (-2.0 * i / dh)
            c, s = math.cos(ang), math.sin(ang)
            a, b = vec[h0 + i], vec[h0 + i + half]
            out[h0 + i] = a * c - b * s
            out[h0 + i + half] = b * c + a * s
    return out


def forward(arch, wts, tokens, rows, cache=None):
    """Compute positions `rows` (a list of absolute indices).  cache=None: rows must be all positions and
    every K/V is fresh; else K/V of positions outside `rows` come from cache[l][pos] = (k_vec, v_vec).
    Returns (hidden per row, kv per layer as dict pos -> (k, v))."""
    S = len(tokens)
    E = wts.f32(W.TID_EMBED)
    x = {p: [float(v) for v in E[int(tokens[p])]] for p in rows}
    H, Hkv, dh = arch.n_heads, arch.n_kv_heads, arch.head_dim
    kv_all = []
    for l in range(arch.n_layers):
        wq, wk, wv, wo = (_mat(wts, W.layer_tid(l, s)) for s in (W.SUB_Q, W.SUB_K, W.SUB_V, W.SUB_O))
        wg, wu, wd = (_mat(wts, W.layer_tid(l, s)) for s in (W.SUB_G, W.SUB_U, W.SUB_D))
        q, kv = {}, {}
        for p in rows:
            u = _rmsnorm(x[p], arch.rms_eps)
            q[p] = _rope(_matvec(wq, u), p, dh, arch.rope_theta)
            kv[p] = (_rope(_matvec(wk, u), p, dh, arch.rope_theta), _matvec(wv, u))
        if cache is not None:
            for p in range(S):
                if p not in kv:
                    kv[p] = cache[l][p]
        kv_all.append(kv)
        for p in rows:
            a = [0.0] * (H * dh)
            for h in range(H):
                g = (h * Hkv) // H
                sc = []
                for j in range(S):
                    kj = kv[j][0]
                    sc.append(sum(q[p][h * dh + e] * kj[g * dh + e] for e in range(dh)) / math.sqrt(dh))
                m = max(sc)
                w = [math.exp(v - m) for v in sc]
                z = sum(w)
                for j in range(S):
                    vj = kv[j][1]
                    for e in range(dh):
                        a[h * dh + e] += (w[j] / z) * vj[g * dh + e]
            o = _matvec(wo, a)
            xp = [x[p][i] + o[i] for i in range(len(o))]
            u = _rmsnorm(xp, arch.rms_eps)
            gg, uu = _matvec(wg, u), _matvec(wu, u)
            act = [gg[i] / (1.0 + math.exp(-gg[i])) * uu[i] for i in range(len(gg))]
            dn = _matvec(wd, act)
            x[p] = [xp[i] + dn[i] for i in range(len(dn))]
    return x, kv_all


def head(arch, wts, hvec):
    lm = _mat(wts, W.TID_LMHEAD)
    h = _rmsnorm(hvec, arch.rms_eps)
    z = [arch.logit_scale * v for v in _matvec(lm, h)]
    z[arch.mask_id] = -math.inf
    best = 0
    for v in range(1, len(z)):
        if z[v] > z[best]:
            best = v
    m = z[best]
    ssum = sum(math.exp(v - m) for v in z)
    return best, 1.0 / ssum, m + math.log(ssum)


def run(arch, wts, prompt, G, B, tau, use_cache=True):
    """Whole trajectory; returns list of steps, each a list of (pos, tok)."""
    P = len(prompt)
    tokens = [int(t) for t in prompt] + [arch.mask_id] * G
    S = P + G
    hist = []
    for b in range(G // B):
        lo, hi = P + b * B, P + (b + 1) * B
        cache = None
        while any(tokens[i] == arch.mask_id for i in range(lo, hi)):
            if cache is None or not use_cache:
                x, cache = forward(arch, wts, tokens, list(range(S)))
            else:
                x, _ = forward(arch, wts, tokens, list(range(lo, hi)), cache)
            pred = {i: head(arch, wts, x[i]) for i in range(lo, hi)}
            M = [i for i in range(lo, hi) if tokens[i] == arch.mask_id]
            best = M[0]
            for i in M:
                if pred[i][1] > pred[best][1]:
                    best = i
            C = [i for i in M if pred[i][1] >= tau or i == best]
            for i in C:
                tokens[i] = pred[i][0]
            hist.append([(i, pred[i][0]) for i in C])
    return tokens, hist
