"""Pins for oracle/model.py: textbook reductions, closed forms, invariants, brute force."""
import math

import numpy as np

from oracle import brute, model, weights as W
from synth_inputs import random_tokens


def _wts(arch, seed=21):
    return W.Weights(arch, seed)


def test_attention_brute_force_and_gqa():
    rng = np.random.default_rng(0)
    tq, s, h, hkv, dh = 5, 11, 6, 2, 8
    q, k, v = rng.standard_normal((tq, h, dh)), rng.standard_normal((s, hkv, dh)), rng.standard_normal((s, hkv, dh))
    got = model.attention(q, k, v)
    # scalar-loop textbook softmax(QK^T/sqrt d)V with query head hh reading KV head floor(hh*hkv/h)
    for i in range(tq):
        for hh in range(h):
            g = hh * hkv // h
            sc = [sum(q[i, hh, e] * k[j, g, e] for e in range(dh)) / math.sqrt(dh) for j in range(s)]
            m = max(sc)
            w = [math.exp(x - m) for x in sc]
            o = [sum(w[j] * v[j, g, e] for j in range(s)) / sum(w) for e in range(dh)]
            assert np.allclose(got[i, hh], o, rtol=0, atol=1e-13)
    # GQA == MHA with K/V repeated per group; H_kv == H is plain MHA
    rep = h // hkv
    assert np.allclose(got, model.attention(q, np.repeat(k, rep, axis=1), np.repeat(v, rep, axis=1)), atol=1e-14)
    # not causal: permuting the key/value positions leaves the result unchanged
    perm = rng.permutation(s)
    assert np.allclose(got, model.attention(q, k[perm], v[perm]), atol=1e-13)
    # one key => output is that value, whatever the query
    assert np.allclose(model.attention(q, k[:1], v[:1]), np.broadcast_to(np.repeat(v[:1], rep, axis=1), (tq, h, dh)))


def test_rope_invariants():
    rng = np.random.default_rng(1)
    x = rng.standard_normal((7, 3, 16))
    pos = np.arange(7, dtype=np.float64) + 3
    y = model.rope(x, pos, 10000.0)
    assert np.allclose(np.linalg.norm(y, axis=-1), np.linalg.norm(x, axis=-1), atol=1e-12)   # rotation
    assert np.allclose(model.rope(x, np.zeros(7), 10000.0), x)                                # angle 0
    # explicit pair (i, i + d_h/2), angle pos * theta^(-2i/d_h)
    t, hh, i = 4, 1, 5
    ang = pos[t] * 10000.0 ** (-2 * i / 16)
    assert math.isclose(y[t, hh, i], x[t, hh, i] * math.cos(ang) - x[t, hh, i + 8] * math.sin(ang), abs_tol=1e-13)
    assert math.isclose(y[t, hh, i + 8], x[t, hh, i + 8] * math.cos(ang) + x[t, hh, i] * math.sin(ang), abs_tol=1e-13)
    # scores depend on position differences only
    k = rng.standard_normal((7, 3, 16))
    s0 = np.einsum("thd,shd->hts", model.rope(x, pos, 1e4), model.rope(k, pos, 1e4))
    s1 = np.einsum("thd,shd->hts", model.rope(x, pos + 37, 1e4), model.rope(k, pos + 37, 1e4))
    assert np.allclose(s0, s1, atol=1e-11)


def test_position_shift_leaves_hidden_unchanged(tiny_arch):
    """Adding a constant to all positions leaves the logits unchanged (RoPE is relative)."""
    wts = _wts(tiny_arch)
    tok = random_tokens(np.random.default_rng(3), 20, tiny_arch.vocab, tiny_arch.mask_id)
    h0, _ = model.full_forward(tiny_arch, wts, tok, pos0=0)
    h1, _ = model.full_forward(tiny_arch, wts, tok, pos0=113)
    assert np.allclose(h0, h1, rtol=0, atol=1e-12)


def test_rmsnorm_and_silu_closed_forms():
    x = np.array([[3.0, -4.0, 0.0, 0.0]])
    assert np.allclose(model.rmsnorm(x, 0.0), x / 2.5)          # rms = sqrt(25/4)
    assert np.allclose(model.rmsnorm(7.0 * x, 0.0), model.rmsnorm(x, 0.0))   # scale invariant
    assert math.isclose(model.silu(np.array([0.0]))[0], 0.0)
    assert math.isclose(model.silu(np.array([2.0]))[0], 2.0 / (1 + math.exp(-2.0)))


class _Patched(W.Weights):
    """Weights with selected tensors forced to zero (closed-form special cases)."""

    def __init__(self, arch, seed, zero_subs=(), zero_lm=False):
        super().__init__(arch, seed)
        self.zero_subs, self.zero_lm = set(zero_subs), zero_lm

    def f32(self, tid):
        w = super().f32(tid)
        if (tid >= 16 and tid % 16 in self.zero_subs) or (tid == W.TID_LMHEAD and self.zero_lm):
            return np.zeros_like(w)
        return w


def test_zero_weight_closed_forms(tiny_arch):
    tok = random_tokens(np.random.default_rng(4), 12, tiny_arch.vocab, tiny_arch.mask_id)
    # zero W_o and W_d => every layer adds nothing => hidden = E[token]
    wz = _Patched(tiny_arch, 5, zero_subs=(W.SUB_O, W.SUB_D))
    h, _ = model.full_forward(tiny_arch, wz, tok)
    assert np.array_equal(h, wz.rows(W.TID_EMBED, tok))
    # zero W_lm => logits all 0 except mask_id = -inf => conf = 1/(V-1), token = id 0, lse = log(V-1)
    wl = _Patched(tiny_arch, 5, zero_lm=True)
    t, conf, lse, margin = model.head(tiny_arch, wl, h)
    assert (t == 0).all() and np.allclose(conf, 1.0 / (tiny_arch.vocab - 1)) and np.allclose(lse, math.log(tiny_arch.vocab - 1))
    assert np.allclose(margin, 0.0)
    # mask_id = 0 => the tie resolves to id 1
    a0 = tiny_arch.replace(mask_id=0)
    t0, *_ = model.head(a0, _Patched(a0, 5, zero_lm=True), h)
    assert (t0 == 1).all()


def test_mask_id_never_predicted(tiny_arch):
    wts = _wts(tiny_arch)
    h = np.random.default_rng(5).standard_normal((50, tiny_arch.d_model))
    z = model.logits(tiny_arch, wts, h)
    assert np.isneginf(z[:, tiny_arch.mask_id]).all()
    t, conf, lse, _ = model.confidence(z)
    assert (t != tiny_arch.mask_id).all()
    # conf is the softmax probability of the argmax over the remaining V-1 ids
    zz = np.delete(z, tiny_arch.mask_id, axis=1)
    p = np.exp(zz - zz.max(1, keepdims=True))
    p /= p.sum(1, keepdims=True)
    assert np.allclose(conf, p.max(1), atol=1e-15) and np.allclose(lse, np.log(np.exp(zz).sum(1)), atol=1e-12)
    assert np.allclose(np.exp(z[np.arange(50), t] - lse), conf, atol=1e-15)


def test_split_vocab_merge_equals_direct_softmax():
    """a11/a12: per-tile (max, sum exp(z-max), argmax) merged in any tile size / order == direct."""
    rng = np.random.default_rng(6)
    z = rng.standard_normal((9, 1000)) * 5
    z[:, 999] = -np.inf
    z[2, 10] = z[2, 700] = z[2].max() + 1.0          # exact tie -> lowest id
    tok, conf, lse, _ = model.confidence(z)
    for tile in (1, 7, 128, 256, 1000):
        bounds = [(a, min(a + tile, 1000)) for a in range(0, 1000, tile)]
        for order in (bounds, bounds[::-1], [bounds[i] for i in rng.permutation(len(bounds))]):
            m = np.full(9, -np.inf)
            s = np.zeros(9)
            idx = np.full(9, 1 << 30)
            for a, b in order:
                zt = z[:, a:b]
                mt = zt.max(1)
                it = zt.argmax(1) + a
                fin = np.isfinite(mt)
                st = np.where(fin, np.exp(zt - np.where(fin, mt, 0)[:, None]).sum(1), 0.0)
                better = (mt > m) | ((mt == m) & (it < idx))
                newm = np.maximum(m, mt)
                with np.errstate(invalid="ignore"):
                    s = np.where(np.isfinite(newm), s * np.exp(m - newm) + st * np.exp(mt - newm), 0.0)
                s = np.nan_to_num(s)
                idx = np.where(better, it, idx)
                m = newm
            assert np.array_equal(idx, tok)
            assert np.allclose(m + np.log(s), lse, atol=1e-12) and np.allclose(1 / s, conf, rtol=1e-12)


def test_brute_twin_forward_and_head(tiny_arch):
    """model.py (numpy linear algebra) vs brute.py (scalar loops) on full and cached passes."""
    for arch, seed in ((tiny_arch, 31), (tiny_arch.replace(n_heads=2, n_kv_heads=2, head_dim=16, n_layers=1), 32)):
        wts = _wts(arch, seed)
        rng = np.random.default_rng(seed)
        tok = random_tokens(rng, 14, arch.vocab, arch.mask_id)
        tok[9:] = arch.mask_id
        h, kv = model.full_forward(arch, wts, tok)
        hb, kvb = brute.forward(arch, wts, tok, list(range(14)))
        assert np.allclose(h, np.array([hb[p] for p in range(14)]), rtol=0, atol=1e-12)
        for l in range(arch.n_layers):
            assert np.allclose(kv[l][0].reshape(14, -1), np.array([kvb[l][p][0] for p in range(14)]), atol=1e-13)
            assert np.allclose(kv[l][1].reshape(14, -1), np.array([kvb[l][p][1] for p in range(14)]), atol=1e-13)
        tok2 = tok.copy()
        tok2[10] = 3                                    # stale cache: block rows recomputed, rest reused
        hc, _ = model.cached_forward(arch, wts, tok2, 8, 12, kv)
        hcb, _ = brute.forward(arch, wts, tok2, [8, 9, 10, 11], kvb)
        assert np.allclose(hc, np.array([hcb[p] for p in (8, 9, 10, 11)]), rtol=0, atol=1e-12)
        t, conf, lse, _ = model.head(arch, wts, hc)
        for r, p in enumerate((8, 9, 10, 11)):
            bt, bc, bl = brute.head(arch, wts, hcb[p])
            assert bt == t[r] and math.isclose(bc, conf[r], rel_tol=1e-11) and math.isclose(bl, lse[r], rel_tol=1e-12)
