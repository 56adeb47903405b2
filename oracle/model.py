"""Mask-predictor forward pass in float64 (section 2.1: "the prompt, concatenated with a
user-specified number of [MASK] tokens, is fed into the model's mask predictor ... predictions for
all masked tokens in parallel in a single forward pass"; "Transformer-based mask predictors with
full bidirectional attention").  TEST INFRASTRUCTURE ONLY.

Layer internals (RMSNorm, RoPE, GQA, SwiGLU) come from BASELINE.json's config lines, the paper being
silent; every such reading is listed in DESIGN.md (G9, G12).  No blocking, fusion or reordering:
each function is the textbook formula.
"""
from __future__ import annotations

import numpy as np

from . import weights as W


def rmsnorm(x: np.ndarray, eps: float) -> np.ndarray:
    """x * rsqrt(mean(x^2) + eps) * g with g = 1 (G9)."""
    return x / np.sqrt((x * x).mean(axis=-1, keepdims=True) + eps)


def rope(x: np.ndarray, pos: np.ndarray, theta: float) -> np.ndarray:
    """Rotary embedding, half-split pairing (G12): for i < d_h/2 the pair (x_i, x_{i+d_h/2}) is rotated
    by angle pos * theta^(-2i/d_h).  x: [T, heads, d_h], pos: [T] absolute index in prompt||generation."""
    dh = x.shape[-1]
    half = dh // 2
    i = np.arange(half, dtype=np.float64)
    ang = pos.astype(np.float64)[:, None] * np.power(np.float64(theta), -2.0 * i / dh)[None, :]
    c, s = np.cos(ang)[:, None, :], np.sin(ang)[:, None, :]
    a, b = x[..., :half], x[..., half:]
    return np.concatenate([a * c - b * s, b * c + a * s], axis=-1)


def attention(q: np.ndarray, k: np.ndarray, v: np.ndarray) -> np.ndarray:
    """softmax_j(q.k_j / sqrt(d_h)) v_j over ALL j, no mask ("full bidirectional attention";
    P:369 "without causal masking").  q: [Tq, H, d_h]; k, v: [S, H_kv, d_h]; query head h reads
    KV head floor(h * H_kv / H).  Returns [Tq, H, d_h]."""
    tq, h, dh = q.shape
    hkv = k.shape[1]
    out = np.empty_like(q)
    for hh in range(h):
        g = (hh * hkv) // h
        sc = (q[:, hh, :] @ k[:, g, :].T) / np.sqrt(np.float64(dh))
        sc = sc - sc.max(axis=-1, keepdims=True)
        p = np.exp(sc)
        p = p / p.sum(axis=-1, keepdims=True)
        out[:, hh, :] = p @ v[:, g, :]
    return out


def silu(x: np.ndarray) -> np.ndarray:
    return x / (1.0 + np.exp(-x))


def layer_qkv(arch, wts, layer: int, x: np.ndarray, pos: np.ndarray):
    """u = RMSNorm(x); q,k,v = u W_q^T, u W_k^T, u W_v^T; q,k rotated by absolute position."""
    u = rmsnorm(x, arch.rms_eps)
    t = x.shape[0]
    q = (u @ wts.get(W.layer_tid(layer, W.SUB_Q)).T).reshape(t, arch.n_heads, arch.head_dim)
    k = (u @ wts.get(W.layer_tid(layer, W.SUB_K)).T).reshape(t, arch.n_kv_heads, arch.head_dim)
    v = (u @ wts.get(W.layer_tid(layer, W.SUB_V)).T).reshape(t, arch.n_kv_heads, arch.head_dim)
    return rope(q, pos, arch.rope_theta), rope(k, pos, arch.rope_theta), v


def layer_post_attention(arch, wts, layer: int, x: np.ndarray, a: np.ndarray) -> np.ndarray:
    """x += a W_o^T;  x += (silu(u W_g^T) * (u W_u^T)) W_d^T with u = RMSNorm(x)."""
    t = x.shape[0]
    x = x + a.reshape(t, -1) @ wts.get(W.layer_tid(layer, W.SUB_O)).T
    u = rmsnorm(x, arch.rms_eps)
    act = silu(u @ wts.get(W.layer_tid(layer, W.SUB_G)).T) * (u @ wts.get(W.layer_tid(layer, W.SUB_U)).T)
    return x + act @ wts.get(W.layer_tid(layer, W.SUB_D)).T


def embed(arch, wts, tokens: np.ndarray) -> np.ndarray:
    return wts.rows(W.TID_EMBED, np.asarray(tokens, dtype=np.int64))


def full_forward(arch, wts, tokens: np.ndarray, pos0: int = 0, trace: dict | None = None):
    """Recompute pass ("the KV tensors for all blocks are recomputed"; "recompute steps
    process all tokens in the sequence").  Returns (hidden [S, d] = last layer's residual output,
    kv = per layer (K post-RoPE [S,H_kv,d_h], V [S,H_kv,d_h]))."""
    s = len(tokens)
    pos = np.arange(s, dtype=np.float64) + pos0
    x = embed(arch, wts, tokens)
    kv = []
    for l in range(arch.n_layers):
        q, k, v = layer_qkv(arch, wts, l, x, pos)
        kv.append((k, v))
        a = attention(q, k, v)
        if trace is not None:
            trace[("q", l)], trace[("attn", l)], trace[("x_in", l)] = q, a, x
        x = layer_post_attention(arch, wts, l, x, a)
        if trace is not None:
            trace[("x_out", l)] = x
    return x, kv


def cached_forward(arch, wts, tokens: np.ndarray, lo: int, hi: int, kv, pos0: int = 0, trace: dict | None = None):
    """Cache pass ("cache steps compute only the tokens inside the current cache block";
    P:109 "cache and reuse the KV tensors for the prefix and suffix blocks throughout the denoising
    steps of the current block").  Rows [lo, hi) are computed; their K/V are fresh, every other
    position's K/V comes from `kv` unchanged.  Returns (hidden [hi-lo, d], fresh block kv per layer)."""
    pos = np.arange(lo, hi, dtype=np.float64) + pos0
    x = embed(arch, wts, tokens[lo:hi])
    fresh = []
    for l in range(arch.n_layers):
        q, k, v = layer_qkv(arch, wts, l, x, pos)
        kc, vc = kv[l]
        kk = np.concatenate([kc[:lo], k, kc[hi:]], axis=0)
        vv = np.concatenate([vc[:lo], v, vc[hi:]], axis=0)
        fresh.append((k, v))
        a = attention(q, kk, vv)
        if trace is not None:
            trace[("q", l)], trace[("attn", l)], trace[("x_in", l)] = q, a, x
        x = layer_post_attention(arch, wts, l, x, a)
        if trace is not None:
            trace[("x_out", l)] = x
    return x, fresh


def logits(arch, wts, hidden: np.ndarray) -> np.ndarray:
    """z = s * RMSNorm(hidden) W_lm^T with z[mask_id] = -inf (G7: the predictor never proposes [MASK],
    so every step makes progress, "to ensure progress")."""
    h = rmsnorm(hidden, arch.rms_eps)
    z = np.float64(arch.logit_scale) * (h @ wts.get(W.TID_LMHEAD).T)
    z[:, arch.mask_id] = -np.inf
    return z


def confidence(z: np.ndarray):
    """"For each predicted token, the model uses its softmax probability as a confidence score".
    tok = argmax z (lowest id on ties, G8); lse = log sum exp z; conf = softmax(z)[tok] computed as
    1 / sum_v exp(z_v - z_max).  Also returns the top-2 probability margin used by the near-tie
    exclusion (G13)."""
    m = z.max(axis=-1)
    tok = z.argmax(axis=-1)            # numpy returns the first (lowest) index on ties
    e = np.exp(z - m[:, None])
    ssum = e.sum(axis=-1)
    lse = m + np.log(ssum)
    conf = 1.0 / ssum
    z2 = z.copy()
    z2[np.arange(len(z)), tok] = -np.inf
    margin = conf - np.exp(z2.max(axis=-1) - lse)
    return tok.astype(np.int64), conf, lse, margin


def head(arch, wts, hidden: np.ndarray):
    return confidence(logits(arch, wts, hidden))
