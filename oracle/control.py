"""Precision-floor CONTROL for protocol P-B (SURVEY 8(c) "print beside it the
oracle-vs-perturbed-oracle control").  TEST INFRASTRUCTURE ONLY.

The same step as oracle/model.py + oracle/step.py, in float64, except that every tensor the bf16 fast path of the
CUDA library rounds to bf16 is rounded here too:

    RMSNorm output (all three norms) | Q, K, V after RoPE (K/V as stored) | softmax weights before the PV product |
    attention output | SwiGLU product

and, optionally, multiplied by (1 + noise * N(0,1)) BEFORE the rounding -- a stand-in for a second bf16
implementation that differs only in fp32 summation order (relative 1e-6).  Nothing else differs from the oracle:
with `rnd = None` the functions below reproduce model.full_forward / model.cached_forward / model.head to 1e-12
(pinned in tests/test_oracle_control.py), so any commit that differs between the oracle and this control is caused
by bf16 rounding of activations alone.  The control is NOT a second oracle: nothing is ever compared against it
for pass/fail except the COUNT of commit disagreements, which bounds what a correct bf16 implementation can reach.
"""
from __future__ import annotations

from typing import Callable, Optional

import numpy as np

from . import model
from . import step as ostep
from . import weights as W


def make_rounder(noise: float = 0.0, seed: int = 0) -> Callable[[np.ndarray], np.ndarray]:
    """x -> bf16(x * (1 + noise * N(0,1))) as float64."""
    rng = np.random.default_rng(seed)

    def rnd(x: np.ndarray) -> np.ndarray:
        if noise:
            x = x * (1.0 + noise * rng.standard_normal(x.shape))
        return W.round_to_bf16(np.asarray(x, dtype=np.float32)).astype(np.float64)

    return rnd


def _identity(x):
    return x


def _attention(q, k, v, rnd):
    """model.attention with the (unnormalised) softmax weights rounded before the PV product."""
    tq, h, dh = q.shape
    hkv = k.shape[1]
    out = np.empty_like(q)
    for hh in range(h):
        g = (hh * hkv) // h
        sc = (q[:, hh, :] @ k[:, g, :].T) / np.sqrt(np.float64(dh))
        p = np.exp(sc - sc.max(axis=-1, keepdims=True))
        out[:, hh, :] = (rnd(p) @ v[:, g, :]) / p.sum(axis=-1, keepdims=True)
    return out


def forward(arch, wts, tokens: np.ndarray, lo: Optional[int], hi: Optional[int], kv, rnd=None):
    """lo is None: recompute pass over all positions (returns hidden [S, d], kv); else cache pass over rows
    [lo, hi) against `kv` (returns hidden [hi - lo, d], the block's fresh kv).  Mirrors model.full_forward /
    model.cached_forward line by line."""
    rnd = rnd or _identity
    full = lo is None
    s = len(tokens)
    rows = np.arange(s) if full else np.arange(lo, hi)
    pos = rows.astype(np.float64)
    t = len(rows)
    x = model.embed(arch, wts, np.asarray(tokens)[rows])
    out_kv = []
    for l in range(arch.n_layers):
        u = rnd(model.rmsnorm(x, arch.rms_eps))
        q = (u @ wts.get(W.layer_tid(l, W.SUB_Q)).T).reshape(t, arch.n_heads, arch.head_dim)
        k = (u @ wts.get(W.layer_tid(l, W.SUB_K)).T).reshape(t, arch.n_kv_heads, arch.head_dim)
        v = (u @ wts.get(W.layer_tid(l, W.SUB_V)).T).reshape(t, arch.n_kv_heads, arch.head_dim)
        q, k, v = rnd(model.rope(q, pos, arch.rope_theta)), rnd(model.rope(k, pos, arch.rope_theta)), rnd(v)
        out_kv.append((k, v))
        if full:
            kk, vv = k, v
        else:
            kc, vc = kv[l]
            kk = np.concatenate([kc[:lo], k, kc[hi:]], axis=0)
            vv = np.concatenate([vc[:lo], v, vc[hi:]], axis=0)
        a = rnd(_attention(q, kk, vv, rnd))
        x = x + a.reshape(t, -1) @ wts.get(W.layer_tid(l, W.SUB_O)).T
        u = rnd(model.rmsnorm(x, arch.rms_eps))
        act = rnd(model.silu(u @ wts.get(W.layer_tid(l, W.SUB_G)).T) * (u @ wts.get(W.layer_tid(l, W.SUB_U)).T))
        x = x + act @ wts.get(W.layer_tid(l, W.SUB_D)).T
    return x, out_kv


def head(arch, wts, hidden: np.ndarray, rnd=None):
    """model.head with the final RMSNorm output rounded."""
    rnd = rnd or _identity
    z = np.float64(arch.logit_scale) * (rnd(model.rmsnorm(hidden, arch.rms_eps)) @ wts.get(W.TID_LMHEAD).T)
    z[:, arch.mask_id] = -np.inf
    return model.confidence(z)


def step(req: ostep.Request, wts, refresh: bool, tau: Optional[float] = None, rnd=None) -> ostep.StepResult:
    """One teacher-forced control step on `req` (an oracle Request that owns its own, rounded, cache): computes and
    reports like step.refresh_step / step.cached_step with dry_run=True -- tokens are never mutated (the caller
    teacher-forces them from the oracle) -- but the cache IS updated the way a real step updates it."""
    b = req.current_block()
    assert b is not None
    tau = req.threshold if tau is None else float(tau)
    lo, hi = req.block_range(b)
    if refresh:
        hidden, kv = forward(req.arch, wts, req.tokens, None, None, None, rnd)
        req.cache, req.cache_valid = kv, True
        hidden = hidden[lo:hi]
    else:
        assert req.cache_valid
        hidden, fresh = forward(req.arch, wts, req.tokens, lo, hi, req.cache, rnd)
        for l, (k, v) in enumerate(fresh):
            req.cache[l][0][lo:hi] = k
            req.cache[l][1][lo:hi] = v
    tok, conf, lse, margin = head(req.arch, wts, hidden, rnd)
    commits = ostep.unmask(req.tokens, lo, hi, tok, conf, tau, req.arch.mask_id, dry_run=True)
    return ostep.StepResult(commits, lse, conf, tok, margin, hidden, lo, req.n_masked(), "refresh" if refresh else "cached")
