"""Pins of oracle/control.py (the precision-floor control of protocol P-B): without rounding it IS the oracle
(1e-12), with bf16 rounding it stays within the north_star tolerance of the oracle and differs from it by about one
bf16 ulp per rounding point, and its step() never mutates tokens.  CPU only."""
import numpy as np

from oracle import compare, control, model as omodel, step as ostep, weights as ow
from synth_inputs import random_tokens


def _setup(tiny_arch, seed=11):
    a = tiny_arch.replace(weight_dtype=1)
    rng = np.random.default_rng(seed)
    prompt = random_tokens(rng, 13, a.vocab, a.mask_id)
    return a, ow.Weights(a, 77), prompt


def test_control_without_rounding_is_the_oracle(tiny_arch):
    a, wts, prompt = _setup(tiny_arch)
    req = ostep.Request(a, prompt, 16, 8, 0.9)
    h_or, kv_or = omodel.full_forward(a, wts, req.tokens)
    h_ct, kv_ct = control.forward(a, wts, req.tokens, None, None, None, None)
    assert np.abs(h_or - h_ct).max() < 1e-12
    for (k0, v0), (k1, v1) in zip(kv_or, kv_ct):
        assert np.abs(k0 - k1).max() < 1e-12 and np.abs(v0 - v1).max() < 1e-12
    toks = req.tokens.copy()
    toks[15] = 5                                   # a committed token: the cached pass then differs from the recompute pass
    lo, hi = 13, 21
    c_or, f_or = omodel.cached_forward(a, wts, toks, lo, hi, kv_or)
    c_ct, f_ct = control.forward(a, wts, toks, lo, hi, kv_ct, None)
    assert np.abs(c_or - c_ct).max() < 1e-12 and np.abs(f_or[1][0] - f_ct[1][0]).max() < 1e-12
    for x, y in zip(omodel.head(a, wts, c_or), control.head(a, wts, c_ct)):
        assert np.allclose(x, y, rtol=0, atol=1e-12)


def test_control_step_reports_like_the_oracle_and_leaves_tokens_alone(tiny_arch):
    a, wts, prompt = _setup(tiny_arch)
    o_req, c_req = ostep.Request(a, prompt, 16, 8, 0.3), ostep.Request(a, prompt, 16, 8, 0.3)
    for it in range(5):
        refresh = not o_req.cache_valid
        before = c_req.tokens.copy()
        c = control.step(c_req, wts, refresh, rnd=None)
        assert np.array_equal(c_req.tokens, before) and c_req.cache_valid
        lo, hi = o_req.block_range(o_req.current_block())
        masked = o_req.tokens[lo:hi] == a.mask_id
        o = ostep.refresh_step(o_req, wts) if refresh else ostep.cached_step(o_req, wts)
        d = compare.compare_commits(o, masked, 0.3, [(x.pos, x.tok, x.conf) for x in c.commits], conf_tol=1e-12)
        assert d.exact, d.detail
        assert np.abs(c.lse - o.lse).max() < 1e-12 and c.kind == o.kind
        c_req.tokens[:] = o_req.tokens             # teacher forcing
        if not o_req.cache_valid:
            c_req.cache_valid = False


def test_bf16_rounding_moves_the_result_by_the_bf16_noise_level(tiny_arch):
    """Rounding at the listed points perturbs the hidden state by more than fp32 noise and less than the north_star bound."""
    a, wts, prompt = _setup(tiny_arch)
    req = ostep.Request(a, prompt, 16, 8, 0.9)
    h_or, _ = omodel.full_forward(a, wts, req.tokens)
    h_bf, _ = control.forward(a, wts, req.tokens, None, None, None, control.make_rounder())
    rel = compare.rel_rows(h_bf, h_or)
    assert 1e-5 < rel.max() < 2e-2
    # the rounder is RNE to 8 significant bits: |r(x) - x| <= 2^-8 |x| (half an ulp of 2^-7), exact on bf16 values, deterministic without noise
    x = np.random.default_rng(0).standard_normal(1000)
    r = control.make_rounder()(x)
    assert np.all(np.abs(r - x) <= 2.0 ** -8 * np.abs(x) * (1 + 1e-6)) and np.array_equal(control.make_rounder()(r), r)
    n1, n2 = control.make_rounder(1e-6, 5)(x), control.make_rounder(1e-6, 5)(x)
    assert np.array_equal(n1, n2) and np.abs(n1 - r).max() <= 2.0 ** -7 * np.abs(x).max()
