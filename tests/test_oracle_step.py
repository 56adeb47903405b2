"""Pins for oracle/step.py: the invariants the paper's prose and north_star fix."""
import numpy as np
import pytest

from oracle import brute, model, step, weights as W
from synth_inputs import random_tokens


def _req(arch, P=10, G=12, B=4, tau=0.9, seed=0):
    prompt = random_tokens(np.random.default_rng(seed), P, arch.vocab, arch.mask_id)
    return step.Request(arch, prompt, G, B, tau)


def test_unmask_rule_cases():
    mask = 99
    tokens = np.array([5, mask, mask, 7, mask, mask, mask, mask])
    tok = np.array([11, 12, 13, 14])                 # block = positions [1, 5)
    conf = np.array([0.2, 0.95, 0.99, 0.91])
    # threshold met by positions 2 (0.95) and 4 (0.91); position 3 is not MASK so its 0.99 is ignored
    t = tokens.copy()
    c = step.unmask(t, 1, 5, tok, conf, 0.9, mask)
    assert [(x.pos, x.tok) for x in c] == [(2, 12), (4, 14)] and t.tolist() == [5, mask, 12, 7, 14, mask, mask, mask]
    # nothing reaches the threshold -> the single most confident MASK position
    t = tokens.copy()
    c = step.unmask(t, 1, 5, tok, conf, 0.96, mask)
    assert [(x.pos, x.tok) for x in c] == [(2, 12)]
    # conf == tau commits (G1: at or above)
    t = tokens.copy()
    assert [x.pos for x in step.unmask(t, 1, 5, tok, conf, 0.91, mask)] == [2, 4]
    # ties in confidence -> lowest position
    t = tokens.copy()
    assert [x.pos for x in step.unmask(t, 1, 5, tok, np.array([0.5, 0.5, 0.9, 0.5]), 2.0, mask)] == [1]
    # no MASK in the block -> nothing; positions outside the block are never touched
    t = np.array([1, 2, 3, mask])
    assert step.unmask(t, 0, 3, np.array([4, 5, 6]), np.array([1.0, 1.0, 1.0]), 0.0, mask) == [] and t[3] == mask
    # dry run reports but does not write
    t = tokens.copy()
    assert len(step.unmask(t, 1, 5, tok, conf, 0.0, mask, dry_run=True)) == 3 and np.array_equal(t, tokens)


@pytest.mark.parametrize("use_cache", [True, False])
def test_tau_above_one_commits_exactly_one_per_step(tiny_arch, use_cache):
    wts = W.Weights(tiny_arch, 41)
    r = _req(tiny_arch, tau=1.5)
    hist = step.run(r, wts, use_cache=use_cache)
    assert len(hist) == r.G and all(len(h.commits) == 1 for h in hist)
    kinds = [h.kind for h in hist]
    if use_cache:     # per block: 1 refresh + (B-1) cached
        assert kinds == (["refresh"] + ["cached"] * (r.B - 1)) * (r.G // r.B)
    else:             # P:680 "without KV caching": refresh every step
        assert set(kinds) == {"refresh"}
    assert r.n_masked() == 0


def test_tau_zero_commits_whole_block_per_step(tiny_arch):
    wts = W.Weights(tiny_arch, 42)
    r = _req(tiny_arch, tau=0.0)
    hist = step.run(r, wts)
    assert len(hist) == r.G // r.B and all(h.kind == "refresh" and len(h.commits) == r.B for h in hist)
    for b, h in enumerate(hist):
        assert [c.pos for c in h.commits] == list(range(r.P + b * r.B, r.P + (b + 1) * r.B))


@pytest.mark.parametrize("tau", [0.02, 0.05, 0.3])
def test_progress_and_immutability(tiny_arch, tau):
    wts = W.Weights(tiny_arch, 43)
    r = _req(tiny_arch, P=9, G=16, B=8, tau=tau, seed=3)
    prev = r.tokens.copy()
    left = r.n_masked()
    per_block = {}
    while r.current_block() is not None:
        b = r.current_block()
        lo, hi = r.block_range(b)
        res = step.next_step(r, wts)
        per_block[b] = per_block.get(b, 0) + 1
        assert len(res.commits) >= 1 and res.n_masked_left == left - len(res.commits) < left    # strict progress
        for c in res.commits:                                # commits lie in current block and were MASK
            assert lo <= c.pos < hi and prev[c.pos] == tiny_arch.mask_id and c.tok != tiny_arch.mask_id
            assert r.tokens[c.pos] == c.tok
        unchanged = np.ones(r.S, bool)
        unchanged[[c.pos for c in res.commits]] = False
        assert np.array_equal(r.tokens[unchanged], prev[unchanged])      # committed tokens never change
        thr = [c for c in res.commits if c.conf >= tau]
        assert len(thr) == len(res.commits) or len(res.commits) == 1     # only the at-least-one rule goes below tau
        prev, left = r.tokens.copy(), res.n_masked_left
    assert all(n <= r.B for n in per_block.values())          # at most B steps per block
    assert np.array_equal(r.tokens[:r.P], prev[:r.P])


def test_cached_step_right_after_refresh_equals_full_recompute(tiny_arch):
    """G15: F_cached(x; KV(x)) == F_full(x) on the block rows, on the same token state."""
    wts = W.Weights(tiny_arch, 44)
    r = _req(tiny_arch, P=11, G=12, B=4, tau=0.5, seed=5)
    r.tokens[r.P + 4 + 1] = 7            # second block partly committed; first block still masked
    a = step.refresh_step(r, wts, dry_run=True)
    b = step.cached_step(r, wts, dry_run=True)
    assert a.block_lo == b.block_lo == r.P
    assert np.allclose(a.hidden, b.hidden, rtol=0, atol=1e-12) and np.allclose(a.lse, b.lse, atol=1e-12)
    assert [(c.pos, c.tok) for c in a.commits] == [(c.pos, c.tok) for c in b.commits]
    # after a real commit the cached result differs from a recompute: that IS the approximation
    step.refresh_step(r, wts, tau=2.0)
    c1 = step.cached_step(r, wts, dry_run=True)
    h_full, _ = model.full_forward(tiny_arch, wts, r.tokens)
    assert np.abs(c1.hidden - h_full[r.P:r.P + 4]).max() > 1e-9


@pytest.mark.parametrize("tau", [0.03, 0.3, 1.5])
def test_single_layer_cached_trajectory_equals_recompute_trajectory(tiny_arch, tau):
    """L = 1: a position's layer-1 K/V depend on its own token only, so stale == fresh for every
    position outside the block and the cached trajectory equals the recompute-every-step one."""
    a1 = tiny_arch.replace(n_layers=1)
    wts = W.Weights(a1, 45)
    ra, rb = _req(a1, tau=tau, seed=6), _req(a1, tau=tau, seed=6)
    ha, hb = step.run(ra, wts, use_cache=True), step.run(rb, wts, use_cache=False)
    assert [[(c.pos, c.tok) for c in h.commits] for h in ha] == [[(c.pos, c.tok) for c in h.commits] for h in hb]
    assert np.array_equal(ra.tokens, rb.tokens)
    for x, y in zip(ha, hb):
        assert np.allclose(x.conf, y.conf, rtol=0, atol=1e-12)


def test_cached_step_needs_valid_cache_and_block_completion_invalidates(tiny_arch):
    wts = W.Weights(tiny_arch, 46)
    r = _req(tiny_arch, tau=0.0)
    with pytest.raises(RuntimeError):
        step.cached_step(r, wts)
    step.refresh_step(r, wts)            # tau = 0 completes block 0
    assert not r.cache_valid and r.current_block() == 1
    with pytest.raises(RuntimeError):
        step.cached_step(r, wts)


@pytest.mark.parametrize("tau", [0.04, 1.5])
def test_migration_at_a_recompute_step_keeps_the_trajectory(tiny_arch, tau):
    """at a block's first step the cache is invalid anyway, so a request that drops its cache there (migration)
    continues exactly as the one that stayed; dropped mid-block it takes a fresh cache instead of the stale one, which
    is a different (L > 1) computation."""
    wts = W.Weights(tiny_arch, 48)
    stay, move = _req(tiny_arch, tau=tau, seed=9), _req(tiny_arch, tau=tau, seed=9)
    while move.current_block() == 0:
        step.next_step(stay, wts), step.next_step(move, wts)
    assert not move.cache_valid
    moved = move.migrate()
    assert moved.cache is None and not moved.cache_valid and moved.steps_done == move.steps_done
    ha, hb = step.run(stay, wts), step.run(moved, wts)
    assert [[(c.pos, c.tok, c.conf) for c in h.commits] for h in ha] == [[(c.pos, c.tok, c.conf) for c in h.commits] for h in hb]
    assert np.array_equal(stay.tokens, moved.tokens)
    assert np.array_equal(step.predictor_features(stay), step.predictor_features(moved))
    # mid-block: the receiver's first step is a refresh (fresh K/V everywhere), the stayer's a cached one
    s2 = _req(tiny_arch, tau=1.5, seed=9)
    step.next_step(s2, wts), step.next_step(s2, wts)
    assert s2.cache_valid
    m2 = s2.migrate()
    a, b = step.next_step(s2, wts), step.next_step(m2, wts)
    assert (a.kind, b.kind) == ("cached", "refresh") and np.abs(a.conf - b.conf).max() > 1e-12


def test_per_step_threshold_override(tiny_arch):
    """the threshold may change at every step."""
    wts = W.Weights(tiny_arch, 47)
    r = _req(tiny_arch, tau=1.5)
    hist = step.run(r, wts, tau_schedule=lambda i: 0.0 if i == 1 else 1.5)
    assert len(hist[0].commits) == 1 and len(hist[1].commits) == r.B - 1 and hist[1].kind == "cached"


@pytest.mark.parametrize("tau", [0.0, 0.04, 0.9, 1.5])
@pytest.mark.parametrize("use_cache", [True, False])
def test_brute_force_twin_trajectories(tau, use_cache):
    from synth_inputs import Arch
    arch = Arch(2, 16, 2, 1, 8, 24, 32, 31, 0, 8.0)
    wts = W.Weights(arch, 48)
    prompt = random_tokens(np.random.default_rng(9), 6, arch.vocab, arch.mask_id)
    r = step.Request(arch, prompt, 8, 4, tau)
    hist = step.run(r, wts, use_cache=use_cache)
    toks, bh = brute.run(arch, wts, prompt, 8, 4, tau, use_cache)
    assert [[(c.pos, c.tok) for c in h.commits] for h in hist] == bh
    assert r.tokens.tolist() == toks


# ------------------------------------------------------------------------------------------------------------------
# Step Predictor features (App. A; reading G22)
# ------------------------------------------------------------------------------------------------------------------
def test_quantile_linear_matches_library_and_hand_cases():
    """Special cases with a textbook answer + the library routine on random data (numpy's default is the same
    linear interpolation between order statistics)."""
    assert step.quantile_linear(np.array([0.0, 1.0]), 0.25) == 0.25
    assert step.quantile_linear(np.array([1.0, 2.0, 3.0, 4.0, 5.0]), 0.5) == 3.0
    assert step.quantile_linear(np.array([1.0, 2.0, 3.0, 4.0]), 0.75) == 3.25      # h = 2.25
    assert step.quantile_linear(np.array([7.0]), 0.25) == 7.0
    rng = np.random.default_rng(3)
    for n in (2, 5, 32, 256, 257):
        v = np.sort(rng.random(n))
        for q in (0.25, 0.5, 0.75):
            assert abs(step.quantile_linear(v, q) - np.quantile(v, q)) < 1e-15


def test_predictor_features_invariants_and_closed_forms(tiny_arch):
    """Fresh request: progress 0, confidences 0.  tau > 1: one commit per step, so after k steps
    full_progress = full_unmask_progress = k / G and block_unmask_progress = (k mod B) / B.  Committed
    positions keep their confidence (frozen), min <= q25 <= median <= q75, avg within [min, max]."""
    arch, wts = tiny_arch, W.Weights(tiny_arch, 47)
    prompt = random_tokens(np.random.default_rng(9), 10, arch.vocab, arch.mask_id)
    req = step.Request(arch, prompt, 16, 8, 1.5)
    f0 = step.predictor_features(req)
    assert list(f0[:2]) == [1.5, 16] and not f0[2:].any()
    frozen = {}
    for k in range(1, 17):
        r = step.next_step(req, wts)
        assert len(r.commits) == 1
        f = step.predictor_features(req, tau=0.7)
        assert f[0] == 0.7 and f[1] == 16
        assert f[2] == k / 16 and f[3] == k / 16
        if k < 16:
            assert f[4] == (k // 8) / 2 and f[5] == (k % 8) / 8
        else:
            assert f[4] == 1.0 and f[5] == 1.0
        assert f[6] <= f[7] <= f[8] <= f[10] <= req.conf_state.max() and f[6] <= f[9] <= req.conf_state.max()
        c = r.commits[0]
        frozen[c.pos] = c.conf
        for pos, v in frozen.items():                 # frozen at commit, never touched again
            assert req.conf_state[pos - req.P] == v
        if k <= 8:                                    # the second block has not been evaluated yet
            assert not req.conf_state[8:].any()
    # a dry-run step leaves the predictor state alone
    req2 = step.Request(arch, prompt, 16, 8, 0.5)
    step.refresh_step(req2, wts, dry_run=True)
    assert req2.steps_done == 0 and not req2.conf_state.any()
