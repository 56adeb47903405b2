"""Pins of oracle/compare.py (the judge every end-to-end parity test rests on): one hand-built case per rule of reading
G13 (north_star: "bit-exact, excluding positions whose top-2 margin or distance to the threshold is
below 1e-3, which are reported as a count") and per never-excused violation of P:74 / G3.  Each case would fail if the
rule it names were dropped, inverted or given the wrong bound.  CPU only."""
import numpy as np
import pytest

from oracle import compare
from oracle.step import Commit, StepResult

LO, B, TAU = 100, 8, 0.9


def _oracle(conf, tok=None, margin=None, masked=None, tau=TAU):
    """An oracle StepResult for a block of len(conf) rows at LO whose commits follow P:74 from the given values."""
    conf = np.asarray(conf, dtype=np.float64)
    n = len(conf)
    tok = np.arange(10, 10 + n) if tok is None else np.asarray(tok)
    margin = np.full(n, 0.5) if margin is None else np.asarray(margin, dtype=np.float64)
    masked = np.ones(n, bool) if masked is None else np.asarray(masked, bool)
    commits = []
    if masked.any():
        best = int(np.argmax(np.where(masked, conf, -np.inf)))
        commits = [Commit(LO + j, int(tok[j]), float(conf[j])) for j in range(n) if masked[j] and (conf[j] >= tau or j == best)]
    o = StepResult(commits, np.zeros(n), conf, tok, margin, np.zeros((n, 1)), LO, int(masked.sum()) - len(commits), "cached")
    return o, masked


def _got(o):
    return [(c.pos, c.tok, c.conf) for c in o.commits]


def test_exact_match_counts_nothing():
    o, m = _oracle([0.95, 0.2, 0.91, 0.1, 0.3, 0.3, 0.3, 0.3])
    d = compare.compare_commits(o, m, TAU, _got(o), conf_tol=1e-6)
    assert d.exact and d.n_mismatch == 0 and d.n_excluded == 0 and d.detail == [] and d.max_conf_err == 0.0
    assert sorted(c.pos for c in o.commits) == [LO, LO + 2]


@pytest.mark.parametrize("margin,excluded", [(2e-3, False), (5e-4, True)])
def test_rule_i_token_differs(margin, excluded):
    """(i) a different token at a committed position is a mismatch unless the oracle's vocabulary top-2 margin < 1e-3."""
    o, m = _oracle([0.95, 0.2, 0.2, 0.2, 0.2, 0.2, 0.2, 0.2], margin=[margin] + [0.5] * 7)
    got = [(LO, 999)]
    d = compare.compare_commits(o, m, TAU, got)
    assert not d.exact
    assert (d.n_excluded, d.n_mismatch) == ((1, 0) if excluded else (0, 1))


@pytest.mark.parametrize("dist,excluded", [(5e-4, True), (2e-3, False)])
@pytest.mark.parametrize("side", [+1, -1])
def test_rule_ii_membership_near_threshold(dist, excluded, side):
    """(ii) membership differs at |conf - tau| = 5e-4 -> excluded; at 2e-3 -> mismatch; on either side of tau."""
    conf = [0.99, TAU + side * dist, 0.1, 0.1, 0.1, 0.1, 0.1, 0.1]
    o, m = _oracle(conf)
    oracle_has = side > 0
    assert (LO + 1 in {c.pos for c in o.commits}) == oracle_has
    got = [(LO, 10)] + ([] if oracle_has else [(LO + 1, 11)])          # the other side decides position 1 the other way
    d = compare.compare_commits(o, m, TAU, got)
    assert not d.exact
    assert (d.n_excluded, d.n_mismatch) == ((1, 0) if excluded else (0, 1))


@pytest.mark.parametrize("gap,excluded", [(5e-4, True), (2e-3, False)])
def test_rule_iii_at_least_one_runner_up(gap, excluded):
    """(iii) nothing reaches tau, the other side commits the runner-up: excluded iff it is within 1e-3 of the best."""
    conf = [0.30, 0.30 - gap, 0.1, 0.1, 0.1, 0.1, 0.1, 0.1]
    o, m = _oracle(conf)
    assert [c.pos for c in o.commits] == [LO]
    d = compare.compare_commits(o, m, TAU, [(LO + 1, 11)])
    assert not d.exact and abs(d.min_gap - gap) < 1e-12
    # the oracle's own pick (gap 0 to the best) is inside the band by definition; the runner-up decides the verdict
    assert (d.n_excluded, d.n_mismatch) == ((2, 0) if excluded else (1, 1))


def test_rule_iii_does_not_apply_when_something_clearly_reaches_tau():
    """A position far below tau committed while another clearly passes tau: the at-least-one band must not excuse it."""
    conf = [0.95, 0.9495, 0.1, 0.1, 0.1, 0.1, 0.1, 0.1]
    o, m = _oracle(conf, tau=0.5)
    d = compare.compare_commits(o, m, 0.5, _got(o) + [(LO + 2, 12)])
    assert d.n_mismatch == 1 and d.n_excluded == 0


def test_commit_at_non_mask_position_is_a_mismatch():
    masked = [True, False, True, True, True, True, True, True]
    o, m = _oracle([0.95, 0.99, 0.2, 0.2, 0.2, 0.2, 0.2, 0.2], masked=masked)
    assert [c.pos for c in o.commits] == [LO]
    d = compare.compare_commits(o, m, TAU, [(LO, 10), (LO + 1, 11)])
    assert not d.exact and d.n_mismatch == 1 and "not MASK" in d.detail[0]


@pytest.mark.parametrize("pos", [LO - 1, LO + B, LO + 5 * B, 0])
def test_commit_outside_the_current_block_is_a_mismatch(pos):
    """G3: the threshold test and the at-least-one rule range over the current block only."""
    o, m = _oracle([0.95, 0.2, 0.2, 0.2, 0.2, 0.2, 0.2, 0.2])
    d = compare.compare_commits(o, m, TAU, _got(o) + [(pos, 5, 0.99)])
    assert not d.exact and d.n_mismatch == 1 and "outside the current block" in d.detail[0]


def test_no_commit_at_all_is_a_mismatch_even_inside_the_band():
    """P:74 "the token with the highest confidence is unmasked to ensure progress": an empty commit list never passes."""
    o, m = _oracle([0.3, 0.2999, 0.1, 0.1, 0.1, 0.1, 0.1, 0.1])
    d = compare.compare_commits(o, m, TAU, [])
    assert not d.exact and d.n_mismatch >= 1
    o2, m2 = _oracle([0.3] * 8, masked=[False] * 8)          # finished block: nothing to commit on either side
    d2 = compare.compare_commits(o2, m2, TAU, [])
    assert d2.exact and d2.n_mismatch == 0


def test_two_commits_when_nothing_reaches_tau_is_a_mismatch():
    """The at-least-one rule adds ONE position: two near-tied commits far below tau are a bug, not a near-tie."""
    o, m = _oracle([0.3, 0.2999, 0.1, 0.1, 0.1, 0.1, 0.1, 0.1])
    d = compare.compare_commits(o, m, TAU, [(LO, 10), (LO + 1, 11)])
    assert d.n_mismatch == 1 and d.n_excluded == 1


def test_duplicate_commit_is_a_mismatch():
    o, m = _oracle([0.95, 0.2, 0.2, 0.2, 0.2, 0.2, 0.2, 0.2])
    d = compare.compare_commits(o, m, TAU, _got(o) + _got(o))
    assert not d.exact and d.n_mismatch == 1


def test_commit_confidence_tolerance():
    o, m = _oracle([0.95, 0.2, 0.2, 0.2, 0.2, 0.2, 0.2, 0.2])
    ok = compare.compare_commits(o, m, TAU, [(LO, 10, 0.95 + 5e-6)], conf_tol=1e-5)
    bad = compare.compare_commits(o, m, TAU, [(LO, 10, 0.95 + 5e-5)], conf_tol=1e-5)
    unchecked = compare.compare_commits(o, m, TAU, [(LO, 10, 0.5)])
    assert ok.exact and ok.n_mismatch == 0 and abs(ok.max_conf_err - 5e-6) < 1e-9
    assert not bad.exact and bad.n_mismatch == 1
    assert unchecked.exact and abs(unchecked.max_conf_err - 0.45) < 1e-12


def test_band_is_in_probability_units_and_evaluated_on_oracle_values():
    """Band 1e-3 exactly: 0.999e-3 inside, 1.001e-3 outside (strict <), measured on the oracle's confidences."""
    for dist, excl in ((0.999e-3, 1), (1.001e-3, 0)):
        o, m = _oracle([0.99, TAU - dist, 0.1, 0.1, 0.1, 0.1, 0.1, 0.1])
        d = compare.compare_commits(o, m, TAU, _got(o) + [(LO + 1, 11)])
        assert (d.n_excluded, d.n_mismatch) == (excl, 1 - excl)


def test_compare_agrees_with_the_oracle_unmask_rule_on_random_blocks():
    """compare_commits(o, ., got = oracle.step.unmask on the same values) is exact for random blocks, and flags a
    mismatch for every single-position corruption whose confidence is far from tau and from the best."""
    from oracle.step import unmask
    rng = np.random.default_rng(0)
    for _ in range(200):
        n = 16
        conf = rng.uniform(0, 1, n)
        masked = rng.uniform(size=n) < 0.7
        if not masked.any():
            masked[0] = True
        tau = float(rng.choice([0.3, 0.6, 0.9, 1.5, 0.0]))
        toks = np.where(masked, 4095, rng.integers(0, 4000, n))
        tok_pred = rng.integers(0, 4000, n)
        commits = unmask(toks.copy(), 0, n, tok_pred, conf, tau, 4095, dry_run=True)
        o = StepResult(commits, np.zeros(n), conf, tok_pred, np.full(n, 0.5), np.zeros((n, 1)), 0, 0, "cached")
        got = [(c.pos, c.tok, c.conf) for c in commits]
        assert compare.compare_commits(o, masked, tau, got, conf_tol=0.0).exact
        best = np.where(masked, conf, -np.inf).max()
        far = [j for j in range(n) if masked[j] and abs(conf[j] - tau) > 2e-3 and best - conf[j] > 2e-3]
        if far:
            j = far[0]
            flipped = [g for g in got if g[0] != j] if any(g[0] == j for g in got) else got + [(j, int(tok_pred[j]), float(conf[j]))]
            assert compare.compare_commits(o, masked, tau, flipped).n_mismatch >= 1


def test_rel_rows():
    """G14: per-row L2-relative error."""
    want = np.array([[3.0, 4.0], [0.0, 2.0]])
    got = np.array([[3.0, 4.5], [0.0, 2.0]])
    assert np.allclose(compare.rel_rows(got, want), [0.1, 0.0])
    assert compare.rel_rows(np.zeros((1, 2)), np.zeros((1, 2)))[0] == 0.0          # 0/0 guarded
