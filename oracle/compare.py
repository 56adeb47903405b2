"""Comparison of a step result produced elsewhere (the CUDA path) with the oracle's, under north_star's
exclusion band (reading G13).  TEST INFRASTRUCTURE ONLY; uses oracle values only.

The rule being judged is P:74: among the MASK positions M of the current block (reading G3) commit
C = {i in M : conf_i >= tau} U {argmax_{i in M} conf_i}, token = argmax over the vocabulary.

Band rules, evaluated on the ORACLE's values, band = 1e-3 in probability units (north_star: "excluding positions
whose top-2 margin or distance to the threshold is below 1e-3, which are reported as a count"):
  (i)   vocabulary top-2 margin at a position < band      -> that position's token id is excluded
  (ii)  |conf_i - tau| < band                              -> that position's membership is excluded
  (iii) when the at-least-one rule decides (no MASK position reaches tau, up to the band), a position whose
        confidence is within band of the best MASK confidence is excluded
Never excused by the band (a difference here is a mismatch whatever the confidences are):
  * a commit outside the current block [lo, lo + B)                      (G3: commits stay inside the current block)
  * a commit at a position that was not MASK before the step             (P:74 only masked tokens are unmasked)
  * the same position reported twice
  * no commit at all while the block still holds a MASK                  ("to ensure progress")
  * more than one commit when no MASK confidence comes within band of tau (the at-least-one rule adds ONE position)
Pinned by tests/test_oracle_compare.py (hand-built cases, one per rule).
"""
from __future__ import annotations

import dataclasses
from typing import List, Sequence

import numpy as np

BAND = 1e-3


@dataclasses.dataclass
class CommitDiff:
    exact: bool                 # identical (pos, tok) lists
    n_excluded: int             # differences that fall inside the band
    n_mismatch: int             # differences outside the band
    detail: List[str]
    max_conf_err: float = 0.0   # max |conf_got - conf_oracle| over the commits both sides made (0 when `got` has no conf)
    min_gap: float = float("inf")  # oracle's best-vs-second MASK confidence gap when the at-least-one rule decided (else inf)


def compare_commits(o, masked_before: np.ndarray, tau: float, got: Sequence[tuple], band: float = BAND,
                    conf_tol: float | None = None) -> CommitDiff:
    """o: oracle StepResult; masked_before[j]: block position j was MASK before the step; got: the other side's
    commits as (pos, tok) or (pos, tok, conf).  conf_tol (optional): a commit made by both sides whose confidence
    differs from the oracle's by more than conf_tol is a mismatch."""
    lo = o.block_lo
    B = len(o.conf)
    want = {c.pos: c.tok for c in o.commits}
    have, have_conf = {}, {}
    excl = mism = 0
    detail = []
    for g in got:
        p, t = int(g[0]), int(g[1])
        if p in have:
            mism += 1
            detail.append(f"pos {p}: reported twice")
        have[p] = t
        if len(g) > 2:
            have_conf[p] = float(g[2])
    exact = sorted(want.items()) == sorted(have.items()) and len(have) == len(got)
    for p in sorted(have):
        if not (lo <= p < lo + B):
            mism += 1
            detail.append(f"pos {p}: commit outside the current block [{lo}, {lo + B})")
    mconf = np.where(masked_before, o.conf, -np.inf)
    any_mask = bool(masked_before.any())
    best = mconf.max() if any_mask else -np.inf
    rule_decides = best < tau + band            # nothing (clearly) reaches the threshold
    min_gap = float("inf")
    if any_mask and best < tau:
        rest = np.sort(mconf[np.isfinite(mconf)])
        min_gap = float(rest[-1] - rest[-2]) if len(rest) > 1 else float("inf")
    in_block = [p for p in have if lo <= p < lo + B]
    if any_mask and not in_block:
        mism += 1
        detail.append("no commit although the block holds MASK positions (P:74 at-least-one rule)")
    if any_mask and best <= tau - band and len([p for p in in_block if masked_before[p - lo]]) > 1:
        mism += 1
        detail.append(f"{len(in_block)} commits although no MASK confidence comes within {band} of tau={tau} (best {best:.6f})")
    max_conf_err = 0.0
    for j in range(B):
        pos = lo + j
        a, b = pos in want, pos in have
        if not masked_before[j]:
            if b:
                mism += 1
                detail.append(f"pos {pos}: committed a position that was not MASK")
            continue
        if a != b:
            near_tau = abs(o.conf[j] - tau) < band
            near_best = rule_decides and (best - o.conf[j]) < band
            if near_tau or near_best:
                excl += 1
            else:
                mism += 1
                detail.append(f"pos {pos}: membership oracle={a} got={b} conf={o.conf[j]:.6f} tau={tau} best={best:.6f}")
        elif a:
            if want[pos] != have[pos]:
                if o.margin[j] < band:
                    excl += 1
                else:
                    mism += 1
                    detail.append(f"pos {pos}: token oracle={want[pos]} got={have[pos]} margin={o.margin[j]:.6f}")
            elif pos in have_conf:
                e = abs(have_conf[pos] - float(o.conf[j]))
                max_conf_err = max(max_conf_err, e)
                if conf_tol is not None and e > conf_tol:
                    mism += 1
                    detail.append(f"pos {pos}: confidence oracle={o.conf[j]:.6f} got={have_conf[pos]:.6f} (tolerance {conf_tol})")
    return CommitDiff(exact and mism == 0, excl, mism, detail, max_conf_err, min_gap)


def rel_rows(got: np.ndarray, want: np.ndarray) -> np.ndarray:
    """Per-row ||got - want||_2 / ||want||_2 (reading G14)."""
    return np.linalg.norm(got.astype(np.float64) - want, axis=-1) / np.maximum(np.linalg.norm(want, axis=-1), 1e-300)
