"""Comparison of a step result produced elsewhere (the CUDA path) with the oracle's, under north_star's
exclusion band (reading G13).  TEST INFRASTRUCTURE ONLY; uses oracle values only.

Band rules, evaluated on the ORACLE's values, band = 1e-3 in probability units:
  (i)   vocabulary top-2 margin at a position < band      -> that position's token id is excluded
  (ii)  |conf_i - tau| < band                              -> that position's membership is excluded
  (iii) when the at-least-one rule decides (no MASK position reaches tau, up to the band), a position whose
        confidence is within band of the best MASK confidence is excluded
"""
from __future__ import annotations

import dataclasses
from typing import List, Sequence, Tuple

import numpy as np

BAND = 1e-3


@dataclasses.dataclass
class CommitDiff:
    exact: bool                 # identical (pos, tok) lists
    n_excluded: int             # differences that fall inside the band
    n_mismatch: int             # differences outside the band
    detail: List[str]


def compare_commits(o, masked_before: np.ndarray, tau: float, got: Sequence[Tuple[int, int]], band: float = BAND) -> CommitDiff:
    """o: oracle StepResult; masked_before[j]: block position j was MASK before the step; got: (pos, tok) list."""
    lo = o.block_lo
    B = len(o.conf)
    want = {c.pos: c.tok for c in o.commits}
    have = {int(p): int(t) for p, t in got}
    exact = sorted(want.items()) == sorted(have.items())
    excl = mism = 0
    detail = []
    mconf = np.where(masked_before, o.conf, -np.inf)
    best = mconf.max() if masked_before.any() else -np.inf
    rule_decides = best < tau + band            # nothing (clearly) reaches the threshold
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
        elif a and want[pos] != have[pos]:
            if o.margin[j] < band:
                excl += 1
            else:
                mism += 1
                detail.append(f"pos {pos}: token oracle={want[pos]} got={have[pos]} margin={o.margin[j]:.6f}")
    return CommitDiff(exact, excl, mism, detail)


def rel_rows(got: np.ndarray, want: np.ndarray) -> np.ndarray:
    """Per-row ||got - want||_2 / ||want||_2 (reading G14)."""
    return np.linalg.norm(got.astype(np.float64) - want, axis=-1) / np.maximum(np.linalg.norm(want, axis=-1), 1e-300)
