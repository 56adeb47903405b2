"""Denoising steps with confidence-threshold unmasking and approximate (block-wise, prefix+suffix)
KV caching.  TEST INFRASTRUCTURE ONLY.  Follows, in the paper's order:

  P:74   "at each denoising step unmasks only those tokens whose confidence exceeds a predefined
          threshold.  If no predicted tokens have confidence exceeding the threshold, the token with the
          highest confidence is unmasked to ensure progress."
  P:109  "partition the output sequence into blocks ... process them sequentially ... cache and reuse the
          KV tensors for the prefix and suffix blocks throughout the denoising steps of the current block
          ... the KV tensors for all blocks are recomputed after the current block is fully unmasked"
  P:347  "cache steps compute only the tokens inside the current cache block, while recompute steps
          process all tokens in the sequence"
  P:582  a block = (cacheBlockSize - 1) cache steps and one recompute step  => every step, the recompute
          (here "refresh") step included, ends with an unmask (reading G4).

Readings: G1 threshold test is conf >= tau; G3 the at-least-one rule and the threshold test
range over the MASK positions of the CURRENT block only; G8 ties -> lowest position / lowest id;
current block = lowest-index block that still holds a MASK.
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional

import numpy as np

from . import model


@dataclasses.dataclass
class Commit:
    pos: int       # absolute position in prompt||generation
    tok: int
    conf: float


@dataclasses.dataclass
class StepResult:
    commits: List[Commit]
    lse: np.ndarray            # [B] log-sum-exp of the block rows' logits
    conf: np.ndarray           # [B] confidence of every block row
    tok: np.ndarray            # [B] predicted token of every block row
    margin: np.ndarray         # [B] top-1 minus top-2 probability (near-tie band, G13)
    hidden: np.ndarray         # [B, d] last layer's residual output on the block rows
    block_lo: int
    n_masked_left: int         # MASK positions left in the whole request after the step
    kind: str


class Request:
    def __init__(self, arch, prompt, gen_len: int, block_len: int, threshold: float, tokens=None):
        assert gen_len % block_len == 0, "G20: generation length must be a multiple of the block length"
        self.arch = arch
        self.P, self.G, self.B = len(prompt), int(gen_len), int(block_len)
        self.S = self.P + self.G
        self.threshold = float(threshold)
        if tokens is None:
            # P:40 "starting from a fully corrupted sequence containing only [MASK] tokens"
            tokens = np.concatenate([np.asarray(prompt, dtype=np.int64),
                                     np.full(self.G, arch.mask_id, dtype=np.int64)])
        self.tokens = np.asarray(tokens, dtype=np.int64).copy()
        assert len(self.tokens) == self.S
        self.cache = None            # per layer (K, V) float64, valid from a refresh until the block completes
        self.cache_valid = False
        # Step Predictor inputs ("confidence statistics ... tracked by the Scheduler", App. A; reading G22):
        self.conf_state = np.zeros(self.G, dtype=np.float64)   # per output position: last confidence seen while masked
        self.steps_done = 0                                    # completed (non-dry) denoising steps

    def migrate(self) -> "Request":
        """The request as another instance receives it ("migrated ... only at recompute steps"; P:365 the command
        carries the request's tokens): everything except the K/V cache, which the receiver recomputes."""
        r = Request(self.arch, self.tokens[:self.P], self.G, self.B, self.threshold, tokens=self.tokens)
        r.conf_state = self.conf_state.copy()
        r.steps_done = self.steps_done
        return r

    def masked(self) -> np.ndarray:
        return self.tokens == self.arch.mask_id

    def n_masked(self) -> int:
        return int(self.masked().sum())

    def current_block(self) -> Optional[int]:
        """Lowest-index block containing a MASK; None when the request is finished."""
        m = self.masked()[self.P:].reshape(-1, self.B).any(axis=1)
        idx = np.flatnonzero(m)
        return int(idx[0]) if len(idx) else None

    def block_range(self, b: int):
        return self.P + b * self.B, self.P + (b + 1) * self.B


def unmask(tokens: np.ndarray, lo: int, hi: int, tok: np.ndarray, conf: np.ndarray, tau: float,
           mask_id: int, dry_run: bool = False) -> List[Commit]:
    """P:74.  M = MASK positions in [lo, hi).  C = {i in M: conf_i >= tau} U {argmax_{i in M} conf_i}
    (lowest i on ties).  tokens[i] = tok_i for i in C.  Returns commits in ascending position."""
    M = [i for i in range(lo, hi) if tokens[i] == mask_id]
    if not M:
        return []
    best = M[0]
    for i in M[1:]:
        if conf[i - lo] > conf[best - lo]:
            best = i
    C = [i for i in M if conf[i - lo] >= tau or i == best]
    out = [Commit(i, int(tok[i - lo]), float(conf[i - lo])) for i in C]
    if not dry_run:
        for c in out:
            tokens[c.pos] = c.tok
    return out


def _finish(req: Request, b: int, hidden: np.ndarray, tau: float, dry_run: bool, kind: str, wts) -> StepResult:
    lo, hi = req.block_range(b)
    tok, conf, lse, margin = model.head(req.arch, wts, hidden)
    if not dry_run:
        was_masked = req.tokens[lo:hi] == req.arch.mask_id   # G22: live while masked, frozen at commit
        req.conf_state[lo - req.P:hi - req.P][was_masked] = conf[was_masked]
        req.steps_done += 1
    commits = unmask(req.tokens, lo, hi, tok, conf, tau, req.arch.mask_id, dry_run)
    if not dry_run and not (req.tokens[lo:hi] == req.arch.mask_id).any():
        req.cache_valid = False          # P:109 recompute "after the current block is fully unmasked"
    return StepResult(commits, lse, conf, tok, margin, hidden, lo, req.n_masked(), kind)


def refresh_step(req: Request, wts, tau: Optional[float] = None, dry_run: bool = False) -> Optional[StepResult]:
    """Recompute step: all S positions pass through the model, every layer's K (post-RoPE) and V are
    stored as the request's cache, then the current block is unmasked.  Legal at any time (G19)."""
    b = req.current_block()
    if b is None:
        return None
    tau = req.threshold if tau is None else float(tau)
    hidden, kv = model.full_forward(req.arch, wts, req.tokens)
    req.cache, req.cache_valid = kv, True
    lo, hi = req.block_range(b)
    return _finish(req, b, hidden[lo:hi], tau, dry_run, "refresh", wts)


def cached_step(req: Request, wts, tau: Optional[float] = None, dry_run: bool = False) -> Optional[StepResult]:
    """Cache step: only the current block's B positions are computed; they attend to their own fresh
    K/V plus the cached K/V of every other position."""
    b = req.current_block()
    if b is None:
        return None
    if not req.cache_valid:
        raise RuntimeError("cached step without a valid cache (G19): a refresh step is due")
    tau = req.threshold if tau is None else float(tau)
    lo, hi = req.block_range(b)
    hidden, fresh = model.cached_forward(req.arch, wts, req.tokens, lo, hi, req.cache)
    if not dry_run:
        for l, (k, v) in enumerate(fresh):     # G6: the block's slots are overwritten in place
            req.cache[l][0][lo:hi] = k
            req.cache[l][1][lo:hi] = v
    return _finish(req, b, hidden, tau, dry_run, "cached", wts)


FEATURE_NAMES = ("confidence_threshold", "output_length", "full_progress", "full_unmask_progress", "block_progress",
                 "block_unmask_progress", "output_min_confidence", "output_q25_confidence", "output_median_confidence",
                 "output_avg_confidence", "output_q75_confidence")


def quantile_linear(sorted_vals: np.ndarray, q: float) -> float:
    """q-quantile of ascending values by linear interpolation between order statistics: h = (n - 1) q,
    v = s[floor h] + (h - floor h) (s[floor h + 1] - s[floor h])."""
    n = len(sorted_vals)
    h = (n - 1) * q
    lo = int(np.floor(h))
    hi = min(lo + 1, n - 1)
    return float(sorted_vals[lo] + (h - lo) * (sorted_vals[hi] - sorted_vals[lo]))


def predictor_features(req: Request, tau: Optional[float] = None) -> np.ndarray:
    """The Step Predictor's 11 scalar features of a request in its current state (App. A), in the
    paper's order (FEATURE_NAMES).  Reading G22: an output token's confidence is the softmax confidence the
    model last gave its position while it was still masked (so it is frozen when the token is committed), 0
    for positions no step has evaluated yet; quartiles by linear interpolation; a finished request reports
    block_progress = block_unmask_progress = 1."""
    tau = req.threshold if tau is None else float(tau)
    G, B = req.G, req.B
    n_blocks = G // B
    b = req.current_block()
    masked = req.masked()[req.P:]
    if b is None:
        block_progress, block_unmask = 1.0, 1.0
    else:
        block_progress = b / n_blocks
        block_unmask = float((~masked[b * B:(b + 1) * B]).sum()) / B
    s = np.sort(req.conf_state)
    return np.array([tau, G, req.steps_done / G, float((~masked).sum()) / G, block_progress, block_unmask,
                     s[0], quantile_linear(s, 0.25), quantile_linear(s, 0.5), float(req.conf_state.sum() / G), quantile_linear(s, 0.75)],
                    dtype=np.float64)


def next_step(req: Request, wts, tau: Optional[float] = None, use_cache: bool = True) -> Optional[StepResult]:
    """The step that is due: refresh at a block's first step (or always, without caching), else cached."""
    if req.current_block() is None:
        return None
    if use_cache and req.cache_valid:
        return cached_step(req, wts, tau)
    return refresh_step(req, wts, tau)


def run(req: Request, wts, use_cache: bool = True, tau_schedule=None, max_steps: int = 1 << 30):
    """Denoise to completion ("continues until no [MASK] tokens remain", G21: no early stop).
    tau_schedule(step_index) -> tau allows a per-step threshold."""
    hist = []
    while req.current_block() is not None and len(hist) < max_steps:
        tau = None if tau_schedule is None else tau_schedule(len(hist))
        hist.append(next_step(req, wts, tau, use_cache))
    return hist
