"""Host-side consumers of the per-step cost table.  TEST INFRASTRUCTURE ONLY.

Written from the paper's control-plane algorithms, with the readings of their garbled lines (G18):

  Alg. 1  SLO-aware threshold pick: the highest allowed threshold whose predicted time left fits the
                      remaining SLO budget; if none fits, the lowest allowed threshold is kept.
  Alg. 4  ReqLoad = cacheSteps * cacheBlockSize + recompStepsLeft * numTokens, cacheSteps = predicted steps
                      left - recompStepsLeft;  per-instance capacity = tput * SLO with
                      tput = (cacheStepLoad (B-1) + numTokenPerReq) / (cacheStepLat (B-1) + recompStepLat),
                      cacheStepLoad = cacheBlockSize * maxNumSeqPerBatch.
  Alg. 5  PredictedTimeLeft = cacheStepLat * cacheStepsLeft + recompStepsLeft * recompStepLat with
                      cacheStepLat = LP[cacheBlockSize * numReqs], recompStepLat = LP[numTokens].

LP is the latency profile: here the rows of dlm_profile_step_costs (kind, tokens, K/V length, usec)
for one instance (TP degree 1).  Lookup: rows of the wanted kind and of the K/V length nearest to the wanted one
(ties -> the shorter), piecewise-linear in the token count, clamped at both ends.
"""
from __future__ import annotations

from typing import Sequence, Tuple

Row = Tuple[str, int, int, float]      # (kind "refresh" | "cached", tokens, kv per request, usec)


def lp_lookup(rows: Sequence[Row], kind: str, tokens: float, kv: int) -> float:
    cand = [r for r in rows if r[0] == kind]
    if not cand:
        raise ValueError(f"no {kind} rows in the latency profile")
    best_kv = min(sorted({r[2] for r in cand}), key=lambda k: (abs(k - kv), k))
    pts = sorted((r[1], r[3]) for r in cand if r[2] == best_kv)
    if tokens <= pts[0][0]:
        return float(pts[0][1])
    if tokens >= pts[-1][0]:
        return float(pts[-1][1])
    for (t0, u0), (t1, u1) in zip(pts, pts[1:]):
        if t0 <= tokens <= t1:
            return float(u0 + (u1 - u0) * (tokens - t0) / (t1 - t0))
    raise AssertionError("unreachable")


def req_load(pred_steps_left: float, recomp_steps_left: int, num_tokens: int, cache_block: int) -> float:
    """Alg. 4 ReqLoad (token-steps of work left in the request)."""
    cache_steps = pred_steps_left - recomp_steps_left
    return cache_steps * cache_block + recomp_steps_left * num_tokens


def instance_capacity(rows: Sequence[Row], cache_block: int, max_seq_per_batch: int, num_token_per_req: int, kv: int,
                      slo_sec: float) -> float:
    """Alg. 4 ClusterCapacity, one instance: tokens it can process inside the SLO window."""
    cache_step_load = cache_block * max_seq_per_batch
    cache_lat = lp_lookup(rows, "cached", cache_step_load, kv) * 1e-6
    recomp_lat = lp_lookup(rows, "refresh", num_token_per_req, kv) * 1e-6
    tput = (cache_step_load * (cache_block - 1) + num_token_per_req) / (cache_lat * (cache_block - 1) + recomp_lat)
    return tput * slo_sec


def time_left(rows: Sequence[Row], pred_steps_left: float, recomp_steps_left: int, cache_block: int, num_reqs: int,
              num_tokens: int, kv: int) -> float:
    """Alg. 5 PredictedTimeLeft in seconds (cache steps batched together, recompute steps batched together)."""
    cache_lat = lp_lookup(rows, "cached", cache_block * num_reqs, kv) * 1e-6
    recomp_lat = lp_lookup(rows, "refresh", num_tokens, kv) * 1e-6
    return cache_lat * (pred_steps_left - recomp_steps_left) + recomp_steps_left * recomp_lat


def pick_threshold(allowed_desc: Sequence[float], pred_steps_left: Sequence[float], slo_left_sec: float, rows: Sequence[Row],
                   recomp_steps_left: int, cache_block: int, num_reqs: int, num_tokens: int, kv: int) -> int:
    """Alg. 1 UpdateConfThreshold with Alg. 5 as PredictedTimeLeft: index into allowed_desc (thresholds in descending
    order) of the first threshold that fits the budget; the last (lowest) one if none fits."""
    for i, _ in enumerate(allowed_desc):
        if time_left(rows, pred_steps_left[i], recomp_steps_left, cache_block, num_reqs, num_tokens, kv) <= slo_left_sec:
            return i
    return len(allowed_desc) - 1
