"""Pins for oracle/sched.py: hand-worked numbers for the paper's Alg. 1 / 4 / 5 on a toy
latency profile, interpolation special cases, monotonicity."""
import pytest

from oracle import sched

# toy profile: cached steps cost 1000 us + 10 us per token at K/V 512 (twice that at K/V 2048); refresh 100 us per token
LP = [("cached", 32, 512, 1320.0), ("cached", 64, 512, 1640.0), ("cached", 256, 512, 3560.0),
      ("cached", 32, 2048, 2640.0), ("cached", 256, 2048, 7120.0),
      ("refresh", 512, 512, 51200.0), ("refresh", 1024, 512, 102400.0), ("refresh", 2048, 2048, 204800.0)]


def test_lp_lookup_cases():
    assert sched.lp_lookup(LP, "cached", 32, 512) == 1320.0                 # a stored point
    assert sched.lp_lookup(LP, "cached", 48, 512) == 1480.0                 # midway between 32 and 64
    assert sched.lp_lookup(LP, "cached", 160, 512) == 2600.0                # midway between 64 and 256
    assert sched.lp_lookup(LP, "cached", 8, 512) == 1320.0                  # clamped below
    assert sched.lp_lookup(LP, "cached", 9999, 512) == 3560.0               # clamped above
    assert sched.lp_lookup(LP, "cached", 32, 1900) == 2640.0                # nearest K/V length: 2048
    assert sched.lp_lookup(LP, "cached", 32, 1280) == 1320.0                # tie between 512 and 2048 -> the shorter
    assert sched.lp_lookup(LP, "refresh", 768, 512) == 76800.0
    with pytest.raises(ValueError):
        sched.lp_lookup([r for r in LP if r[0] == "cached"], "refresh", 10, 512)


def test_alg4_load_and_capacity_by_hand():
    # 40 predicted steps left of which 2 are recomputes; 512 tokens; block 32: 38 * 32 + 2 * 512 = 2240 token-steps
    assert sched.req_load(40, 2, 512, 32) == 2240
    assert sched.req_load(2, 2, 512, 32) == 1024                            # only recomputes left
    # capacity: cacheStepLoad = 32 * 8 = 256 -> 3560 us; recompute of 512 tokens -> 51200 us
    # tput = (256 * 31 + 512) / (3560e-6 * 31 + 51200e-6) = 8448 / 0.16156 tokens/s; SLO 10 s
    cap = sched.instance_capacity(LP, 32, 8, 512, 512, 10.0)
    assert abs(cap - 8448 / 0.16156 * 10.0) < 1e-6


def test_alg5_time_left_and_alg1_pick_by_hand():
    # 4 requests on the instance (cache batch 128 tokens -> 1000 + 1280 = 2280 us by interpolation), 1024 tokens in all
    t = sched.time_left(LP, 40, 2, 32, 4, 1024, 512)
    assert abs(t - (2280e-6 * 38 + 2 * 102400e-6)) < 1e-12
    # thresholds 0.95 / 0.9 / 0.7 / 0.5 need 60 / 40 / 25 / 12 more steps
    allowed, steps = [0.95, 0.9, 0.7, 0.5], [60, 40, 25, 12]
    costs = [sched.time_left(LP, s, 2, 32, 4, 1024, 512) for s in steps]
    assert costs == sorted(costs, reverse=True)                             # fewer steps, less time
    assert sched.pick_threshold(allowed, steps, costs[0] + 1e-9, LP, 2, 32, 4, 1024, 512) == 0   # everything fits: highest
    assert sched.pick_threshold(allowed, steps, costs[1], LP, 2, 32, 4, 1024, 512) == 1           # equality fits (<=)
    assert sched.pick_threshold(allowed, steps, (costs[2] + costs[3]) / 2, LP, 2, 32, 4, 1024, 512) == 3
    assert sched.pick_threshold(allowed, steps, 0.0, LP, 2, 32, 4, 1024, 512) == 3                # nothing fits: lowest kept
