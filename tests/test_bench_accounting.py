"""bench.py's algorithmic-work accounting pinned to SURVEY.md section 8(d)'s table (the roofline denominators of every reported
fraction), and its step-mix helpers.  CPU only."""
import types

import numpy as np

import bench
from synth_inputs import ARCH_LLADA8B, ARCH_QWEN7B, workload_c2


def test_params_per_layer_and_totals_match_the_survey():
    assert round(bench.layer_params(ARCH_LLADA8B) / 1e6, 1) == 218.1           # 218.1 M per layer (LLaDA shape)
    assert round(bench.layer_params(ARCH_QWEN7B) / 1e6, 1) == 233.0            # 233.0 M (Qwen shape)
    assert round(ARCH_LLADA8B.vocab * ARCH_LLADA8B.d_model / 1e6, 1) == 518.0   # LM head 518.0 M


def test_c2_cached_and_refresh_work_match_the_survey_table():
    """SURVEY 8(d) rows "C2 cached" (447 / 33 / 9 GFLOP, 14.99 / 0.27 / 0.02 GB) and "C2 refresh" (7 147 / 33 / 137, 14.99 / 0.27 / 0.27)."""
    a = ARCH_LLADA8B
    c = bench.step_work(a, [32], [512], 32)
    lin = 2 * 32 * bench.layer_params(a) * a.n_layers
    assert round(lin / 1e9) == 447 and round((c["flops_linear"] - lin) / 1e9) == 33 and round(c["flops_attn"] / 1e9) == 9
    assert round(c["weight_bytes"] / 1e9, 2) == 14.99 and round(c["kv_read_bytes"] / 1e9, 2) == 0.27
    assert round((c["bytes"] - c["weight_bytes"] - c["kv_read_bytes"]) / 1e9, 2) == 0.02
    r = bench.step_work(a, [512], [512], 32)
    assert round((r["flops_linear"] - 2 * 32 * a.d_model * a.vocab) / 1e9) == 7147 and round(r["flops_attn"] / 1e9) == 137
    assert round((r["bytes"] - r["weight_bytes"] - r["kv_read_bytes"]) / 1e9, 2) == 0.27
    peaks = {"hbm_gbs": 6437.9, "bf16_tflops": 1692.7, "bf16_tflops_sustained": 1692.7}        # the survey's denominators
    t_c, b_c = bench.roofline_ms(c, peaks)
    t_r, b_r = bench.roofline_ms(r, peaks)
    assert b_c == "hbm" and abs(t_c - 2.37) < 0.01 and b_r == "tensor" and abs(t_r - 4.32) < 0.01


def test_c4_cached_work_matches_the_survey_table():
    """SURVEY 8(d) row "C4 cached (n=8, S=4608, B=64)": 7 147 / 530 / 1 237 GFLOP, 14.99 / 19.33 / 0.27 GB."""
    a = ARCH_LLADA8B
    w = bench.step_work(a, [64] * 8, [4608] * 8, 512)
    assert round(w["flops_attn"] / 1e9) == 1237 and round(w["kv_read_bytes"] / 1e9, 2) == 19.33
    assert round(2 * 512 * a.d_model * a.vocab / 1e9) == 530


def test_step_mix_and_cpu_baseline_mix():
    spec = workload_c2()[0]
    assert bench.nominal_mix(spec, 20) == (1, 19) and bench.nominal_mix(spec, 32) == (1, 31) and bench.nominal_mix(spec, 64) == (2, 62)
    assert bench.nominal_mix(spec, 33) == (2, 31)
    assert abs(bench.mix_steps_per_s(spec, 2.0, 1.0) - 32 / 33.0) < 1e-12
    assert bench.job_value(2, 10, 1e6) == 20.0
