#!/usr/bin/env python3
"""bench.py -- denoising-step throughput of libdlm on B200 (BASELINE.json metric: denoise steps/s and committed
tokens/s on 1 B200, LLaDA-8B shape; % of roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C2|C3|C4|C5] [--impl ours|reference]

A "step" is one denoising step of the workload's batch through the whole hot path (DESIGN.md rows a0-a14): refresh
steps where a block starts, cached steps inside a block, exactly as the free-running trajectory demands.  After the
warm-up the run advances (untimed) to the next block boundary, so the K timed steps start with the refresh step of a
block and contain both step kinds in the workload's own proportion (`config.step_mix`).
`value`  = steps / device time (CUDA events on the library's stream around each step's kernels, inputs resident).
`e2e`    = steps / wall time of the same C-ABI calls with HOST buffers (request upload, per-step descriptor H2D,
           result D2H and the synchronize all inside the timed region).
`step_roofline` = per step kind, measured ms against the step's roofline (sum of rooflines / sum of times), plus the
           block-cycle figure (1 refresh + B-1 cached steps).
`roofline` = the dominant kernel class of the cached steps (the weight-streaming / CTA-pair tcgen05 GEMMs), timed INSIDE the
           production launch (CUDA graph + programmatic dependent launch) by the library's in-kernel %globaltimer trace
           (DLM_OPT_TRACE): a launch's time = wait(next launch) - wait(this launch), so the classes add up to the step.
`kernels`  = the same attribution for every kernel class, with achieved HBM GB/s of attention (K/V bytes) and of the
           combine + unmask pass (LM-head partials).
`cpu_baseline` = the fp64 oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample, for the same
           mix of step kinds as the timed region.
N > 1: one process per GPU (torchrun), independent replicas of the workload (requests are independent, P:426
"16 TP-1 workers"), no data-path collective; time = max over ranks; scaling "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from synth_inputs import (ARCH_LLADA8B, ARCH_QWEN7B, WEIGHT_SEED, initial_tokens, workload_c2, workload_c3,  # noqa: E402
                          workload_c4, workload_c5)

FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "source": "measured"}
    return dict(FALLBACK_PEAKS, source="fallback")


# ---------------------------------------------------------------------------------------------------------
# algorithmic work of a step: what the method must move / multiply
# ---------------------------------------------------------------------------------------------------------
def layer_params(a):
    return a.d_model * (a.n_heads + 2 * a.n_kv_heads) * a.head_dim + a.n_heads * a.head_dim * a.d_model + 3 * a.d_model * a.d_ffn


def step_work(a, q_lens, kv_lens, rows):
    """FLOPs and HBM bytes of one step: q_lens[i] tokens of request i computed against kv_lens[i] positions."""
    T, R = sum(q_lens), rows
    L = a.n_layers
    kv_tok = 4 * a.n_kv_heads * a.head_dim                       # bytes of K and V per token per layer (bf16)
    flops_lin = 2 * T * layer_params(a) * L
    flops_lm = 2 * R * a.d_model * a.vocab
    flops_attn = 4 * sum(q * s for q, s in zip(q_lens, kv_lens)) * a.n_heads * a.head_dim * L
    bytes_w = 2 * (layer_params(a) * L + a.vocab * a.d_model)
    bytes_kv_rd = sum(kv_lens) * kv_tok * L
    bytes_kv_wr = T * kv_tok * L
    return {"flops": flops_lin + flops_lm + flops_attn, "bytes": bytes_w + bytes_kv_rd + bytes_kv_wr,
            "weight_bytes": bytes_w, "kv_read_bytes": bytes_kv_rd, "flops_linear": flops_lin + flops_lm, "flops_attn": flops_attn}


def roofline_ms(work, peaks, sustained=True):
    tf = peaks["bf16_tflops_sustained" if sustained else "bf16_tflops"] * 1e12
    t_f = work["flops"] / tf
    t_b = work["bytes"] / (peaks["hbm_gbs"] * 1e9)
    return 1e3 * max(t_f, t_b), ("tensor" if t_f > t_b else "hbm")


def burst_applies(clocks):
    """Which tensor peak a tensor-bound step is scored against: the BURST figure when the sampled SM clock stayed within 5 % of
    its maximum and no power cap was seen during the timed region (a step that runs at full clock between HBM-bound steps),
    else the SUSTAINED one (seconds of back-to-back GEMMs under sw_power_cap).  HBM-bound steps do not depend on it."""
    mhz, mx = clocks.get("sm_mhz"), clocks.get("sm_max_mhz")
    if not mhz or not mx:
        return False
    return mhz >= 0.95 * mx and "sw_power_cap" not in clocks.get("reasons", [])


# ---------------------------------------------------------------------------------------------------------
# clocks during the timed region
# ---------------------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                    else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                for bit, name in self.REASONS.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.05)

    def __enter__(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": int(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------------------
# workloads
# ---------------------------------------------------------------------------------------------------------
def get_workload(name: str):
    if name == "C2":
        return ARCH_LLADA8B, WEIGHT_SEED["C2"], workload_c2(), "configs[1]: LLaDA-8B shape, batch 1, prompt 256, gen 256, block 32, tau 0.9"
    if name == "C3":
        return ARCH_LLADA8B, WEIGHT_SEED["C3"], workload_c3(), "configs[2]: LLaDA-8B shape, ragged batch 32, prompts U[128,1024], gen 256, block 32, mixed tau/phases"
    if name == "C4":
        return ARCH_LLADA8B, WEIGHT_SEED["C4"], workload_c4(), "configs[3]: LLaDA-8B shape, batch 8, prompt 4096, gen 512, block 64, tau 0.9"
    if name == "C5":
        return ARCH_QWEN7B, WEIGHT_SEED["C5"], workload_c5(), "configs[4]: Qwen2.5-7B shape (GQA 28/4), batch 64, prompts U[256,2048], gen 256, block 32"
    raise SystemExit(f"unknown workload {name}")


class Runner:
    """Drives a batch of requests through libdlm the way the paper's scheduler would: every
    request gets the step kind that is due; refresh and cached requests of one iteration go in two calls."""

    def __init__(self, pkg, arch, seed, specs, mixed_launch=True):
        self.pkg, self.arch, self.specs, self.mixed_launch = pkg, arch, specs, mixed_launch
        max_seq = max(len(s.prompt) + s.gen_len for s in specs)
        max_seq = (max_seq + 63) // 64 * 64
        self.max_block = max(s.block_len for s in specs)
        tot = sum(len(s.prompt) + s.gen_len for s in specs)
        self.eng = pkg.Engine(arch, seed, max_requests=len(specs), max_seq=max_seq, max_block=self.max_block,
                              max_batch_tokens=max(tot, 128))
        self.ids = [None] * len(specs)
        self.h2d = 0
        self.d2h = 0
        # host-side mirror of what the scheduler knows about each request (it decides the step kind from the tokens it was
        # sent back): MASK positions left in total and in the current block, and whether the cache it built is still valid --
        # no dlm_request_info round trip per request and step
        self.left, self.blk_left, self.valid = [0] * len(specs), [0] * len(specs), [False] * len(specs)
        for i in range(len(specs)):
            self._add(i)

    def _add(self, i):
        s = self.specs[i]
        if self.ids[i] is not None:
            self.eng.remove_request(self.ids[i])
        self.ids[i] = self.eng.add_request(s.prompt, s.gen_len, s.block_len, s.threshold)
        self.h2d += 4 * (len(s.prompt) + s.gen_len)
        if s.filled is not None and len(s.filled):
            self.eng.set_tokens(self.ids[i], initial_tokens(s, self.arch.mask_id))
            self.h2d += 4 * (len(s.prompt) + s.gen_len)
        self._sync_state(i)

    def _sync_state(self, i):
        """Mirror of request i from the library (at submission, and if the mirror is ever contradicted)."""
        s = self.specs[i]
        st = self.eng.info(self.ids[i])
        self.left[i], self.valid[i] = st["n_masked"], st["cache_valid"]
        lo = len(s.prompt) + st["cur_block"] * s.block_len
        self.blk_left[i] = int((self.eng.tokens(self.ids[i])[lo:lo + s.block_len] == self.arch.mask_id).sum()) if st["n_masked"] else 0

    def step(self):
        """One denoising step of the whole batch.  Returns (device_usec, commits, n_refresh_reqs, n_cached_reqs, work)."""
        eng = self.eng
        refresh, cached = [], []
        for i in range(len(self.ids)):
            if self.left[i] == 0:               # finished: the client submits it again (prompt upload inside the region)
                self._add(i)
            (cached if self.valid[i] else refresh).append(i)
        usec, commits = 0.0, 0
        q_lens, kv_lens, rows = [], [], 0
        if refresh and cached and self.mixed_launch:
            calls = (("mixed", refresh + cached),)          # one ragged launch, weights streamed once (dlm_mixed_step)
        else:
            calls = (("refresh", refresh), ("cached", cached))
        for kind, idx in calls:
            if not idx:
                continue
            rids = [self.ids[i] for i in idx]
            is_ref = set(refresh)
            g = eng.refresh_step(rids) if kind == "refresh" else (eng.cached_step(rids) if kind == "cached" else eng.mixed_step(rids))
            usec += g.usec
            commits += g.total
            for j, i in enumerate(idx):         # the block completes when its last MASK goes: the next step of it is a recompute step
                self.left[i] = int(g.n_masked_left[j])
                self.blk_left[i] -= int(g.n_committed[j])
                self.valid[i] = self.blk_left[i] > 0
                if self.blk_left[i] <= 0:
                    self.blk_left[i] = min(self.specs[i].block_len, self.left[i])
            self.h2d += 4 * (10 * len(rids) + sum((len(self.specs[i].prompt) + self.specs[i].gen_len) if (kind == "refresh" or (kind == "mixed" and i in is_ref))
                                                   else self.specs[i].block_len for i in idx))
            self.d2h += 4 * (len(self.specs) + 6 * len(self.specs) * self.max_block)
            for i in idx:
                s = self.specs[i]
                S = len(s.prompt) + s.gen_len
                q_lens.append(S if (kind == "refresh" or (kind == "mixed" and i in is_ref)) else s.block_len)
                kv_lens.append(S)
                rows += s.block_len
        return usec, commits, len(refresh), len(cached), step_work(self.arch, q_lens, kv_lens, rows)

    def close(self):
        self.eng.close()


# ---------------------------------------------------------------------------------------------------------
# the CPU oracle, timed as it stands on a bounded sample (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------------------
def oracle_sample(arch, seed, spec, layers: int, n_cached: int):
    """Time the fp64 oracle on the first `layers` layers (+ the LM head) of one request: one refresh step and
    `n_cached` cached steps.  Returns per-step seconds extrapolated to the full depth (layer time x L/layers)."""
    from oracle import model as omodel, step as ostep, weights as ow
    sub = arch.replace(n_layers=layers)
    wts = ow.Weights(sub, seed)
    t0 = time.perf_counter()
    for l in range(layers):                       # weight generation is set-up, not part of the step
        for s in range(7):
            wts.f32(ow.layer_tid(l, s))
    wts.f32(ow.TID_LMHEAD)
    t_gen = time.perf_counter() - t0
    req = ostep.Request(sub, spec.prompt, spec.gen_len, spec.block_len, spec.threshold)
    if spec.filled is not None and len(spec.filled):
        req.tokens[:] = initial_tokens(spec, arch.mask_id)
    lo, hi = req.block_range(req.current_block())
    t0 = time.perf_counter()
    hidden, kv = omodel.full_forward(sub, wts, req.tokens)
    t_ref_layers = time.perf_counter() - t0
    req.cache, req.cache_valid = kv, True
    t0 = time.perf_counter()
    tok, conf, lse, margin = omodel.head(sub, wts, hidden[lo:hi])
    ostep.unmask(req.tokens, lo, hi, tok, conf, spec.threshold, arch.mask_id)
    t_head = time.perf_counter() - t0
    t_cached_layers = []
    for _ in range(n_cached):
        if req.current_block() is None or not (req.tokens[lo:hi] == arch.mask_id).any():
            break
        t0 = time.perf_counter()
        hidden, _ = omodel.cached_forward(sub, wts, req.tokens, lo, hi, req.cache)
        t_cached_layers.append(time.perf_counter() - t0)
        tok, conf, lse, margin = omodel.head(sub, wts, hidden)
        ostep.unmask(req.tokens, lo, hi, tok, conf, spec.threshold, arch.mask_id)
    f = arch.n_layers / layers
    t_cached = (float(np.mean(t_cached_layers)) if t_cached_layers else 0.0) * f + t_head
    return {"t_refresh": t_ref_layers * f + t_head, "t_cached": t_cached, "t_gen": t_gen, "n_cached": len(t_cached_layers)}


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([int(p.get("num_threads", 1)) for p in threadpool_info()] or [os.cpu_count() or 1])
    except Exception:
        return os.cpu_count() or 1


def mix_steps_per_s(spec, t_refresh, t_cached):
    """steps/s of the block cycle the workload runs: 1 refresh + (B - 1) cached steps."""
    b = spec.block_len
    return b / (t_refresh + (b - 1) * t_cached)


def nominal_mix(spec, steps):
    """Step kinds of `steps` steps that start at a block boundary in the paper's worst-case block shape: one recompute step
    and B - 1 cache steps per block."""
    n_refresh = (steps + spec.block_len - 1) // spec.block_len
    return n_refresh, steps - n_refresh


def cpu_baseline(arch, seed, specs, layers=1, n_cached=2, mix=None):
    """The oracle on request 0, one layer + the LM head, extrapolated to the full depth; steps/s of the batch for the given
    (refresh request-steps, cached request-steps) mix -- the oracle processes requests one after the other."""
    spec = specs[0]
    o = oracle_sample(arch, seed, spec, layers, n_cached)
    n = len(specs)
    n_ref, n_cac = mix if mix is not None else (1, spec.block_len - 1)
    batch_steps = (n_ref + n_cac) / n
    value = batch_steps / (n_ref * o["t_refresh"] + n_cac * o["t_cached"])
    return {"value": value, "unit": "steps/s", "cores": blas_threads(), "kind": "oracle",
            "sample": f"fp64 numpy oracle, request 0 of {n}, first {layers} of {arch.n_layers} layers + LM head: 1 refresh step and "
                      f"{o['n_cached']} cached steps timed, layer time x{arch.n_layers // layers}; mix of {n_ref} refresh + {n_cac} cached request-steps"
                      + (f" = {batch_steps:g} steps of the {n}-request batch, requests processed serially" if n > 1 else ""),
            "t_refresh_s": round(o["t_refresh"], 3), "t_cached_s": round(o["t_cached"], 3), "weight_gen_s": round(o["t_gen"], 1)}


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores; each step = one bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    arch, seed, specs, desc = get_workload(args.workload)
    steps, warm = max(1, args.steps), max(0, args.warmup)
    vals = []
    mix = nominal_mix(specs[0], steps) if len(specs) == 1 else None
    for i in range(warm + steps):
        cb = cpu_baseline(arch, seed, specs, layers=1, n_cached=1, mix=mix)
        if i >= warm:
            vals.append(cb)
    v = float(np.mean([c["value"] for c in vals]))
    out = {"impl": "reference", "metric": "denoise_steps_per_s", "value": v, "unit": "steps/s", "n_gpus": args.gpus, "steps": steps,
           "warmup": warm, "ms_per_step": 1e3 / v, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic", "config": {"workload": f"{args.workload}: {desc}", "step_mix": None if mix is None else {"refresh": mix[0], "cached": mix[1]}},
           "cpu_baseline": {"value": v, "unit": "steps/s", "cores": vals[-1]["cores"], "kind": "oracle", "sample": vals[-1]["sample"]},
           "e2e": {"value": v, "unit": "steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out), flush=True)


def run_lmhead_micro(args):
    """BASELINE.json configs[4]: isolated micro-benchmark of the fused LM-head + softmax-max + argmax + unmask path on
    unit-RMS random hidden states [2048, 3584] (64 requests x 32 block rows) against the Qwen-shape vocabulary matrix
    [152064, 3584]: rows a11-a13 only, logits never written.  One JSON line (not the headline metric)."""
    import torch
    import paper_2606_29094_b200 as pkg
    from synth_inputs import unit_rms_hidden
    peaks = load_peaks()
    a = ARCH_QWEN7B
    n, B = 64, 32
    R, K, V = n * B, a.d_model, a.vocab
    hidden = torch.from_numpy(unit_rms_hidden(2005, R, K)).to(torch.bfloat16).cuda()
    g = torch.Generator(device="cuda").manual_seed(WEIGHT_SEED["C5"])
    W = (torch.randn(V, K, device="cuda", generator=g) * a.init_std).to(torch.bfloat16)
    tau = torch.full((n,), 0.9, device="cuda")
    tokens0 = torch.full((n, B), a.mask_id, dtype=torch.int32, device="cuda")
    scratch = torch.empty(pkg.lib().dlm_op_lmhead_scratch_bytes(R, V), device="cuda", dtype=torch.uint8)
    outs = (torch.empty(n, device="cuda", dtype=torch.int32), torch.empty(R, device="cuda", dtype=torch.int32),
            torch.empty(R, device="cuda", dtype=torch.int32), torch.empty(R, device="cuda", dtype=torch.float32))
    K_steps, Wm = max(1, args.steps), max(3, args.warmup)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2 * K_steps)]
    committed = 0
    with ClockSampler(0) as clk:
        for i in range(Wm + K_steps):
            tio = tokens0.clone()
            if i >= Wm:
                ev[2 * (i - Wm)].record()
            pkg.op_lmhead_unmask_bf16(hidden, W, n, B, a.logit_scale, a.mask_id, tau, tio, scratch=scratch, outs=outs)
            if i >= Wm:
                ev[2 * (i - Wm) + 1].record()
        torch.cuda.synchronize()
        committed = int(outs[0].sum().item())
    ms = [ev[2 * i].elapsed_time(ev[2 * i + 1]) for i in range(K_steps)]
    t = float(np.mean(ms)) * 1e-3
    flops = 2.0 * R * K * V
    ach = flops / t * 1e-12
    out = {"metric": "lmhead_unmask_micro_tflops", "value": ach, "unit": "TFLOP/s", "n_gpus": 1, "steps": K_steps, "warmup": Wm, "ms_per_step": t * 1e3,
           "higher_is_better": True, "dtype": "bf16", "data": "synthetic",
           "config": {"workload": "C5 micro: fused LM head + split-vocab (max, sum-exp, argmax) + combine + threshold unmask, hidden [2048, 3584] x W [152064, 3584], 64 requests x 32 rows, tau 0.9",
                      "l2": "the vocabulary matrix (1.09 GB) is larger than L2", "timing": "CUDA events around the C-ABI op (includes its 1 KB descriptor copy)"},
           "roofline": {"bound": "tensor", "achieved": ach, "peak": peaks["bf16_tflops"], "unit": "TFLOP/s", "frac": ach / peaks["bf16_tflops"], "traffic": None,
                        "kernel": "gemm_pair_kernel<LM head> + combine_unmask_kernel", "peak_source": peaks["source"] + " (burst: kernel timed alone)"},
           "logits_bytes_avoided": R * V * 4 * 2, "logits_time_avoided_ms_at_hbm_peak": R * V * 4 * 2 / (peaks["hbm_gbs"] * 1e9) * 1e3,
           "committed_rows": committed, "clocks": clk.summary()}
    print(json.dumps(out), flush=True)


def run_cost_table(args):
    """a15: dlm_profile_step_costs on the workload's architecture -- the per-step cost table the paper's scheduler
    consumes (LP[tp][tokens]), split by step kind, with the K/V length added; plus the per-token
    costs alpha (refresh) and beta (cached) of P:349."""
    import torch
    import paper_2606_29094_b200 as pkg
    arch, seed, specs, desc = get_workload(args.workload)
    eng = pkg.Engine(arch, seed, max_requests=64, max_seq=4608, max_block=32, max_batch_tokens=32768)
    rows = eng.profile_step_costs(cap=256)
    eng.close()
    table = [{"kind": r["kind"], "n": r["n_requests"], "tokens": r["n_tokens"], "kv": r["kv_tokens"], "usec": round(r["usec"], 1)} for r in rows]
    ref = [r for r in table if r["kind"] == "refresh"]
    cac = [r for r in table if r["kind"] == "cached"]
    out = {"metric": "step_cost_table", "unit": "usec", "data": "synthetic", "config": {"workload": f"{args.workload} architecture: {desc}"},
           "rows": table,
           "alpha_usec_per_token_refresh": round(float(np.median([r["usec"] / r["tokens"] for r in ref])), 3) if ref else None,
           "beta_usec_per_token_cached": round(float(np.median([r["usec"] / r["tokens"] for r in cac])), 3) if cac else None}
    print(json.dumps(out), flush=True)


def reduce_over_ranks(dist, device, dev_us, wall, commits, launches):
    """Replicas-only scaling: every rank runs its own replica of the workload with no data-path
    collective; the job's time is the MAX over ranks (device and wall clock), its commits and launches the SUM."""
    import torch
    t = torch.tensor([dev_us, wall], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([commits, launches], device=device, dtype=torch.float64)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t[0]), float(t[1]), int(c[0]), int(c[1])


def job_value(world, steps, dev_us):
    """Whole-job steps/s of `world` replicas that each ran `steps` steps, timed as the slowest rank."""
    return world * steps / (dev_us * 1e-6)


def kind_roofline(rs, peaks, burst):
    """Measured time of the steps `rs` (one step kind) against the sum of their rooflines.  `frac` uses the tensor peak that
    applies to the run (burst_applies); frac_burst / frac_sustained give both, they differ only for tensor-bound steps."""
    n = len(rs)
    t_meas = sum(r["us"] for r in rs) * 1e-3
    roofs = {sus: [roofline_ms(r["work"], peaks, sustained=sus) for r in rs] for sus in (True, False)}
    t_sus, t_bur = sum(x[0] for x in roofs[True]), sum(x[0] for x in roofs[False])
    used = roofs[not burst]
    bounds = sorted({x[1] for x in used})
    t_roof = t_bur if burst else t_sus
    return {"n": n, "ms": t_meas / n, "ms_min": min(r["us"] for r in rs) * 1e-3, "roofline_ms": t_roof / n,
            "bound": bounds[0] if len(bounds) == 1 else "mixed", "frac": t_roof / t_meas, "frac_burst": t_bur / t_meas, "frac_sustained": t_sus / t_meas,
            "tensor_peak_used": "burst" if burst else "sustained",
            "gflop": sum(r["work"]["flops"] for r in rs) / n * 1e-9, "gbytes": sum(r["work"]["bytes"] for r in rs) / n * 1e-9}


def other_workload(pkg, name, steps, warm, peaks, clk_index):
    """A short run of another BASELINE.json config inside the default line: `steps` timed steps after `warm`
    untimed ones, per step kind the measured ms against the step's roofline, with the run's own clock record."""
    arch, seed, specs, desc = get_workload(name)
    run = Runner(pkg, arch, seed, specs)
    try:
        for _ in range(warm):
            run.step()
        recs, wall, clocks = timed_steps(run, steps, clk_index)
    finally:
        run.close()
    burst = burst_applies(clocks)
    us = sum(r["us"] for r in recs)
    kinds = {}
    for kind in ("refresh", "cached", "mixed"):
        rs = [r for r in recs if r["kind"] == kind]
        if rs:
            kinds[kind] = kind_roofline(rs, peaks, burst)
    return {"workload": desc, "steps": steps, "warmup": warm, "ms_per_step": us / steps * 1e-3, "steps_per_s": steps / (us * 1e-6),
            "e2e_steps_per_s": steps / wall, "committed_tokens_per_s": sum(r["commits"] for r in recs) / (us * 1e-6),
            "frac": sum(roofline_ms(r["work"], peaks, sustained=not burst)[0] for r in recs) / (us * 1e-3), "step_roofline": kinds, "clocks": clocks}


# ---------------------------------------------------------------------------------------------------------
def at_block_boundary(run):
    """True when the step that is due opens a block for the workload's first request (its K/V cache is not valid)."""
    return run.left[0] == 0 or not run.valid[0]


def timed_steps(run, K, clk_index):
    """K steps, device time summed from the library's per-step CUDA events; returns the per-step records."""
    recs = []
    with ClockSampler(clk_index) as clk:
        import torch
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(K):
            us, cm, nr, nc, work = run.step()
            recs.append({"us": us, "commits": cm, "n_refresh": nr, "n_cached": nc, "work": work,
                         "kind": "mixed" if (nr and nc) else ("refresh" if nr else "cached")})
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
    return recs, wall, clk.summary()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=64)
    ap.add_argument("--warmup", type=int, default=8)
    ap.add_argument("--workload", default="C2")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-kernel-pass", action="store_true")
    ap.add_argument("--no-other-workloads", action="store_true", help="C2 only: skip the short C4 / C3 / C5 runs the default line appends")
    ap.add_argument("--micro", default=None, choices=["lmhead"], help="isolated micro-benchmark instead of the step benchmark")
    ap.add_argument("--cost-table", action="store_true", help="print dlm_profile_step_costs for the workload's architecture")
    ap.add_argument("--two-call", action="store_true", help="mixed iterations as dlm_refresh_step + dlm_cached_step instead of one dlm_mixed_step")
    ap.add_argument("--tau", type=float, default=None, help="override every request's confidence threshold")
    ap.add_argument("--trace-rows", type=int, default=0, help="add the first N launches of one traced step (begin / wait / end in us) to the JSON line")
    ap.add_argument("--layer-kernel", action="store_true", help="run cached steps of <= 64 tokens through the whole-stack persistent kernel (DLM_OPT_LAYER_KERNEL) and report its phase times")
    ap.add_argument("--tau-sweep", action="store_true", help="add a sweep over the paper's candidate thresholds (P:123; BASELINE.json configs[4]: 0.5-0.95)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.micro == "lmhead":
        return run_lmhead_micro(args)
    if args.cost_table:
        return run_cost_table(args)

    import torch
    rank, world, local = (int(os.environ.get(k, d)) for k, d in (("RANK", "0"), ("WORLD_SIZE", "1"), ("LOCAL_RANK", "0")))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libdlm has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2606_29094_b200 as pkg
    arch, seed, specs, desc = get_workload(args.workload)
    if args.tau is not None:
        for sp in specs:
            sp.threshold = float(args.tau)
    peaks = load_peaks()
    K, W = max(1, args.steps), max(3, args.warmup)

    run = Runner(pkg, arch, seed, specs, mixed_launch=not args.two_call)
    if args.layer_kernel:
        run.eng.set_option(pkg.OPT_LAYER_KERNEL, 1)
    for _ in range(W):
        run.step()
    # advance (untimed) to a block boundary: the timed region then opens with a block's recompute step and holds both step
    # kinds in the workload's own proportion.  Ragged batches (C3, C5) have a request at a boundary in almost every step.
    aligned = 0
    while len(specs) == 1 and not at_block_boundary(run) and aligned < 2 * specs[0].block_len:
        run.step()
        aligned += 1
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    run.h2d = run.d2h = 0
    launches0 = run.eng.launch_count()
    recs, wall, clocks = timed_steps(run, K, local)
    launches = run.eng.launch_count() - launches0
    dev_us = sum(r["us"] for r in recs)
    commits = sum(r["commits"] for r in recs)
    if dist:
        dev_us, wall, commits, launches = reduce_over_ranks(dist, "cuda", dev_us, wall, commits, launches)
    n_req = len(specs)
    value = job_value(world, K, dev_us)
    mix = {"refresh_request_steps": sum(r["n_refresh"] for r in recs), "cached_request_steps": sum(r["n_cached"] for r in recs),
           "refresh": sum(r["kind"] == "refresh" for r in recs), "cached": sum(r["kind"] == "cached" for r in recs),
           "mixed": sum(r["kind"] == "mixed" for r in recs)}
    out = {"metric": "denoise_steps_per_s", "value": value, "unit": "steps/s", "n_gpus": world, "steps": K, "warmup": W,
           "ms_per_step": dev_us / K * 1e-3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
           "data": "synthetic",
           "config": {"workload": f"{args.workload}: {desc}", "requests_per_gpu": n_req, "parallelism": f"replicas x{world}, no collective",
                      "step_mix": mix, "untimed_alignment_steps": aligned, "tau": args.tau,
                      "l2": "every step streams all weights (15 GB >> 126 MB L2): inputs larger than L2, no flush",
                      "timing": "value: sum over steps of CUDA-event time around each step's kernels (library stream); e2e: wall clock of the same calls"},
           "committed_tokens_per_s": commits / (dev_us * 1e-6), "request_steps_per_s": value * n_req,
           "e2e": {"value": world * K / wall, "unit": "steps/s", "h2d_bytes_per_step": run.h2d // K, "d2h_bytes_per_step": run.d2h // K,
                   "committed_tokens_per_s": commits / wall},
           "gpu_launches": int(launches), "clocks": clocks}
    # ---- per step kind: measured vs the step's roofline (north_star: >= 60 %); work summed step by step ----
    steps_rf = {}
    burst = burst_applies(clocks)
    for kind in ("refresh", "cached", "mixed"):
        rs = [r for r in recs if r["kind"] == kind]
        if not rs:
            continue
        steps_rf[kind] = kind_roofline(rs, peaks, burst)
    if "refresh" in steps_rf and "cached" in steps_rf and n_req == 1:
        Bk = specs[0].block_len                    # the block cycle of P:582: one recompute step + B - 1 cache steps
        t_cyc = steps_rf["refresh"]["ms"] + (Bk - 1) * steps_rf["cached"]["ms"]
        r_cyc = steps_rf["refresh"]["roofline_ms"] + (Bk - 1) * steps_rf["cached"]["roofline_ms"]
        steps_rf["block_cycle"] = {"steps": Bk, "ms": t_cyc / Bk, "steps_per_s": 1e3 * Bk / t_cyc, "roofline_ms": r_cyc / Bk, "frac": r_cyc / t_cyc}
    out["step_roofline"] = steps_rf
    out["roofline_frac_all_steps"] = sum(roofline_ms(r["work"], peaks, sustained=not burst)[0] for r in recs) / (sum(r["us"] for r in recs) * 1e-3)
    out["tensor_peak_used"] = "burst" if burst else "sustained"
    out["peaks"] = peaks

    # ---- dominant kernel class, timed inside the production launch by the in-kernel trace ----
    if rank == 0 and not args.no_kernel_pass:
        out["roofline"], out["kernels"] = trace_pass(run, pkg, arch, peaks, burst=burst)
    if rank == 0 and args.trace_rows > 0:
        out["trace_rows"] = trace_rows(run, pkg, args.trace_rows)
    if rank == 0 and args.layer_kernel:
        out["layer_kernel_phases_us"] = layer_kernel_phases(run, pkg, arch)
        out["config"]["layer_kernel"] = True
    if rank == 0 and args.tau_sweep:
        out["tau_sweep"] = tau_sweep(pkg, arch, seed, specs, not args.two_call)
    if rank == 0 and world == 1 and args.workload == "C2" and not args.no_other_workloads:
        run.close()                                  # one model in HBM at a time
        out["other_workloads"] = {}
        for name, k in (("C4", 8), ("C3", 6), ("C5", 6)):
            try:
                out["other_workloads"][name] = other_workload(pkg, name, k, 3, peaks, local)
            except Exception as e:                   # never take the headline down
                out["other_workloads"][name] = {"failed": repr(e)}
    if rank == 0 and not args.no_cpu_baseline and world == 1:
        try:
            out["cpu_baseline"] = cpu_baseline(arch, seed, specs, mix=(mix["refresh_request_steps"], mix["cached_request_steps"]))
        except Exception as e:      # the oracle must never take the GPU line down
            out["cpu_baseline"] = {"value": None, "unit": "steps/s", "cores": os.cpu_count(), "kind": "oracle", "sample": f"failed: {e!r}"}
    run.close()
    if rank == 0:
        print(json.dumps(out), flush=True)
    if dist:
        dist.barrier()
        dist.destroy_process_group()


def tau_sweep(pkg, arch, seed, specs, mixed_launch, taus=(0.5, 0.6, 0.7, 0.8, 0.9, 0.95), steps=12, warm=3):
    """Throughput against the confidence threshold (the paper's knob: P:88-99, candidate set P:123): the same workload
    with every request at threshold tau.  Lower thresholds commit more tokens per step, so requests finish in fewer steps."""
    import copy
    rows = []
    for tau in taus:
        sp = copy.deepcopy(specs)
        for x in sp:
            x.threshold = float(tau)
        run = Runner(pkg, arch, seed, sp, mixed_launch=mixed_launch)
        for _ in range(warm):
            run.step()
        us = cm = 0.0
        for _ in range(steps):
            u, c, _, _, _ = run.step()
            us += u
            cm += c
        run.close()
        rows.append({"tau": tau, "steps_per_s": steps / (us * 1e-6), "committed_tokens_per_s": cm / (us * 1e-6), "commits_per_step": cm / steps})
    return rows


def trace_rows(run, pkg, n):
    """The first n launches of one traced step of the workload's dominant kind: [class, begin_us, wait_us, end_us]."""
    eng = run.eng
    eng.set_option(pkg.OPT_TRACE, 1)
    rows = []
    for _ in range(40):
        us, cm, nr, nc, work = run.step()
        if len(run.specs) == 1 and nr:
            continue
        rows = eng.step_trace()
        if rows:
            break
    eng.set_option(pkg.OPT_TRACE, 0)
    return [[k, round(b, 2), round(w, 2), round(e, 2)] for k, b, w, e in rows[:n]]


def layer_kernel_phases(run, pkg, arch):
    """Mean duration (us) of each of the whole-stack kernel's 7 phases per layer in CTA 0 (first and last layer left out)."""
    eng = run.eng
    eng.set_option(pkg.OPT_LAYER_KERNEL_PHASE_TS, 1)
    ph = None
    for _ in range(40):
        us, cm, nr, nc, work = run.step()
        if not nr and eng.last_step_kernels() & pkg.PATH_LAYER_KERNEL:
            ph = eng.layer_kernel_phases()
    eng.set_option(pkg.OPT_LAYER_KERNEL_PHASE_TS, 0)
    if ph is None or len(ph) < 7 * arch.n_layers + 1:
        return None
    d = np.diff(ph)[: 7 * arch.n_layers].reshape(arch.n_layers, 7)[1:-1]
    names = ("qkv_gemm+rope", "attention", "o_gemm", "fold+norm", "gateup_gemm+swiglu", "down_gemm", "fold+norm(next layer)")
    return {n: round(float(d[:, j].mean()), 2) for j, n in enumerate(names)} | {"layer_total": round(float(d.sum(1).mean()), 2)}


def trace_pass(run, pkg, arch, peaks, n_steps=12, burst=False):
    """A few more steps of the same run with DLM_OPT_TRACE: every kernel stamps %globaltimer inside the production launch
    (CUDA graph + programmatic dependent launch; overhead < 1 %).  A launch holds the step's critical path from the moment
    its griddepcontrol.wait returns (the launch before it has completed) until the next launch's wait returns, so the
    per-class times add up to the step's duration -- which event pairs around overlapping kernels cannot give.  Only steps
    of the workload's dominant kind are kept (cached for one request, mixed / cached for batches)."""
    eng = run.eng
    eng.set_option(pkg.OPT_TRACE, 1)
    kept, cls, work_sum, span = 0, {}, None, 0.0
    guard = 0
    want = None
    while kept < n_steps and guard < 8 * n_steps:
        guard += 1
        us, cm, nr, nc, work = run.step()
        tr = eng.step_trace()
        kind = "mixed" if (nr and nc) else ("refresh" if nr else "cached")
        if len(run.specs) == 1 and kind != "cached":
            continue
        if want is None:
            want = kind
        if kind != want or not tr:
            continue
        kept += 1
        for i, (k, b, w, e) in enumerate(tr):
            nxt = tr[i + 1][2] if i + 1 < len(tr) else e
            a = cls.setdefault(k, [0, 0.0])
            a[0] += 1
            a[1] += max(0.0, nxt - w)
        span += tr[-1][3] - tr[0][2]
        work_sum = work if work_sum is None else {k: work_sum[k] + v for k, v in work.items()}
    eng.set_option(pkg.OPT_TRACE, 0)
    if not kept:
        return None, None
    tot = sum(t for _, t in cls.values())
    kernels = {k: {"launches_per_step": n / kept, "us_per_step": t / kept, "share": t / tot} for k, (n, t) in cls.items()}
    w = {k: v / kept for k, v in work_sum.items()}
    # attention over cached K/V and the combine + unmask pass: achieved HBM rate against the measured peak (north_star (c), (e))
    if "attention" in kernels:
        kernels["attention"].update({"kv_read_gbytes": w["kv_read_bytes"] * 1e-9, "hbm_gbs": w["kv_read_bytes"] / (kernels["attention"]["us_per_step"] * 1e-6) * 1e-9,
                                     "hbm_frac": w["kv_read_bytes"] / (kernels["attention"]["us_per_step"] * 1e-6) * 1e-9 / peaks["hbm_gbs"]})
    if "combine_unmask" in kernels:
        rows = sum(s.block_len for s in run.specs)
        tile = 256 if rows > 128 else 128
        part_bytes = rows * ((arch.vocab + tile - 1) // tile) * 16
        kernels["combine_unmask"].update({"partials_bytes": part_bytes, "hbm_gbs": part_bytes / (kernels["combine_unmask"]["us_per_step"] * 1e-6) * 1e-9})
    gemm = [k for k in kernels if k.startswith("gemm_") or k == "lmhead"]
    g_launch = sum(kernels[k]["launches_per_step"] for k in gemm)
    g_us = sum(kernels[k]["us_per_step"] for k in gemm)
    T = sum(s.block_len for s in run.specs)
    t_b = w["weight_bytes"] / (peaks["hbm_gbs"] * 1e9)
    t_f = w["flops_linear"] / (peaks["bf16_tflops_sustained"] * 1e12)
    if t_b >= t_f:
        # A weight-streaming launch fills its shared-memory rings BEFORE its griddepcontrol.wait returns (weights do not depend on
        # the upstream kernel): gemm_skinny.cuh keeps 2 CTAs x 5 stages x 16 KB of W per SM, i.e. up to 2 x 148 x 80 KB = 23.7 MB per
        # launch move while the previous kernel still holds the critical path.  `achieved` leaves those bytes out of the class's
        # account (they were not moved in the time the class is charged); the figure with them in is an upper bound, kept as
        # achieved_critical_path.  The whole-step number (step_roofline) needs no such correction.
        prefill = min(w["weight_bytes"] / g_launch, 2 * 148 * 5 * 16384) if T <= 128 else 0.0
        ach_cp = w["weight_bytes"] / (g_us * 1e-6) * 1e-9
        ach = (w["weight_bytes"] - g_launch * prefill) / (g_us * 1e-6) * 1e-9
        rf = {"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
              "achieved_critical_path": ach_cp, "frac_critical_path": ach_cp / peaks["hbm_gbs"], "ring_prefill_bytes_per_launch": prefill,
              "algorithmic_bytes_per_launch": w["weight_bytes"] / g_launch}
    else:
        ach = w["flops_linear"] / (g_us * 1e-6) * 1e-12
        pk = peaks["bf16_tflops" if burst else "bf16_tflops_sustained"]
        rf = {"bound": "tensor", "achieved": ach, "peak": pk, "unit": "TFLOP/s", "frac": ach / pk,
              "frac_burst": ach / peaks["bf16_tflops"], "frac_sustained": ach / peaks["bf16_tflops_sustained"],
              "tensor_peak_used": "burst" if burst else "sustained", "algorithmic_flops_per_launch": w["flops_linear"] / g_launch}
    rf.update({"traffic": None, "traffic_note": "dram bytes are not measured by this run; the ncu --set full capture of the same command is under profiles/",
               "kernel": ("gemm_pair_kernel (CTA-pair tcgen05 GEMM: QKV+RoPE, O, gate/up+SwiGLU, down, LM head)" if T > 128 else
                          "gemm_skinny_kernel (QKV, O, gate/up+SwiGLU, down) + gemm_tc_kernel<LM head>: the weight-streaming GEMMs") + f" inside {want} steps",
               "launches_per_step": g_launch, "avg_launch_us": g_us / g_launch, "share_of_step": g_us / (tot / kept),
               "step_us_traced": tot / kept, "timing": "in-kernel %globaltimer stamps under CUDA-graph replay + PDL (DLM_OPT_TRACE); class times sum to the step",
               "algorithmic": f"weights streamed once per step ({w['weight_bytes'] * 1e-9:.2f} GB bf16) over the GEMM launches; tokens per step T={T}",
               "peak_source": peaks["source"], "steps_sampled": kept})
    return rf, kernels


if __name__ == "__main__":
    main()
