"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NO arithmetic of the method (no hashing of weights, no forward pass,
no softmax, no unmask rule): only the architecture tables of BASELINE.json's five configs
and the seeded draws of prompt lengths / token ids / thresholds / block phases that both
the CPU oracle (oracle/) and the CUDA path (paper_2606_29094_b200/) are fed.

The shapes stand in for the paper's workloads, which are not in this container
(Tables 3-4: prompt lengths 261/737/1020, output 256, block 32;
PAPER.md:392: block size 32, default threshold 0.9; candidate thresholds).
Token ids are uniform over [0, V) minus {mask_id}; mask_id = V-1 (synthetic choice).
"""
from __future__ import annotations

import dataclasses
from typing import List

import numpy as np


@dataclasses.dataclass(frozen=True)
class Arch:
    """Plain description of a model shape (mirrors include/dlm.h `dlm_arch`)."""
    n_layers: int
    d_model: int
    n_heads: int
    n_kv_heads: int
    head_dim: int
    d_ffn: int
    vocab: int
    mask_id: int
    weight_dtype: int          # 0 = fp32 weights (config 1), 1 = bf16 weights
    logit_scale: float
    rms_eps: float = 1e-5
    rope_theta: float = 10000.0
    init_std: float = 0.02

    def replace(self, **kw) -> "Arch":
        return dataclasses.replace(self, **kw)


# BASELINE.json configs[0..4]; rope_theta / eps / logit scale of C5: DESIGN.md readings G10, G12.
ARCH_C1 = Arch(2, 256, 4, 4, 64, 688, 4096, 4095, 0, 8.0, 1e-5, 10000.0, 0.02)
ARCH_LLADA8B = Arch(32, 4096, 32, 32, 128, 12288, 126464, 126463, 1, 4.0, 1e-5, 500000.0, 0.02)
ARCH_QWEN7B = Arch(28, 3584, 28, 4, 128, 18944, 152064, 152063, 1, 4.0, 1e-5, 1000000.0, 0.02)

WEIGHT_SEED = {"C1": 1001, "C2": 1002, "C3": 1003, "C4": 1004, "C5": 1005}


@dataclasses.dataclass
class RequestSpec:
    prompt: np.ndarray          # int32 [P]
    gen_len: int
    block_len: int
    threshold: float
    # constructed progress (configs 3 and 5): the request has finished `block_index` blocks and
    # has `phase` positions of its current block already committed (filled with `filled` ids).
    block_index: int = 0
    phase: int = 0
    filled: np.ndarray | None = None   # int32 [block_index*block_len + phase] ids already committed
    filled_pos: np.ndarray | None = None  # generation-relative positions of `filled`


def random_tokens(rng: np.random.Generator, n: int, vocab: int, mask_id: int) -> np.ndarray:
    """Uniform ids over [0, vocab) \\ {mask_id}."""
    t = rng.integers(0, vocab - 1, size=n, dtype=np.int64)
    t = np.where(t >= mask_id, t + 1, t)
    return t.astype(np.int32)


def workload_c1() -> List[RequestSpec]:
    rng = np.random.default_rng(2001)
    a = ARCH_C1
    return [RequestSpec(random_tokens(rng, 64, a.vocab, a.mask_id), 64, 32, 0.9)]


def workload_c2() -> List[RequestSpec]:
    rng = np.random.default_rng(2002)
    a = ARCH_LLADA8B
    return [RequestSpec(random_tokens(rng, 256, a.vocab, a.mask_id), 256, 32, 0.9)]


def _constructed(rng, arch, plen, gen, blk, tau, block_index, phase) -> RequestSpec:
    n_filled = block_index * blk + phase
    filled = random_tokens(rng, n_filled, arch.vocab, arch.mask_id)
    # finished blocks are fully committed; inside the current block the `phase` committed
    # positions are a seeded random subset (commits do not happen left to right)
    cur = rng.permutation(blk)[:phase] + block_index * blk
    pos = np.concatenate([np.arange(block_index * blk), np.sort(cur)]).astype(np.int32)
    return RequestSpec(random_tokens(rng, plen, arch.vocab, arch.mask_id), gen, blk, tau,
                       block_index, phase, filled, pos)


def workload_c3(n: int = 32) -> List[RequestSpec]:
    """Ragged batch, mixed block phases: request i is phi_i = (7i+3) mod 32 commits into block i mod 8,
    so exactly one request (i = 23 for n = 32) sits at phi = 0 and is due a refresh step."""
    rng = np.random.default_rng(2003)
    a = ARCH_LLADA8B
    plens = rng.integers(128, 1025, size=n)
    taus = np.array([0.5, 0.7, 0.9, 0.95] * ((n + 3) // 4))[:n]
    rng.shuffle(taus)
    return [_constructed(rng, a, int(plens[i]), 256, 32, float(taus[i]), i % 8, (7 * i + 3) % 32)
            for i in range(n)]


def workload_c4(n: int = 8, prompt_len: int = 4096, gen: int = 512, blk: int = 64) -> List[RequestSpec]:
    rng = np.random.default_rng(2004)
    a = ARCH_LLADA8B
    return [RequestSpec(random_tokens(rng, prompt_len, a.vocab, a.mask_id), gen, blk, 0.9) for _ in range(n)]


def workload_c5(n: int = 64, tau: float = 0.9) -> List[RequestSpec]:
    rng = np.random.default_rng(2005)
    a = ARCH_QWEN7B
    plens = rng.integers(256, 2049, size=n)
    return [_constructed(rng, a, int(plens[i]), 256, 32, tau, i % 8, (7 * i + 3) % 32) for i in range(n)]


def initial_tokens(spec: RequestSpec, mask_id: int) -> np.ndarray:
    """prompt || generation, generation all [MASK] except the constructed `filled` positions."""
    g = np.full(spec.gen_len, mask_id, dtype=np.int32)
    if spec.filled is not None and len(spec.filled):
        g[spec.filled_pos] = spec.filled
    return np.concatenate([spec.prompt.astype(np.int32), g])


def unit_rms_hidden(seed: int, rows: int, d: int) -> np.ndarray:
    """Random hidden states with unit RMS per row (config 5 LM-head micro-bench input), float32."""
    rng = np.random.default_rng(seed)
    h = rng.standard_normal((rows, d)).astype(np.float32)
    h /= np.sqrt((h.astype(np.float64) ** 2).mean(-1, keepdims=True)).astype(np.float32)
    return h
