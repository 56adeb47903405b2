"""Weight definition W (the paper is silent on weights, BASELINE.json
says "random-init ~N(0,0.02) from seed").  TEST INFRASTRUCTURE ONLY.

value(tensor_id, i), i = row-major flat index over the tensor's [out, in] shape:

    key = mix64(seed + GOLD*(tensor_id+1))                 (all arithmetic mod 2^64)
    h   = mix64(key  + GOLD*(i+1))
    s   = (h & 0xFFFF) + ((h>>16) & 0xFFFF) + ((h>>32) & 0xFFFF) + (h>>48) - 131070
    w   = fp32(s) * c      one fp32 multiply, c = fp32(fp64(fp32(init_std)) / sqrt((2^32-1)/3))
    if weight_dtype == bf16: w = RNE_bf16(w)

mix64 is the splitmix64 finaliser (Steele, Lea, Flood 2014): z ^= z>>30; z *= 0xBF58476D1CE4E5B9;
z ^= z>>27; z *= 0x94D049BB133111EB; z ^= z>>31.   s is a centred Irwin-Hall(4) variate with
variance (2^32-1)/3, so w has standard deviation init_std (to fp32 rounding of c).
RMSNorm gains are 1 and there are no biases (reading G9).
"""
from __future__ import annotations

import concurrent.futures as _cf
import os

import numpy as np

GOLD = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)

TID_EMBED = 0
TID_LMHEAD = 1
SUB_Q, SUB_K, SUB_V, SUB_O, SUB_G, SUB_U, SUB_D = range(7)


def layer_tid(layer: int, sub: int) -> int:
    return 16 * (layer + 1) + sub


def mix64(z: np.ndarray) -> np.ndarray:
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def scale_constant(init_std: float) -> np.float32:
    return np.float32(np.float64(np.float32(init_std)) / np.sqrt(np.float64(4294967295.0) / np.float64(3.0)))


def round_to_bf16(w32: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even float32 -> bfloat16, returned as float32 holding the bf16 value."""
    u = np.ascontiguousarray(w32, dtype=np.float32).view(np.uint32)
    lsb = (u >> np.uint32(16)) & np.uint32(1)
    r = (u + np.uint32(0x7FFF) + lsb) & np.uint32(0xFFFF0000)
    return r.view(np.float32)


def _chunk(seed: int, tid: int, lo: int, hi: int, c: np.float32, to_bf16: bool) -> np.ndarray:
    with np.errstate(over="ignore"):
        key = mix64(np.uint64(seed) + GOLD * np.uint64(tid + 1))
        i = np.arange(lo + 1, hi + 1, dtype=np.uint64)
        h = mix64(key + GOLD * i)
    m = np.uint64(0xFFFF)
    s = ((h & m) + ((h >> np.uint64(16)) & m) + ((h >> np.uint64(32)) & m) + (h >> np.uint64(48))).astype(np.int64)
    s -= 131070
    w = s.astype(np.float32) * c
    return round_to_bf16(w) if to_bf16 else w


def tensor_f32(seed: int, tid: int, shape, init_std: float, to_bf16: bool, threads: int | None = None) -> np.ndarray:
    """The whole tensor as float32 (exact: a bf16 value is representable in float32)."""
    n = int(np.prod(shape))
    c = scale_constant(init_std)
    step = 1 << 22
    bounds = [(lo, min(lo + step, n)) for lo in range(0, n, step)]
    out = np.empty(n, dtype=np.float32)
    threads = threads or min(8, os.cpu_count() or 1)

    def work(b):
        out[b[0]:b[1]] = _chunk(seed, tid, b[0], b[1], c, to_bf16)

    if len(bounds) > 1 and threads > 1:
        with _cf.ThreadPoolExecutor(threads) as ex:
            list(ex.map(work, bounds))
    else:
        for b in bounds:
            work(b)
    return out.reshape(shape)


class Weights:
    """All tensors of one model, generated on demand and kept as float32 (exact values);
    `get` returns float64 copies so the forward pass runs in fp64."""

    def __init__(self, arch, seed: int, cache_bytes: int = 24 << 30, keep_f64: bool = False):
        self.arch, self.seed = arch, int(seed)
        self._cache: dict = {}
        self._bytes = 0
        self._cap = cache_bytes
        self._f64: dict | None = {} if keep_f64 else None      # memo of the float64 copies (many requests through one small model)

    def shape(self, tid: int):
        a = self.arch
        if tid in (TID_EMBED, TID_LMHEAD):
            return (a.vocab, a.d_model)
        sub = tid % 16
        hq, hkv = a.n_heads * a.head_dim, a.n_kv_heads * a.head_dim
        return {SUB_Q: (hq, a.d_model), SUB_K: (hkv, a.d_model), SUB_V: (hkv, a.d_model),
                SUB_O: (a.d_model, hq), SUB_G: (a.d_ffn, a.d_model), SUB_U: (a.d_ffn, a.d_model),
                SUB_D: (a.d_model, a.d_ffn)}[sub]

    def f32(self, tid: int) -> np.ndarray:
        w = self._cache.get(tid)
        if w is None:
            w = tensor_f32(self.seed, tid, self.shape(tid), self.arch.init_std, self.arch.weight_dtype == 1)
            if self._bytes + w.nbytes <= self._cap:
                self._cache[tid] = w
                self._bytes += w.nbytes
        return w

    def get(self, tid: int) -> np.ndarray:
        if self._f64 is None:
            return self.f32(tid).astype(np.float64)
        w = self._f64.get(tid)
        if w is None:
            w = self._f64[tid] = self.f32(tid).astype(np.float64)
        return w

    def rows(self, tid: int, idx: np.ndarray) -> np.ndarray:
        """Selected rows (embedding gather) without materialising the whole tensor when uncached."""
        if tid in self._cache:
            return self._cache[tid][idx].astype(np.float64)
        shape = self.shape(tid)
        c = scale_constant(self.arch.init_std)
        out = np.empty((len(idx), shape[1]), dtype=np.float64)
        for j, r in enumerate(np.asarray(idx).tolist()):
            out[j] = _chunk(self.seed, tid, r * shape[1], (r + 1) * shape[1], c, self.arch.weight_dtype == 1)
        return out

    def drop(self, tid: int):
        w = self._cache.pop(tid, None)
        if w is not None:
            self._bytes -= w.nbytes
