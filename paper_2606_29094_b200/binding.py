"""ctypes binding of libdlm.so (include/dlm.h, include/dlm_ops.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; this module never computes.  PyTorch is
used for device memory (the `dlm_mem` provider hands out torch-owned buffers) and for the stream.
The library must be built (``python -c "import __graft_entry__ as g; g.build()"``); importing fails loudly
when it is missing, and every compute call fails with DLM_E_CUDA when there is no CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdlm.so")

DLM_OK, DLM_E_ARG, DLM_E_CAPACITY, DLM_E_STATE, DLM_E_CUDA = 0, -1, -2, -3, -4
DLM_DRY_RUN = 1
OPT_SIMPLE_KERNELS, OPT_DEBUG_DUMP, OPT_CUDA_GRAPH, OPT_FLASH_ATTENTION, OPT_KERNEL_TIMING, OPT_PDL, OPT_SKINNY_GEMM, OPT_PAIR_GEMM, OPT_TC_ATTENTION, OPT_FUSE_ROPE = 1, 2, 3, 4, 5, 6, 7, 8, 9, 10
OPT_TRACE, OPT_TCT_MIN_ITEMS, OPT_LAYER_KERNEL, OPT_LAYER_KERNEL_PHASE_TS = 11, 12, 13, 14
DTYPE_F32, DTYPE_BF16, DTYPE_BF16_PRECISE = 0, 1, 2
PATH_GEMM_SKINNY, PATH_GEMM_PAIR, PATH_GEMM_TC, PATH_GEMM_PLAIN, PATH_ATTN_TC, PATH_ATTN_TCT, PATH_ATTN_FLASH, PATH_ATTN_PLAIN, PATH_ROPE_FUSED, PATH_GRAPH_REPLAY, PATH_LAYER_KERNEL = (1 << i for i in range(11))
KERNEL_NAMES = ("embed", "rmsnorm", "gemm_qkv", "rope_kv", "attention", "gemm_o", "gemm_gateup", "gemm_down", "lmhead",
                "combine_unmask", "layers")
KIND_REFRESH, KIND_CACHED, KIND_MIXED = 0, 1, 2
N_FEATURES = 11
FEATURE_NAMES = ("confidence_threshold", "output_length", "full_progress", "full_unmask_progress", "block_progress", "block_unmask_progress",
                 "output_min_confidence", "output_q25_confidence", "output_median_confidence", "output_avg_confidence", "output_q75_confidence")
T_X_IN, T_NORM1, T_Q, T_K, T_V, T_ATTN, T_X_MID, T_NORM2, T_ACT, T_X_OUT, T_FINAL_NORM, T_KCACHE, T_VCACHE = range(13)
EPI_F32, EPI_BF16, EPI_RESID, EPI_SWIGLU = 0, 1, 2, 3


class DlmError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libdlm error {code}: {msg}")
        self.code = code


class _Arch(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_layers", "d_model", "n_heads", "n_kv_heads", "head_dim", "d_ffn", "vocab",
                                         "mask_id", "weight_dtype")] + \
               [(n, C.c_float) for n in ("logit_scale", "rms_eps", "rope_theta", "init_std")] + \
               [(n, C.c_int32) for n in ("max_requests", "max_seq", "max_block", "kv_page_tokens", "max_batch_tokens")] + \
               [("kv_pool_tokens", C.c_int64)]


_ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
_FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class _Mem(C.Structure):
    _fields_ = [("alloc", _ALLOC_FN), ("free", _FREE_FN), ("user", C.c_void_p), ("cuda_stream", C.c_void_p)]


class _Batch(C.Structure):
    _fields_ = [("n", C.c_int32), ("req", C.POINTER(C.c_int32)), ("threshold", C.POINTER(C.c_float)), ("flags", C.c_uint32)]


class _Result(C.Structure):
    _fields_ = [("n_committed", C.POINTER(C.c_int32)), ("pos", C.POINTER(C.c_int32)), ("tok", C.POINTER(C.c_int32)),
                ("conf", C.POINTER(C.c_float)), ("capacity", C.c_int32), ("total", C.c_int32),
                ("n_masked_left", C.POINTER(C.c_int32)), ("lse", C.POINTER(C.c_float)),
                ("row_conf", C.POINTER(C.c_float)), ("row_tok", C.POINTER(C.c_int32)), ("features", C.POINTER(C.c_float))]


class _CostRow(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n_requests", C.c_int32), ("n_tokens", C.c_int32), ("kv_tokens", C.c_int32),
                ("usec", C.c_float)]


class _KernelTime(C.Structure):
    _fields_ = [("kernel", C.c_int32), ("launches", C.c_int32), ("usec", C.c_float)]


class _TraceRow(C.Structure):
    _fields_ = [("kernel", C.c_int32), ("slot", C.c_int32), ("begin_us", C.c_float), ("wait_us", C.c_float), ("end_us", C.c_float)]


_lib = None


def lib() -> C.CDLL:
    """Load libdlm.so once; no fallback of any kind."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with __graft_entry__.build() "
                              "(nvcc -gencode arch=compute_100a,code=sm_100a); there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, f32 = C.c_void_p, C.c_int32, C.c_int64, C.c_float
        L.dlm_init.argtypes = [C.POINTER(_Arch), C.c_uint64, C.POINTER(vp)]
        L.dlm_init_ex.argtypes = [C.POINTER(_Arch), C.c_uint64, C.POINTER(_Mem), C.POINTER(vp)]
        L.dlm_destroy.argtypes = [vp]
        L.dlm_destroy.restype = None
        L.dlm_request_add.argtypes = [vp, C.POINTER(i32), i32, i32, i32, f32, C.POINTER(i32)]
        L.dlm_request_set_tokens.argtypes = [vp, i32, C.POINTER(i32), i32, i32]
        L.dlm_request_remove.argtypes = [vp, i32]
        L.dlm_request_tokens.argtypes = [vp, i32, C.POINTER(i32), i32]
        L.dlm_request_info.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32)]
        L.dlm_request_export.argtypes = [vp, i32, vp, i64]
        L.dlm_request_export.restype = i64
        L.dlm_request_import.argtypes = [vp, vp, i64, C.POINTER(i32)]
        L.dlm_refresh_step.argtypes = [vp, C.POINTER(_Batch), C.POINTER(_Result)]
        L.dlm_cached_step.argtypes = [vp, C.POINTER(_Batch), C.POINTER(f32), C.POINTER(_Result)]
        L.dlm_mixed_step.argtypes = [vp, C.POINTER(_Batch), C.POINTER(f32), C.POINTER(_Result)]
        L.dlm_profile_step_costs.argtypes = [vp, C.POINTER(_CostRow), i32, C.POINTER(i32)]
        L.dlm_profile_step_costs_ex.argtypes = [vp, i32, i32, C.POINTER(_CostRow), i32, C.POINTER(i32)]
        L.dlm_last_step_kernels.argtypes = [vp]
        L.dlm_last_step_kernels.restype = C.c_uint32
        L.dlm_step_trace.argtypes = [vp, C.POINTER(_TraceRow), i32, C.POINTER(i32)]
        L.dlm_layer_kernel_phases.argtypes = [vp, C.POINTER(f32), i32]
        L.dlm_set_option.argtypes = [vp, i32, i32]
        L.dlm_kernel_times.argtypes = [vp, C.POINTER(_KernelTime), i32, C.POINTER(i32), i32]
        L.dlm_debug_tensor.argtypes = [vp, i32, i32, i32, C.POINTER(f32), i64]
        L.dlm_debug_tensor.restype = i64
        L.dlm_launch_count.argtypes = [vp]
        L.dlm_launch_count.restype = i64
        L.dlm_last_step_usec.argtypes = [vp]
        L.dlm_last_step_usec.restype = f32
        L.dlm_last_error.argtypes = [vp]
        L.dlm_last_error.restype = C.c_char_p
        f64 = C.c_double
        L.dlm_lp_lookup.argtypes = [C.POINTER(_CostRow), i32, i32, f64, i32]
        L.dlm_lp_lookup.restype = f64
        L.dlm_req_load.argtypes = [f64, i32, i32, i32]
        L.dlm_req_load.restype = f64
        L.dlm_instance_capacity.argtypes = [C.POINTER(_CostRow), i32, i32, i32, i32, i32, f64]
        L.dlm_instance_capacity.restype = f64
        L.dlm_time_left.argtypes = [C.POINTER(_CostRow), i32, f64, i32, i32, i32, i32, i32]
        L.dlm_time_left.restype = f64
        L.dlm_pick_threshold.argtypes = [C.POINTER(f32), C.POINTER(f64), i32, f64, C.POINTER(_CostRow), i32, i32, i32, i32, i32, i32]
        L.dlm_op_gemm_bf16.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, vp]
        L.dlm_op_gemm_pair_bf16.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, i32, vp]
        L.dlm_op_gemm_plain_bf16.argtypes = [vp, vp, vp, i32, i32, i32, vp]
        L.dlm_op_gemm_pair_plan.argtypes = [i32, i32, i32, i32, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32)]
        L.dlm_op_gemm_skinny_bf16.argtypes = [vp, vp, vp, i32, i32, i32, i32, i32, vp]
        L.dlm_op_lmhead_scratch_bytes.argtypes = [i32, i32]
        L.dlm_op_lmhead_scratch_bytes.restype = i64
        L.dlm_op_lmhead_bf16.argtypes = [vp, vp, i32, i32, i32, f32, i32, vp, vp, vp, vp, vp]
        L.dlm_op_lmhead_unmask_bf16.argtypes = [vp, vp, i32, i32, i32, i32, f32, i32, vp, vp, vp, vp, vp, vp, vp, vp]
        L.dlm_op_lmhead_static_bytes.argtypes = [i32, i32]
        L.dlm_op_lmhead_static_bytes.restype = i64
        L.dlm_op_lmhead_static_bf16.argtypes = [vp, vp, i32, i32, i32, f32, i32, vp, vp, vp, vp]
        L.dlm_op_attention_bf16.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, vp]
        _lib = L
    return _lib


def exported_symbols() -> List[str]:
    """Names declared DLM_API in include/*.h (parsed from the headers, used by the symbol test)."""
    import re
    out = []
    inc = os.path.join(os.path.dirname(_HERE), "include")
    for f in sorted(os.listdir(inc)):
        if f.endswith(".h"):
            out += re.findall(r"DLM_API[^;(]*?\b(dlm_\w+)\s*\(", open(os.path.join(inc, f)).read())
    return out


def _ip(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _fp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_float))


class StepResult:
    """Host copy of a dlm_result: per-request commit lists plus the per-row statistics."""

    def __init__(self, n, max_block, n_committed, pos, tok, conf, n_masked_left, lse, row_conf, row_tok, usec, features=None):
        self.n_committed = n_committed
        self.features = features          # [n, 11] Step Predictor features (FEATURE_NAMES) when requested
        self.n_masked_left = n_masked_left
        self.lse, self.row_conf, self.row_tok = lse.reshape(n, max_block), row_conf.reshape(n, max_block), row_tok.reshape(n, max_block)
        self.usec = usec
        self.commits = []
        o = 0
        for i in range(n):
            k = int(n_committed[i])
            self.commits.append([(int(pos[o + j]), int(tok[o + j]), float(conf[o + j])) for j in range(k)])
            o += k
        self.total = o


class Engine:
    """A model instance (the paper's L1 executor): dlm_init + request table + the two step calls."""

    def __init__(self, arch, seed: int, max_requests: int = 1, max_seq: int = 512, max_block: int = 32,
                 kv_page_tokens: int = 64, max_batch_tokens: Optional[int] = None, kv_pool_tokens: int = 0,
                 use_torch_memory: bool = True):
        import torch
        self._torch = torch
        self.arch = arch
        self.max_block, self.max_requests, self.max_seq = max_block, max_requests, max_seq
        a = _Arch(arch.n_layers, arch.d_model, arch.n_heads, arch.n_kv_heads, arch.head_dim, arch.d_ffn, arch.vocab,
                  arch.mask_id, arch.weight_dtype, arch.logit_scale, arch.rms_eps, arch.rope_theta, arch.init_std,
                  max_requests, max_seq, max_block, kv_page_tokens,
                  max_batch_tokens if max_batch_tokens else max_requests * max_seq, kv_pool_tokens)
        self._bufs = {}
        L = lib()
        self._h = C.c_void_p()
        if use_torch_memory and torch.cuda.is_available():
            def _alloc(nbytes, _user):
                try:
                    t = torch.empty(int(nbytes), dtype=torch.uint8, device="cuda")
                except Exception:       # out of memory -> NULL -> DLM_E_CAPACITY
                    return None
                self._bufs[t.data_ptr()] = t
                return t.data_ptr()

            def _free(ptr, _user):
                self._bufs.pop(ptr, None)

            self._alloc_cb, self._free_cb = _ALLOC_FN(_alloc), _FREE_FN(_free)
            self.stream = torch.cuda.current_stream()
            mem = _Mem(self._alloc_cb, self._free_cb, None, self.stream.cuda_stream)
            rc = L.dlm_init_ex(C.byref(a), seed, C.byref(mem), C.byref(self._h))
        else:
            rc = L.dlm_init(C.byref(a), seed, C.byref(self._h))
        if rc:
            raise DlmError(rc, L.dlm_last_error(None).decode())
        R = max_requests * max_block
        self._nc = np.zeros(max_requests, np.int32)
        self._pos, self._tok = np.zeros(R, np.int32), np.zeros(R, np.int32)
        self._conf = np.zeros(R, np.float32)
        self._left = np.zeros(max_requests, np.int32)
        self._lse, self._rconf = np.zeros(R, np.float32), np.zeros(R, np.float32)
        self._rtok = np.zeros(R, np.int32)
        self._feat = np.zeros(max_requests * N_FEATURES, np.float32)

    # -- lifetime --
    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().dlm_destroy(self._h)
            self._h = C.c_void_p()
            self._bufs.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc < 0:
            raise DlmError(rc, lib().dlm_last_error(self._h).decode())
        return rc

    # -- requests --
    def add_request(self, prompt: Sequence[int], gen_len: int, block_len: int, threshold: float) -> int:
        p = np.ascontiguousarray(prompt, dtype=np.int32)
        out = C.c_int32(-1)
        self._check(lib().dlm_request_add(self._h, _ip(p), len(p), gen_len, block_len, threshold, C.byref(out)))
        return out.value

    def set_tokens(self, req: int, tokens: Sequence[int], keep_cache: bool = False):
        t = np.ascontiguousarray(tokens, dtype=np.int32)
        self._check(lib().dlm_request_set_tokens(self._h, req, _ip(t), len(t), 1 if keep_cache else 0))

    def remove_request(self, req: int):
        self._check(lib().dlm_request_remove(self._h, req))

    def tokens(self, req: int) -> np.ndarray:
        buf = np.zeros(self.max_seq, np.int32)
        n = self._check(lib().dlm_request_tokens(self._h, req, _ip(buf), len(buf)))
        return buf[:n].copy()

    def info(self, req: int):
        a, b, c = C.c_int32(), C.c_int32(), C.c_int32()
        self._check(lib().dlm_request_info(self._h, req, C.byref(a), C.byref(b), C.byref(c)))
        return {"cur_block": a.value, "cache_valid": bool(b.value), "n_masked": c.value}

    def export_request(self, req: int) -> bytes:
        """The request without its K/V cache, as the host blob include/dlm.h describes (migration)."""
        need = self._check(lib().dlm_request_export(self._h, req, None, 0))
        buf = C.create_string_buffer(need)
        self._check(lib().dlm_request_export(self._h, req, buf, need))
        return buf.raw

    def import_request(self, blob: bytes) -> int:
        out = C.c_int32(-1)
        buf = C.create_string_buffer(blob, len(blob))
        self._check(lib().dlm_request_import(self._h, buf, len(blob), C.byref(out)))
        return out.value

    # -- steps --
    def _step(self, kind: int, reqs: Sequence[int], thresholds, dry_run: bool, features: bool = False) -> StepResult:
        n = len(reqs)
        r = np.ascontiguousarray(reqs, dtype=np.int32)
        thr = None if thresholds is None else np.ascontiguousarray(thresholds, dtype=np.float32)
        b = _Batch(n, _ip(r), _fp(thr) if thr is not None else None, DLM_DRY_RUN if dry_run else 0)
        res = _Result(_ip(self._nc), _ip(self._pos), _ip(self._tok), _fp(self._conf), len(self._pos), 0, _ip(self._left),
                      _fp(self._lse), _fp(self._rconf), _ip(self._rtok), _fp(self._feat) if features else None)
        L = lib()
        if kind == KIND_REFRESH:
            rc = L.dlm_refresh_step(self._h, C.byref(b), C.byref(res))
        elif kind == KIND_MIXED:
            rc = L.dlm_mixed_step(self._h, C.byref(b), None, C.byref(res))
        else:
            rc = L.dlm_cached_step(self._h, C.byref(b), None, C.byref(res))
        self._check(rc)
        mb = self.max_block
        return StepResult(n, mb, self._nc[:n].copy(), self._pos, self._tok, self._conf, self._left[:n].copy(),
                          self._lse[:n * mb].copy(), self._rconf[:n * mb].copy(), self._rtok[:n * mb].copy(),
                          L.dlm_last_step_usec(self._h), self._feat[:n * N_FEATURES].reshape(n, N_FEATURES).copy() if features else None)

    def refresh_step(self, reqs, thresholds=None, dry_run=False, features=False) -> StepResult:
        return self._step(KIND_REFRESH, reqs, thresholds, dry_run, features)

    def cached_step(self, reqs, thresholds=None, dry_run=False, features=False) -> StepResult:
        return self._step(KIND_CACHED, reqs, thresholds, dry_run, features)

    def mixed_step(self, reqs, thresholds=None, dry_run=False, features=False) -> StepResult:
        """One ragged launch: every request takes the step kind that is due (refresh if its cache is invalid)."""
        return self._step(KIND_MIXED, reqs, thresholds, dry_run, features)

    # -- misc --
    def set_option(self, key: int, value: int):
        self._check(lib().dlm_set_option(self._h, key, value))

    def launch_count(self) -> int:
        return int(lib().dlm_launch_count(self._h))

    def last_step_usec(self) -> float:
        return float(lib().dlm_last_step_usec(self._h))

    def debug_tensor(self, req: int, layer: int, which: int, rows: int, width: int) -> np.ndarray:
        out = np.zeros(rows * width, np.float32)
        n = self._check(lib().dlm_debug_tensor(self._h, req, layer, which, _fp(out), out.size))
        return out[:n].reshape(-1, width)

    def kernel_times(self, reset: bool = True):
        """{kernel class: (launches, total usec)} accumulated while OPT_KERNEL_TIMING was on."""
        rows = (_KernelTime * 32)()
        n = C.c_int32(0)
        self._check(lib().dlm_kernel_times(self._h, rows, 32, C.byref(n), 1 if reset else 0))
        return {KERNEL_NAMES[rows[i].kernel]: (rows[i].launches, rows[i].usec) for i in range(n.value)}

    def layer_kernel_phases(self) -> np.ndarray:
        """Phase end times (us) of the last whole-stack launch taken with OPT_LAYER_KERNEL_PHASE_TS."""
        buf = np.zeros(7 * self.arch.n_layers + 1, np.float32)
        n = self._check(lib().dlm_layer_kernel_phases(self._h, _fp(buf), len(buf)))
        return buf[:n].copy()

    def last_step_kernels(self) -> int:
        """PATH_* bit set of the kernel families the last step launched."""
        return int(lib().dlm_last_step_kernels(self._h))

    def step_trace(self):
        """Timeline of the last step taken with OPT_TRACE: [(kernel class name, begin_us, wait_us, end_us)] in launch order."""
        rows = (_TraceRow * 2048)()
        n = C.c_int32(0)
        self._check(lib().dlm_step_trace(self._h, rows, 2048, C.byref(n)))
        return [(KERNEL_NAMES[rows[i].kernel], rows[i].begin_us, rows[i].wait_us, rows[i].end_us) for i in range(n.value)]

    def profile_step_costs(self, cap: int = 128, block_len: Optional[int] = None, repeats: int = 10):
        rows = (_CostRow * cap)()
        n = C.c_int32(0)
        if block_len is None:
            self._check(lib().dlm_profile_step_costs(self._h, rows, cap, C.byref(n)))
        else:
            self._check(lib().dlm_profile_step_costs_ex(self._h, block_len, repeats, rows, cap, C.byref(n)))
        return [dict(kind="refresh" if rows[i].kind == KIND_REFRESH else "cached", n_requests=rows[i].n_requests,
                     n_tokens=rows[i].n_tokens, kv_tokens=rows[i].kv_tokens, usec=rows[i].usec) for i in range(n.value)]


# ---------------------------------------------------------------------------------------------------------
# host-side consumers of the cost table (include/dlm_sched.h; rows = [(kind, tokens, kv, usec)] or profile_step_costs dicts)
# ---------------------------------------------------------------------------------------------------------
def _cost_rows(rows):
    arr = (_CostRow * len(rows))()
    for i, r in enumerate(rows):
        if isinstance(r, dict):
            kind, n, tokens, kv, usec = r["kind"], r.get("n_requests", 0), r["n_tokens"], r["kv_tokens"], r["usec"]
        else:
            kind, tokens, kv, usec = r
            n = 0
        arr[i] = _CostRow(KIND_REFRESH if kind in ("refresh", KIND_REFRESH) else KIND_CACHED, n, int(tokens), int(kv), float(usec))
    return arr, len(rows)


def lp_lookup(rows, kind, tokens, kv):
    a, n = _cost_rows(rows)
    return lib().dlm_lp_lookup(a, n, KIND_REFRESH if kind in ("refresh", KIND_REFRESH) else KIND_CACHED, float(tokens), int(kv))


def req_load(pred_steps_left, recomp_steps_left, num_tokens, cache_block):
    return lib().dlm_req_load(float(pred_steps_left), recomp_steps_left, num_tokens, cache_block)


def instance_capacity(rows, cache_block, max_seq_per_batch, num_token_per_req, kv, slo_sec):
    a, n = _cost_rows(rows)
    return lib().dlm_instance_capacity(a, n, cache_block, max_seq_per_batch, num_token_per_req, kv, float(slo_sec))


def time_left(rows, pred_steps_left, recomp_steps_left, cache_block, num_reqs, num_tokens, kv):
    a, n = _cost_rows(rows)
    return lib().dlm_time_left(a, n, float(pred_steps_left), recomp_steps_left, cache_block, num_reqs, num_tokens, kv)


def pick_threshold(allowed_desc, pred_steps_left, slo_left_sec, rows, recomp_steps_left, cache_block, num_reqs, num_tokens, kv):
    a, n = _cost_rows(rows)
    th = (C.c_float * len(allowed_desc))(*allowed_desc)
    st = (C.c_double * len(pred_steps_left))(*pred_steps_left)
    rc = lib().dlm_pick_threshold(th, st, len(allowed_desc), float(slo_left_sec), a, n, recomp_steps_left, cache_block, num_reqs, num_tokens, kv)
    if rc < 0:
        raise DlmError(rc, "dlm_pick_threshold: bad arguments")
    return rc


# ---------------------------------------------------------------------------------------------------------
# kernel-level ops (device tensors in, device tensors out; torch only owns the memory)
# ---------------------------------------------------------------------------------------------------------
def _stream_ptr():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _op_check(rc):
    if rc < 0:
        raise DlmError(rc, lib().dlm_last_error(None).decode())


def op_gemm_bf16(A, W, epilogue: int = EPI_F32, bn: int = 0, out=None):
    import torch
    M, K = A.shape
    N = W.shape[0] // 2 if epilogue == EPI_SWIGLU else W.shape[0]
    if out is None:
        out = torch.empty(M, N, device=A.device, dtype=torch.float32 if epilogue in (EPI_F32, EPI_RESID) else torch.bfloat16)
    _op_check(lib().dlm_op_gemm_bf16(A.data_ptr(), W.data_ptr(), out.data_ptr(), M, N, K, epilogue, bn, _stream_ptr()))
    return out


def op_gemm_pair_bf16(A, W, epilogue: int = EPI_F32, bn: int = 0, out=None, splits: int = 1, return_splits: bool = False):
    """Persistent CTA-pair tcgen05 GEMM (the engine's M > 128 path); splits: see include/dlm_ops.h."""
    import torch
    M, K = A.shape
    N = W.shape[0] // 2 if epilogue == EPI_SWIGLU else W.shape[0]
    if out is None:
        out = torch.empty(M, N, device=A.device, dtype=torch.float32 if epilogue in (EPI_F32, EPI_RESID) else torch.bfloat16)
    rc = lib().dlm_op_gemm_pair_bf16(A.data_ptr(), W.data_ptr(), out.data_ptr(), M, N, K, epilogue, bn, splits, _stream_ptr())
    _op_check(rc)
    return (out, rc) if return_splits else out


def op_gemm_pair_plan(M: int, N: int, K: int, epilogue: int):
    """(bn, bn2, n_wide) of the automatic tile plan (bn2 = 0: one width)."""
    a, b, c = C.c_int32(), C.c_int32(), C.c_int32()
    _op_check(lib().dlm_op_gemm_pair_plan(M, N, K, epilogue, C.byref(a), C.byref(b), C.byref(c)))
    return a.value, b.value, c.value


def op_gemm_skinny_bf16(X, W, epilogue: int = EPI_F32, splits: int = 0):
    """Returns (out, K splits used)."""
    import torch
    T, K = X.shape
    N = W.shape[0] // 2 if epilogue == EPI_SWIGLU else W.shape[0]
    out = torch.empty(T, N, device=X.device, dtype=torch.float32 if epilogue == EPI_F32 else torch.bfloat16)
    rc = lib().dlm_op_gemm_skinny_bf16(X.data_ptr(), W.data_ptr(), out.data_ptr(), T, N, K, epilogue, splits, _stream_ptr())
    _op_check(rc)
    return out, rc


def op_gemm_plain_bf16(A, W):
    import torch
    M, K = A.shape
    out = torch.empty(M, W.shape[0], device=A.device, dtype=torch.float32)
    _op_check(lib().dlm_op_gemm_plain_bf16(A.data_ptr(), W.data_ptr(), out.data_ptr(), M, W.shape[0], K, _stream_ptr()))
    return out


def op_lmhead_bf16(hidden, W_lm, scale: float, mask_id: int):
    import torch
    R, K = hidden.shape
    V = W_lm.shape[0]
    tok = torch.empty(R, device=hidden.device, dtype=torch.int32)
    conf = torch.empty(R, device=hidden.device, dtype=torch.float32)
    lse = torch.empty(R, device=hidden.device, dtype=torch.float32)
    scratch = torch.empty(lib().dlm_op_lmhead_scratch_bytes(R, V), device=hidden.device, dtype=torch.uint8)
    _op_check(lib().dlm_op_lmhead_bf16(hidden.data_ptr(), W_lm.data_ptr(), R, V, K, scale, mask_id, tok.data_ptr(),
                                       conf.data_ptr(), lse.data_ptr(), scratch.data_ptr(), _stream_ptr()))
    return tok, conf, lse


LMHEAD_STATIC_MAX_ROWS, LMHEAD_STATIC_SCRATCH_BYTES = 128, 4 << 20


def op_lmhead_static_bf16(hidden, W_lm, scale: float, mask_id: int, outs=None):
    """dlm_op_lmhead_static_bf16: the fused LM head for callers that cannot allocate device memory (a serving loop
    whose HBM was all handed to a pool at start-up, a section that cannot take cudaMalloc's device-wide
    synchronisation, a plug-in that is only given input and output buffers).  The scratch is an array inside libdlm.so,
    LMHEAD_STATIC_SCRATCH_BYTES per GPU, shared by every call: at most LMHEAD_STATIC_MAX_ROWS rows, and calls whose
    kernels could overlap on the GPU must be serialised by the caller.  Pass `outs` = (tok int32 [R], conf fp32 [R],
    lse fp32 [R]) to make this wrapper allocation-free as well; without it the three outputs come from torch."""
    import torch
    R, K = hidden.shape
    V = W_lm.shape[0]
    if outs is None:
        outs = (torch.empty(R, device=hidden.device, dtype=torch.int32), torch.empty(R, device=hidden.device, dtype=torch.float32),
                torch.empty(R, device=hidden.device, dtype=torch.float32))
    tok, conf, lse = outs
    _op_check(lib().dlm_op_lmhead_static_bf16(hidden.data_ptr(), W_lm.data_ptr(), R, V, K, scale, mask_id, tok.data_ptr(),
                                              conf.data_ptr(), lse.data_ptr(), _stream_ptr()))
    return tok, conf, lse


def op_lmhead_unmask_bf16(hidden, W_lm, n: int, B: int, scale: float, mask_id: int, tau, tokens_io, scratch=None, outs=None):
    import torch
    R, K = hidden.shape
    V = W_lm.shape[0]
    dev = hidden.device
    if scratch is None:
        scratch = torch.empty(lib().dlm_op_lmhead_scratch_bytes(R, V), device=dev, dtype=torch.uint8)
    if outs is None:
        outs = (torch.empty(n, device=dev, dtype=torch.int32), torch.empty(R, device=dev, dtype=torch.int32),
                torch.empty(R, device=dev, dtype=torch.int32), torch.empty(R, device=dev, dtype=torch.float32))
    ncomm, pos, tok, conf = outs
    _op_check(lib().dlm_op_lmhead_unmask_bf16(hidden.data_ptr(), W_lm.data_ptr(), n, B, V, K, scale, mask_id, tau.data_ptr(),
                                              tokens_io.data_ptr(), ncomm.data_ptr(), pos.data_ptr(), tok.data_ptr(),
                                              conf.data_ptr(), scratch.data_ptr(), _stream_ptr()))
    return ncomm, pos, tok, conf


def op_attention_bf16(q, k, v, flash=True):
    """flash: False/0 plain, True/1 mma.sync kernel, 2 tcgen05 kernel (auto K/V split), 2 + s tcgen05 with s splits."""
    import torch
    Tq, H, dh = q.shape
    S, Hkv, _ = k.shape
    out = torch.empty_like(q)
    _op_check(lib().dlm_op_attention_bf16(q.data_ptr(), k.data_ptr(), v.data_ptr(), out.data_ptr(), Tq, S, H, Hkv, dh,
                                          int(flash), _stream_ptr()))
    return out
