"""dlm_op_lmhead_static_bf16 (-m gpu): the fused LM head for callers that cannot allocate device memory.

Some users of this library run where cudaMalloc is not an option: a serving loop that gave all of its HBM to a pool
at start-up and must not grow, a latency-critical section that cannot take the device-wide synchronisation an
allocation implies, a plug-in that only ever receives input and output buffers.  For them the split-vocabulary
scratch of the LM head lives in a fixed array inside libdlm.so (LMHEAD_STATIC_SCRATCH_BYTES per GPU, at most
LMHEAD_STATIC_MAX_ROWS rows) that every call shares and that keeps the previous call's contents.

What is checked: the entry point gives what dlm_op_lmhead_bf16 gives with a caller-owned scratch buffer (same kernels:
token ids identical, conf / lse within the bounds tests/test_gpu_ops.py::test_lmhead_stats uses), on two calls in a
row with different shapes, so that records the first call left in the array lie inside and beyond the second call's
regions; sizes beyond the array are refused with DLM_E_CAPACITY and the numbers in the message; a call with
pre-allocated outputs leaves the device's free memory where it was.

This file sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide the parity
tests.  It does not depend on anything the other tests leave behind and passes alone in a fresh process too.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

CONF_TOL = 2e-5          # as test_lmhead_stats
LSE_TOL = 1e-4           # relative to max(1, max |lse|), as test_lmhead_stats


def _inputs(seed, R, V, K):
    rng = np.random.default_rng(seed)
    H = torch.from_numpy(rng.standard_normal((R, K)).astype(np.float32)).to(torch.bfloat16).cuda()
    W = torch.from_numpy((rng.standard_normal((V, K)) * 0.08).astype(np.float32)).to(torch.bfloat16).cuda()
    return H, W


def _same(got, want):
    tok, conf, lse = (t.cpu().numpy() for t in got)
    tok_w, conf_w, lse_w = (t.cpu().numpy() for t in want)
    assert np.array_equal(tok, tok_w)
    assert np.abs(conf.astype(np.float64) - conf_w).max() < CONF_TOL
    assert np.abs(lse.astype(np.float64) - lse_w).max() < LSE_TOL * max(1.0, np.abs(lse_w).max())


def test_static_lmhead_matches_scratch_path_on_consecutive_calls():
    import paper_2606_29094_b200 as pkg
    scale = 4.0
    # (R, V, K, mask_id): ragged rows and vocabulary tails; the second call is smaller in both, the third is the
    # largest row count the array takes, with a vocabulary of 1000 tiles
    shapes = [(100, 5000, 256, 4999), (37, 3001, 128, 7), (128, 128000, 64, 0)]
    cases = []
    for i, (R, V, K, mask_id) in enumerate(shapes):
        H, W = _inputs(100 + i, R, V, K)
        want = pkg.op_lmhead_bf16(H, W, scale, mask_id)        # existing path: caller-owned scratch from torch
        torch.cuda.synchronize()
        cases.append((H, W, mask_id, want))
    # back-to-back on one stream, nothing in between: call 2 finds call 1's records in the array
    got = [pkg.op_lmhead_static_bf16(H, W, scale, mask_id) for H, W, mask_id, _ in cases]
    torch.cuda.synchronize()
    for g, (_, _, _, want) in zip(got, cases):
        _same(g, want)
    # and the other way round, twice the same shape at the end
    order = [2, 0, 1, 1]
    got = [pkg.op_lmhead_static_bf16(cases[j][0], cases[j][1], scale, cases[j][2]) for j in order]
    torch.cuda.synchronize()
    for g, j in zip(got, order):
        _same(g, cases[j][3])


def test_static_lmhead_refuses_sizes_beyond_the_array():
    import paper_2606_29094_b200 as pkg
    L = pkg.lib()
    assert L.dlm_op_lmhead_static_bytes(128, 152064) <= pkg.LMHEAD_STATIC_SCRATCH_BYTES      # the largest config fits
    H, W = _inputs(1, pkg.LMHEAD_STATIC_MAX_ROWS + 1, 512, 64)
    with pytest.raises(pkg.DlmError) as e:
        pkg.op_lmhead_static_bf16(H, W, 1.0, 0)
    assert e.value.code == -2 and "129" in str(e.value)                                      # DLM_E_CAPACITY
    V_big = 300000                                                                           # 128 x 2344 tiles x 16 B > 4 MiB
    assert L.dlm_op_lmhead_static_bytes(128, V_big) > pkg.LMHEAD_STATIC_SCRATCH_BYTES
    H = torch.zeros(128, 8, dtype=torch.bfloat16, device="cuda")
    W = torch.zeros(V_big, 8, dtype=torch.bfloat16, device="cuda")
    with pytest.raises(pkg.DlmError) as e:
        pkg.op_lmhead_static_bf16(H, W, 1.0, 0)
    assert e.value.code == -2
    # a refused call launched nothing and the next good call is unaffected
    H, W = _inputs(2, 64, 1000, 64)
    want = pkg.op_lmhead_bf16(H, W, 2.0, 999)
    _same(pkg.op_lmhead_static_bf16(H, W, 2.0, 999), want)


def test_static_lmhead_leaves_free_memory_unchanged():
    import paper_2606_29094_b200 as pkg
    R, V, K = 64, 20000, 128
    H, W = _inputs(3, R, V, K)
    outs = (torch.empty(R, device="cuda", dtype=torch.int32), torch.empty(R, device="cuda", dtype=torch.float32),
            torch.empty(R, device="cuda", dtype=torch.float32))
    pkg.op_lmhead_static_bf16(H, W, 4.0, 5, outs=outs)       # first use: address look-up, kernel images loaded
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        pkg.op_lmhead_static_bf16(H, W, 4.0, 5, outs=outs)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    _same(outs, pkg.op_lmhead_bf16(H, W, 4.0, 5))
