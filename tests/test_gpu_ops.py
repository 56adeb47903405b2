"""Kernel-level parity (-m gpu): each CUDA kernel reached through the C ABI (include/dlm_ops.h) against the
oracle / numpy float64 on the same seeded inputs (tier T1; DESIGN.md protocol P-C stages)."""
import numpy as np
import pytest

from oracle import model as omodel, step as ostep

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


# fp32 accumulation in tensor memory over K <= 12 288: measured max |error| 1.5e-6 .. 5.2e-6 of max |out| on B200
# (K = 4096 / 12 288, 32 and 512 rows); the bound is twice the largest value measured.
GEMM_TOL = 1e-5

def _bf16(x):
    return torch.from_numpy(x).to(torch.bfloat16)


def _f64(t):
    return t.to(torch.float32).cpu().numpy().astype(np.float64)


def _mk(rng, rows, cols, scale=1.0):
    t = _bf16((rng.standard_normal((rows, cols)) * scale).astype(np.float32))
    return t.cuda(), _f64(t)


GEMM_SHAPES = [  # (M, N, K): several tiles + ragged tails in every dimension
    (32, 256, 128), (1, 64, 64), (100, 384, 688), (300, 200, 512), (129, 96, 4096), (512, 768, 256), (33, 1056, 200)]


@pytest.mark.parametrize("M,N,K", GEMM_SHAPES)
@pytest.mark.parametrize("bn", [0, 32, 64, 96, 128, 192, 256])
def test_gemm_tc_store_and_residual(M, N, K, bn):
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(M * 7 + N * 3 + K + bn)
    A, a = _mk(rng, M, K)
    W, w = _mk(rng, N, K, 0.05)
    want = a @ w.T
    tol = GEMM_TOL * np.abs(want).max() + 1e-6
    got = pkg.op_gemm_bf16(A, W, pkg.EPI_F32, bn)
    torch.cuda.synchronize()
    assert np.abs(_f64(got) - want).max() <= tol
    # residual: x += A W^T
    x0 = rng.standard_normal((M, N)).astype(np.float32)
    x = torch.from_numpy(x0).cuda()
    pkg.op_gemm_bf16(A, W, pkg.EPI_RESID, bn, out=x)
    torch.cuda.synchronize()
    assert np.abs(_f64(x) - (x0.astype(np.float64) + want)).max() <= tol + 1e-6
    # bf16 store
    gb = pkg.op_gemm_bf16(A, W, pkg.EPI_BF16, bn)
    torch.cuda.synchronize()
    assert np.all(np.abs(_f64(gb) - want) <= np.abs(want) * 2 ** -8 + tol)


@pytest.mark.parametrize("M,F,K", [(32, 128, 128), (70, 688, 256), (256, 352, 512), (5, 64, 64)])
@pytest.mark.parametrize("bn", [0, 64, 128, 192, 256])
def test_gemm_tc_swiglu(M, F, K, bn):
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(M + F + K + bn)
    A, a = _mk(rng, M, K)
    W, w = _mk(rng, 2 * F, K, 0.1)
    g, u = a @ w[:F].T, a @ w[F:].T
    want = omodel.silu(g) * u
    got = pkg.op_gemm_bf16(A, W, pkg.EPI_SWIGLU, bn)
    torch.cuda.synchronize()
    assert got.shape == (M, F)
    assert np.all(np.abs(_f64(got) - want) <= np.abs(want) * 2 ** -8 + 1e-4)


PAIR_SHAPES = [  # (M, N, K): one and several 256-row tiles, ragged tails in every dimension, > 1 tile per pair
    (129, 256, 128), (300, 200, 512), (512, 768, 256), (257, 96, 4096), (1000, 1056, 200), (2240, 512, 320), (130, 4608, 64)]


@pytest.mark.parametrize("M,N,K", PAIR_SHAPES)
@pytest.mark.parametrize("bn", [0, 64, 96, 160, 256])
def test_gemm_pair_store_and_residual(M, N, K, bn):
    """Persistent CTA-pair tcgen05 GEMM (refresh-step a3/a6/a9) vs fp64 matmul."""
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(M * 7 + N * 3 + K + bn)
    A, a = _mk(rng, M, K)
    W, w = _mk(rng, N, K, 0.05)
    want = a @ w.T
    tol = GEMM_TOL * np.abs(want).max() + 1e-6
    got = pkg.op_gemm_pair_bf16(A, W, pkg.EPI_F32, bn)
    torch.cuda.synchronize()
    assert np.abs(_f64(got) - want).max() <= tol
    x0 = rng.standard_normal((M, N)).astype(np.float32)
    x = torch.from_numpy(x0).cuda()
    pkg.op_gemm_pair_bf16(A, W, pkg.EPI_RESID, bn, out=x)
    torch.cuda.synchronize()
    assert np.abs(_f64(x) - (x0.astype(np.float64) + want)).max() <= tol + 1e-6
    gb = pkg.op_gemm_pair_bf16(A, W, pkg.EPI_BF16, bn)
    torch.cuda.synchronize()
    assert np.all(np.abs(_f64(gb) - want) <= np.abs(want) * 2 ** -8 + tol)


@pytest.mark.parametrize("M,N,K", [(512, 512, 4096), (300, 200, 1024), (257, 96, 4096), (1000, 1056, 640)])
@pytest.mark.parametrize("splits", [0, 2, 3, 4])
def test_gemm_pair_split_k(M, N, K, splits):
    """Split-K units of the CTA-pair kernel (O / down projections of a 512-token step): slices summed in order."""
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(M + N + K + splits)
    A, a = _mk(rng, M, K)
    W, w = _mk(rng, N, K, 0.05)
    want = a @ w.T
    tol = GEMM_TOL * np.abs(want).max() + 1e-6
    got, ns = pkg.op_gemm_pair_bf16(A, W, pkg.EPI_F32, 0 if splits == 0 else 256, splits=splits, return_splits=True)
    torch.cuda.synchronize()
    assert 1 <= ns <= 4 and (splits == 0 or ns <= splits)
    assert np.abs(_f64(got) - want).max() <= tol


@pytest.mark.parametrize("M,F,K", [(200, 128, 128), (270, 688, 256), (600, 352, 512), (129, 64, 64), (512, 1536, 1024)])
@pytest.mark.parametrize("bn", [0, 64, 128, 192, 256])
def test_gemm_pair_swiglu(M, F, K, bn):
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(M + F + K + bn)
    A, a = _mk(rng, M, K)
    W, w = _mk(rng, 2 * F, K, 0.1 if K < 1024 else 0.03)
    want = omodel.silu(a @ w[:F].T) * (a @ w[F:].T)
    got = pkg.op_gemm_pair_bf16(A, W, pkg.EPI_SWIGLU, bn)
    torch.cuda.synchronize()
    assert got.shape == (M, F)
    assert np.all(np.abs(_f64(got) - want) <= np.abs(want) * 2 ** -8 + 2e-4)


@pytest.mark.parametrize("M,F,K", [(512, 12288, 256), (1000, 12200, 128), (300, 11000, 192)])
def test_gemm_pair_swiglu_mixed_tile_widths(M, F, K):
    """Gate/up projections of <= 1024 rows with many column blocks: the automatic plan deals the first column blocks wide and the
    rest narrow (two tile widths in one launch); results against fp64 on every element, ragged tails in the
    rows and in the features (12 200 and 11 000 are multiples of neither width), and the plan really is mixed."""
    import paper_2606_29094_b200 as pkg
    bn, bn2, n_wide = pkg.op_gemm_pair_plan(M, F, K, pkg.EPI_SWIGLU)
    assert bn2 in (64, 128, 192) and bn2 < bn and 0 < n_wide < (F + bn // 2 - 1) // (bn // 2), (bn, bn2, n_wide)
    rng = np.random.default_rng(M + F + K)
    A, a = _mk(rng, M, K)
    W, w = _mk(rng, 2 * F, K, 0.1)
    want = omodel.silu(a @ w[:F].T) * (a @ w[F:].T)
    got = pkg.op_gemm_pair_bf16(A, W, pkg.EPI_SWIGLU, 0)
    uniform = pkg.op_gemm_pair_bf16(A, W, pkg.EPI_SWIGLU, 256)
    torch.cuda.synchronize()
    assert np.all(np.abs(_f64(got) - want) <= np.abs(want) * 2 ** -8 + 2e-4)
    assert np.array_equal(_f64(got), _f64(uniform))            # same K order per element whatever the tile width: bit-identical


SKINNY_SHAPES = [  # (T, N, K): tails in every dimension, one and several K blocks per split
    (32, 256, 128), (1, 128, 64), (32, 4096, 4096), (17, 384, 688), (64, 200, 512), (100, 1056, 200), (128, 768, 256), (33, 96, 4096)]


@pytest.mark.parametrize("T,N,K", SKINNY_SHAPES)
@pytest.mark.parametrize("splits", [0, 1, 3, 16])
def test_gemm_skinny_partial(T, N, K, splits):
    """Weight-streaming swap-AB split-K GEMM (cached step a3/a6/a9) vs fp64 matmul."""
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(T * 5 + N + K + splits)
    X, x = _mk(rng, T, K)
    W, w = _mk(rng, N, K, 0.05)
    want = x @ w.T
    tol = GEMM_TOL * np.abs(want).max() + 1e-6
    got, ns = pkg.op_gemm_skinny_bf16(X, W, pkg.EPI_F32, splits)
    torch.cuda.synchronize()
    assert 1 <= ns <= 16 and (splits in (0,) or ns <= splits)
    assert np.abs(_f64(got) - want).max() <= tol


@pytest.mark.parametrize("T,F,K", [(32, 128, 128), (70, 688, 256), (128, 352, 512), (5, 64, 64), (32, 12288, 4096)])
def test_gemm_skinny_swiglu(T, F, K):
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(T + F + K)
    X, x = _mk(rng, T, K)
    W, w = _mk(rng, 2 * F, K, 0.1 if K < 1024 else 0.02)
    want = omodel.silu(x @ w[:F].T) * (x @ w[F:].T)
    got, _ = pkg.op_gemm_skinny_bf16(X, W, pkg.EPI_SWIGLU)
    torch.cuda.synchronize()
    assert got.shape == (T, F)
    assert np.all(np.abs(_f64(got) - want) <= np.abs(want) * 2 ** -8 + 2e-4)


def test_gemm_plain_matches():
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(3)
    A, a = _mk(rng, 70, 200)
    W, w = _mk(rng, 130, 200, 0.05)
    got = pkg.op_gemm_plain_bf16(A, W)
    torch.cuda.synchronize()
    assert np.abs(_f64(got) - a @ w.T).max() < 1e-4


@pytest.mark.parametrize("R,V,K,mask_id", [(32, 4096, 256, 4095), (7, 1000, 64, 0), (130, 126464 // 8, 512, 77), (64, 300, 128, 299)])
def test_lmhead_stats(R, V, K, mask_id):
    """S7: final-normed rows -> fused LM head (no logits in HBM) -> (tok, conf, lse) vs oracle.confidence."""
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(R + V)
    H, h = _mk(rng, R, K)
    wn = (rng.standard_normal((V, K)) * 0.08).astype(np.float32)
    # exact tie for row 0 across two vocabulary tiles: two identical weight rows aligned with h[0] (lowest id wins, G8)
    i1, i2 = (mask_id + 5) % V, (mask_id + 5 + min(V - 10, 200)) % V
    wn[i1] = wn[i2] = (h[0] * 0.05).astype(np.float32)
    Wt = _bf16(wn)
    W, w = Wt.cuda(), _f64(Wt)
    scale = 4.0
    z = scale * (h @ w.T)
    z[:, mask_id] = -np.inf
    tok_o, conf_o, lse_o, margin = omodel.confidence(z)
    assert tok_o[0] in (i1, i2) and abs(margin[0]) < 1e-12      # a tie up to BLAS summation order in fp64
    tok, conf, lse = pkg.op_lmhead_bf16(H, W, scale, mask_id)
    torch.cuda.synchronize()
    tok, conf, lse = tok.cpu().numpy(), conf.cpu().numpy().astype(np.float64), lse.cpu().numpy().astype(np.float64)
    assert tok[0] == min(i1, i2)                                 # exact tie on the device -> lowest id (G8)
    clear = margin >= 1e-3
    assert np.array_equal(tok[clear], tok_o[clear])
    assert (tok != mask_id).all() and (tok >= 0).all() and (tok < V).all()
    assert np.abs(conf - conf_o).max() < 2e-5
    assert np.abs(lse - lse_o).max() < 1e-4 * max(1.0, np.abs(lse_o).max())
    # near ties: the GPU's choice must be one of the (near-)maximal ids
    for r in np.flatnonzero(~clear):
        assert z[r, tok[r]] >= z[r].max() - 1e-2


def test_lmhead_unmask_fused_bit_exact_vs_rule():
    """S8: the unmask rule applied by the kernel to ITS OWN (tok, conf) equals oracle.unmask on those values:
    bit-exact, no band (both sides compare in fp32)."""
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(11)
    n, B, V, K, mask_id = 12, 32, 2048, 128, 2047
    H, _ = _mk(rng, n * B, K)
    W, _ = _mk(rng, V, K, 0.5)          # peaked distributions -> confidences spread over (0, 1)
    tok_r, conf_r, _ = pkg.op_lmhead_bf16(H, W, 1.0, mask_id)
    torch.cuda.synchronize()
    tok_r, conf_r = tok_r.cpu().numpy(), conf_r.cpu().numpy()
    taus = np.array([0.0, 0.3, 0.5, 0.7, 0.9, 0.95, 1.5, 0.5, 0.9, 0.2, 0.6, 2.0], np.float32)
    tokens = np.full((n, B), mask_id, np.int32)
    for i in range(n):                  # some positions already committed; request 7 fully committed
        keep = rng.random(B) < (0.4 if i != 7 else 1.1)
        tokens[i, keep] = rng.integers(0, mask_id, keep.sum())
    tio = torch.from_numpy(tokens.copy()).cuda()
    ncomm, pos, tok, conf = pkg.op_lmhead_unmask_bf16(H, W, n, B, 1.0, mask_id, torch.from_numpy(taus).cuda(), tio)
    torch.cuda.synchronize()
    ncomm, pos, tok, conf, tio = (t.cpu().numpy() for t in (ncomm, pos, tok, conf, tio))
    for i in range(n):
        t = tokens[i].astype(np.int64).copy()
        want = ostep.unmask(t, 0, B, tok_r[i * B:(i + 1) * B], conf_r[i * B:(i + 1) * B], taus[i], mask_id)
        k = int(ncomm[i])
        assert k == len(want)
        assert [(int(pos[i * B + j]), int(tok[i * B + j])) for j in range(k)] == [(c.pos, c.tok) for c in want]
        assert np.array_equal(conf[i * B:i * B + k], np.array([c.conf for c in want], np.float32))
        assert np.array_equal(tio[i], t.astype(np.int32))
        if taus[i] > 1 and (tokens[i] == mask_id).any():
            assert k == 1
        if taus[i] <= 0:
            assert k == (tokens[i] == mask_id).sum()


@pytest.mark.parametrize("Tq,S,H,Hkv", [(32, 512, 4, 4), (64, 200, 8, 2), (5, 64, 2, 1), (100, 1000, 7, 1), (512, 512, 2, 2)])
@pytest.mark.parametrize("flash", [True, False])
def test_attention(Tq, S, H, Hkv, flash):
    """S2: softmax(QK^T/sqrt d)V without mask, GQA, ragged lengths, vs oracle.attention (fp64)."""
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(Tq + S + H)
    dh = 128
    q = _bf16(rng.standard_normal((Tq, H, dh)).astype(np.float32)).cuda()
    k = _bf16(rng.standard_normal((S, Hkv, dh)).astype(np.float32)).cuda()
    v = _bf16(rng.standard_normal((S, Hkv, dh)).astype(np.float32)).cuda()
    want = omodel.attention(_f64(q), _f64(k), _f64(v))
    got = _f64(pkg.op_attention_bf16(q, k, v, flash))
    assert np.isfinite(got).all()
    err = np.abs(got - want).max()
    assert err < (6e-3 if flash else 3e-3), err      # P rounded to bf16 for the PV MMA + bf16 output


@pytest.mark.parametrize("Tq,S,H,Hkv", [(32, 512, 4, 4), (64, 200, 8, 2), (5, 64, 2, 1), (100, 1000, 7, 1), (512, 512, 2, 2),
                                        (32, 4608, 2, 2), (300, 300, 4, 2), (64, 129, 1, 1), (9, 700, 14, 2), (33, 1000, 3, 3)])
@pytest.mark.parametrize("mode", [2, 3, 5, 102, 104])
def test_attention_tcgen05(Tq, S, H, Hkv, mode):
    """tcgen05/TMEM attention vs oracle.attention (fp64): ragged tails in rows and K/V, GQA stacking, several tiles per
    item, optional K/V split.  Modes 2.. take the transposed-score kernel when Tq * H / H_kv <= 64 and the row-major
    kernel (128-row query tiles, lazy rescale) otherwise; modes 102.. force the row-major kernel."""
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(Tq + S + H + mode)
    dh = 128
    q = _bf16((rng.standard_normal((Tq, H, dh)) * 1.5).astype(np.float32)).cuda()
    k = _bf16(rng.standard_normal((S, Hkv, dh)).astype(np.float32)).cuda()
    v = _bf16(rng.standard_normal((S, Hkv, dh)).astype(np.float32)).cuda()
    want = omodel.attention(_f64(q), _f64(k), _f64(v))
    got = _f64(pkg.op_attention_bf16(q, k, v, mode))
    assert np.isfinite(got).all()
    err = np.abs(got - want).max()
    assert err < 8e-3, err      # P rounded to bf16 for the PV MMA + bf16 output


def test_attention_tcgen05_growing_scores():
    """Scores that keep growing along K/V force the lazy-rescale path (running max raised by > 2^8 several times)."""
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(77)
    Tq, S, H, dh = 40, 1024, 2, 128
    qn = rng.standard_normal((Tq, H, dh)).astype(np.float32)
    kn = rng.standard_normal((S, H, dh)).astype(np.float32) * 0.3
    kn += (np.arange(S, dtype=np.float32)[:, None, None] / S) * 2.5 * np.sign(qn[0:1, :, :])   # drift along q[0]
    q, k = _bf16(qn).cuda(), _bf16(kn).cuda()
    v = _bf16(rng.standard_normal((S, H, dh)).astype(np.float32)).cuda()
    want = omodel.attention(_f64(q), _f64(k), _f64(v))
    for mode in (2, 3, 102, 103):        # transposed-score kernel (exact-maxima pass) and row-major kernel (lazy rescale)
        got = _f64(pkg.op_attention_bf16(q, k, v, mode))
        assert np.isfinite(got).all()
        assert np.abs(got - want).max() < 8e-3


def test_attention_plain_small_head():
    import paper_2606_29094_b200 as pkg
    rng = np.random.default_rng(5)
    q = _bf16(rng.standard_normal((9, 4, 64)).astype(np.float32)).cuda()
    k = _bf16(rng.standard_normal((70, 2, 64)).astype(np.float32)).cuda()
    v = _bf16(rng.standard_normal((70, 2, 64)).astype(np.float32)).cuda()
    want = omodel.attention(_f64(q), _f64(k), _f64(v))
    assert np.abs(_f64(pkg.op_attention_bf16(q, k, v, False)) - want).max() < 3e-3
    with pytest.raises(pkg.DlmError):
        pkg.op_attention_bf16(q, k, v, True)       # flash kernel is d_h = 128 only and says so
