"""Pins for oracle/weights.py (Definition W): published splitmix64 vectors, hand-derived
bf16 rounding cases, the closed-form moments of the centred Irwin-Hall(4) draw, and torch's own
float32->bfloat16 conversion as an independent library routine."""
import os

import numpy as np
import pytest

from oracle import weights as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLDEN, name)) as f:
        return [l.split() for l in f if l.strip() and not l.startswith("#")]


def test_mix64_published_vectors():
    for k, want in _rows("splitmix64.txt"):
        z = np.uint64((0x9E3779B97F4A7C15 * int(k)) % 2**64)
        assert int(W.mix64(z)) == int(want, 16)


def test_bf16_rne_hand_cases():
    for bits, want, *_ in _rows("bf16_rne.txt"):
        x = np.array([int(bits, 16)], dtype=np.uint32).view(np.float32)
        got = W.round_to_bf16(x).view(np.uint32)[0] >> 16
        assert got == int(want, 16), (bits, hex(got))


def test_bf16_rne_matches_torch():
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(7)
    x = (rng.standard_normal(200000) * np.exp(rng.uniform(-20, 20, 200000))).astype(np.float32)
    want = torch.from_numpy(x).to(torch.bfloat16).to(torch.float32).numpy()
    assert np.array_equal(W.round_to_bf16(x), want)


def test_value_formula_by_hand():
    """One element recomputed with Python big integers, independent of numpy's uint64 wrap-around."""
    M = 2**64
    G = 0x9E3779B97F4A7C15

    def mix(z):
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) % M
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) % M
        return z ^ (z >> 31)

    seed, tid, shape = 1001, W.layer_tid(1, W.SUB_G), (5, 7)
    w = W.tensor_f32(seed, tid, shape, 0.02, False)
    key = mix((seed + G * (tid + 1)) % M)
    c = W.scale_constant(0.02)
    for i in (0, 1, 17, 34):
        h = mix((key + G * (i + 1)) % M)
        s = (h & 0xFFFF) + ((h >> 16) & 0xFFFF) + ((h >> 32) & 0xFFFF) + (h >> 48) - 131070
        assert w.reshape(-1)[i] == np.float32(s) * c


def test_moments_closed_form():
    """Centred Irwin-Hall(4) of 16-bit uniforms: mean 0, variance (2^32-1)/3 * c^2 = init_std^2,
    excess kurtosis -6/(5*4) = -0.3, |w| <= 131070*c (about 3.46 sigma)."""
    w = W.tensor_f32(5, 3, (2000, 1000), 0.02, False).astype(np.float64).reshape(-1)
    assert abs(w.mean()) < 5 * 0.02 / np.sqrt(len(w))
    assert abs(w.std() / 0.02 - 1) < 3e-3
    k = ((w - w.mean()) ** 4).mean() / w.var() ** 2 - 3.0
    assert abs(k - (-0.3)) < 0.02
    assert np.abs(w).max() <= 131070 * float(W.scale_constant(0.02)) * (1 + 1e-6)
    # distinct tensors / seeds decorrelate
    w2 = W.tensor_f32(5, 4, (2000, 1000), 0.02, False).astype(np.float64).reshape(-1)
    assert abs(np.corrcoef(w, w2)[0, 1]) < 5e-3


def test_chunking_and_rows_agree(tiny_arch):
    wt = W.Weights(tiny_arch, 11)
    full = W.tensor_f32(11, W.TID_EMBED, (tiny_arch.vocab, tiny_arch.d_model), 0.02, False, threads=1)
    assert np.array_equal(wt.rows(W.TID_EMBED, np.array([0, 5, 63])), full[[0, 5, 63]].astype(np.float64))
    big = W.tensor_f32(3, 9, (3, (1 << 22) + 5), 0.02, True)
    assert np.array_equal(big.reshape(-1)[(1 << 22) - 2:(1 << 22) + 3],
                          W._chunk(3, 9, (1 << 22) - 2, (1 << 22) + 3, W.scale_constant(0.02), True))
