"""Pins of oracle/rope.py against what the mathematics fixes (no GPU).

Each test would fail for one plausible mistake: a flipped sine sign, interleaved instead of
rotate-half pairing, position off by one, frequencies indexed by the wrong half, V rotated,
a fused multiply-add or a wrong rounding mode in the bf16 decision.
"""
import numpy as np
import pytest

from oracle import attention as ora
from oracle import rope

COS1, SIN1 = 0.5403023058681398, 0.8414709848078965          # cos 1, sin 1 (tables)
COS_HALF, SIN_HALF = 0.8775825618903728, 0.479425538604203   # cos 0.5, sin 0.5


def _bits(x):
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    return ((u + (((u >> 16) & 1) + np.uint32(0x7FFF))) >> 16).astype(np.uint16)


def _f64(b):
    return (np.asarray(b, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def test_closed_form_single_pair_sign_convention():
    w = np.array([1.0])
    x = np.array([[[1.0, 0.0]], [[0.0, 1.0]]])                 # two tokens, both at position 1
    y = rope.rope_f64(x, np.array([1, 1]), w)
    np.testing.assert_allclose(y[0, 0], [COS1, SIN1], atol=1e-15)
    np.testing.assert_allclose(y[1, 0], [-SIN1, COS1], atol=1e-15)


def test_closed_form_rotate_half_pairing_and_frequency_index():
    w = np.array([1.0, 0.5])
    x = np.eye(4)[:, None, :]                                  # rows e_0 .. e_3, all at position 1
    y = rope.rope_f64(x, np.ones(4, dtype=np.int64), w)[:, 0]
    np.testing.assert_allclose(y[0], [COS1, 0, SIN1, 0], atol=1e-15)            # e_0 pairs with element 2
    np.testing.assert_allclose(y[1], [0, COS_HALF, 0, SIN_HALF], atol=1e-15)    # e_1 uses w_1
    np.testing.assert_allclose(y[2], [-SIN1, 0, COS1, 0], atol=1e-15)
    np.testing.assert_allclose(y[3], [0, -SIN_HALF, 0, COS_HALF], atol=1e-15)


def test_default_inv_freq():
    w = rope.default_inv_freq(128, 10000.0)
    assert w.shape == (64,) and w[0] == 1.0
    np.testing.assert_allclose(w[1:] / w[:-1], 10000.0 ** (-1.0 / 64), rtol=1e-12)
    np.testing.assert_allclose(w[-1], 1.1548e-4, rtol=1e-3)   # 10^(-4 * 126/128)


def test_matches_complex_multiplication_form():
    rng = np.random.default_rng(1)
    T, H, D = 9, 3, 16
    x = rng.standard_normal((T, H, D))
    pos = rng.integers(0, 40000, size=T)
    w = rope.default_inv_freq(D)
    z = (x[..., : D // 2] + 1j * x[..., D // 2:]) * np.exp(1j * pos[:, None, None] * w[None, None, :])
    want = np.concatenate([z.real, z.imag], axis=-1)
    np.testing.assert_allclose(rope.rope_f64(x, pos, w), want, atol=1e-12)


def test_identity_composition_norm_and_relative_position():
    rng = np.random.default_rng(2)
    T, H, D = 7, 2, 32
    x = rng.standard_normal((T, H, D))
    w = rope.default_inv_freq(D, 500000.0)
    zero = np.zeros(T, dtype=np.int64)
    assert np.array_equal(rope.rope_f64(x, zero, w), x)
    a, b = rng.integers(0, 3000, size=T), rng.integers(0, 3000, size=T)
    np.testing.assert_allclose(rope.rope_f64(rope.rope_f64(x, a, w), b, w), rope.rope_f64(x, a + b, w), atol=1e-10)
    y = rope.rope_f64(x, a, w)
    np.testing.assert_allclose(y[..., : D // 2] ** 2 + y[..., D // 2:] ** 2,
                               x[..., : D // 2] ** 2 + x[..., D // 2:] ** 2, atol=1e-12)
    q, k = rng.standard_normal((1, 1, D)), rng.standard_normal((1, 1, D))
    dots = [float((rope.rope_f64(q, [m + s], w) * rope.rope_f64(k, [n + s], w)).sum())
            for (m, n) in [(17, 5)] for s in (0, 1, 1000, 31000)]
    np.testing.assert_allclose(dots, dots[0], atol=1e-9)
    assert abs(dots[0] - float((q * k).sum())) > 1e-3          # ... and it does depend on m - n


def test_token_positions():
    np.testing.assert_array_equal(rope.token_positions([3, 1, 2], [0, 99, 48]), [0, 1, 2, 99, 48, 49])


def test_bf16_decision_is_half_ulp_from_definition_and_exact_at_position_zero():
    rng = np.random.default_rng(3)
    T, H, D = 64, 4, 128
    xb = _bits(rng.standard_normal((T, H, D), dtype=np.float32))
    pos = rng.integers(0, 131072, size=T)
    w = rope.default_inv_freq(D)
    got = _f64(rope.rope_bf16(xb, pos, w))
    want = rope.rope_f64(_f64(xb), pos, w)
    ulp = 2.0 ** (np.floor(np.log2(np.maximum(np.abs(want), 1e-30))) - 7)       # bf16: 8 significant bits
    assert (np.abs(got - want) <= 0.5 * ulp + 4e-7 * np.abs(want).max()).all()
    assert np.array_equal(rope.rope_bf16(xb, np.zeros(T, dtype=np.int64), w), xb)


def test_bf16_decision_rounds_to_nearest_even():
    # 1 + 2^-8 lies exactly between the bf16 neighbours 1 and 1 + 2^-7: ties go to the even code (1.0)
    x = np.array([[[1.0 + 2.0 ** -8, 0.0]]], dtype=np.float32)
    xb = (x.view(np.uint32) >> 16).astype(np.uint16)            # truncation: 1.0 exactly
    assert xb[0, 0, 0] == 0x3F80
    tie = np.array([1.0 + 2.0 ** -8], dtype=np.float32)
    assert rope._f32_to_bf16_bits_rne(tie)[0] == 0x3F80
    assert rope._f32_to_bf16_bits_rne(np.array([1.0 + 3 * 2.0 ** -8], dtype=np.float32))[0] == 0x3F82


@pytest.mark.parametrize("cuts", [[24], [1, 7, 16], [5, 5, 5, 5, 4]])
def test_chunking_invariance_with_rope(cuts):
    """A prompt rotated by absolute position and processed in chunks equals the unchunked
    prompt (north_star's chunking invariance carries over: positions are absolute)."""
    rng = np.random.default_rng(4)
    L, Hq, Hkv, D, B = 24, 4, 2, 32, 16
    assert sum(cuts) == L
    w = rope.default_inv_freq(D)
    qb = _bits(rng.standard_normal((L, Hq, D), dtype=np.float32))
    kb = _bits(rng.standard_normal((L, Hkv, D), dtype=np.float32))
    vb = _bits(rng.standard_normal((L, Hkv, D), dtype=np.float32))
    table = [np.array([1, 0], dtype=np.int32)]
    scale = float(1.0 / np.sqrt(D))

    def run(chunks):
        cache = np.zeros((2, 2, Hkv, B, D), dtype=np.uint16)
        outs, off = [], 0
        for n in chunks:
            pos = rope.token_positions([n], [off])
            ora.kv_append(rope.rope_bf16(kb[off:off + n], pos, w), vb[off:off + n], cache, [n], [off], table)
            outs.append(ora.attention(rope.rope_bf16(qb[off:off + n], pos, w), cache, [n], [off], table, scale))
            off += n
        return np.concatenate(outs), cache

    whole, cache_w = run([L])
    parts, cache_p = run(cuts)
    assert np.array_equal(cache_w, cache_p)
    np.testing.assert_allclose(parts, whole, atol=1e-12)
    # V is not rotated: the V half of the pages holds the input bits
    assert np.array_equal(cache_w[1, 1, :, :B, :].transpose(1, 0, 2), vb[:B])
