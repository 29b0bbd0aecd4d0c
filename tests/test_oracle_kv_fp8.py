"""Pins of oracle/kv_fp8.py (FP8 e4m3 KV pages; readings DESIGN.md R13-R15) against things
other than itself: the format definition written out value by value, torch's own float8_e4m3fn type (a library
routine), closed forms of the scale rule, round-to-nearest-even ties, saturation, exact round trips, and the
identity "attention over fp8 pages = the fp64 attention oracle over the dequantised values".  No GPU."""
import numpy as np
import pytest

from oracle import attention as ora
from oracle import kv_fp8 as q8
from paper_2606_09061_b200 import workloads as wl


def test_table_against_the_format_definition_and_torch():
    t = q8.e4m3_table()
    # hand-written values of the definition (OCP FP8 E4M3: bias 7, subnormals m * 2^-9, max 448, no infinity)
    assert t[0x00] == 0.0 and t[0x01] == 2.0 ** -9 and t[0x07] == 7 * 2.0 ** -9 and t[0x08] == 2.0 ** -6
    assert t[0x38] == 1.0 and t[0x39] == 1.125 and t[0x40] == 2.0 and t[0x7E] == 448.0 and t[0x77] == 240.0
    assert np.isnan(t[0x7F]) and np.isnan(t[0xFF]) and t[0xB8] == -1.0 and t[0xFE] == -448.0
    assert np.all(np.diff(t[:0x7F]) > 0)                         # strictly increasing magnitudes
    torch = pytest.importorskip("torch")
    ref = torch.arange(256, dtype=torch.uint8).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    ok = ~np.isnan(t)
    assert np.array_equal(np.isnan(ref), np.isnan(t)) and np.array_equal(ref[ok], t[ok])


def test_encode_is_round_to_nearest_even_and_saturates():
    t = q8.e4m3_table()
    codes = np.arange(0x7F, dtype=np.uint8)
    assert np.array_equal(q8.encode_e4m3(t[:0x7F]), codes)       # every representable value keeps its code
    assert np.array_equal(q8.encode_e4m3(-t[1:0x7F]), codes[1:] | 0x80)
    # ties: 17 lies midway between 16 (0x58, even mantissa) and 18 (0x59); 19 between 18 and 20 (0x5A, even)
    assert q8.encode_e4m3(np.array([17.0]))[0] == 0x58 and q8.encode_e4m3(np.array([19.0]))[0] == 0x5A
    assert q8.encode_e4m3(np.array([17.0001]))[0] == 0x59 and q8.encode_e4m3(np.array([16.9999]))[0] == 0x58
    # subnormal grid: step 2^-9; 1.5 * 2^-9 is a tie between codes 1 and 2 -> 2 (even)
    assert q8.encode_e4m3(np.array([1.5 * 2.0 ** -9]))[0] == 0x02 and q8.encode_e4m3(np.array([0.4 * 2.0 ** -9]))[0] == 0x00
    # saturation, no NaN code is ever produced
    assert q8.encode_e4m3(np.array([1e9]))[0] == 0x7E and q8.encode_e4m3(np.array([-1e9]))[0] == 0xFE
    assert q8.encode_e4m3(np.array([464.0]))[0] == 0x7E
    # brute force on a dense grid: the chosen code is a nearest one
    y = np.linspace(-500, 500, 20001)
    d = np.abs(np.minimum(np.abs(y), 448.0)[:, None] - t[None, :0x7F])
    assert np.allclose(np.abs(t[q8.encode_e4m3(y) & 0x7F] - np.minimum(np.abs(y), 448.0)), d.min(axis=1), rtol=0, atol=0)


def test_encode_matches_torch_cast_in_range():
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(0)
    y = np.concatenate([rng.uniform(-448, 448, 5000), rng.standard_normal(5000) * 3, rng.uniform(-0.02, 0.02, 5000)])
    y = y.astype(np.float32).astype(np.float64)
    ref = torch.from_numpy(y.astype(np.float32)).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    got = q8.encode_e4m3(y)
    nz = (got & 0x7F) != 0                                        # the sign of a rounded-to-zero value is a convention
    assert np.array_equal(got[nz], ref[nz]) and np.all((ref[~nz] & 0x7F) == 0)


def test_scale_rule_closed_forms():
    e = q8.scale_exponent
    assert e(np.array([448.0]))[0] == 0 and e(np.array([448.0001]))[0] == 1 and e(np.array([224.0]))[0] == -1
    assert e(np.array([224.0001]))[0] == 0 and e(np.array([3.5]))[0] == -7 and e(np.array([3.6]))[0] == -6
    assert e(np.array([0.0]))[0] == q8.E_MIN and e(np.array([1e-9]))[0] == q8.E_MIN and e(np.array([1e9]))[0] == q8.E_MAX
    rng = np.random.default_rng(1)
    amax = np.exp(rng.uniform(np.log(0.02), np.log(50000.0), 2000))
    ee = e(amax).astype(np.float64)
    assert np.all(448.0 * 2.0 ** ee >= amax) and np.all(448.0 * 2.0 ** (ee - 1) < amax)    # the SMALLEST such power of two


def test_round_trip_properties():
    rng = np.random.default_rng(2)
    x = wl.bf16_bits_to_f64(wl.f32_to_bf16_bits(rng.standard_normal((64, 8, 128), dtype=np.float32) * np.float32(2.5)))
    codes, e = q8.quantize_rows(x)
    back = q8.dequantize(codes, e)
    amax = np.abs(x).max(axis=-1)
    # the row maximum lands in the top binade of the format: x / 2^e in (224, 448], so its code value in [224, 448]
    top = np.abs(q8.e4m3_table()[codes]).max(axis=-1)
    assert np.all(top >= 224.0) and np.all(top <= 448.0)
    scaled = amax * 2.0 ** -e.astype(np.float64)
    assert np.all(scaled > 224.0) and np.all(scaled <= 448.0)
    # error bound of a 3-bit mantissa: half an ulp = 2^-4 relative for normal values, 2^-10 * 2^e absolute below
    err = np.abs(back - x)
    bound = np.maximum(np.abs(x) * 2.0 ** -4, 2.0 ** -10 * 2.0 ** e.astype(np.float64)[..., None])
    assert np.all(err <= bound)
    # idempotent in value: the dequantised row is a fixed point (codes / scale may shift by one binade when the
    # row maximum rounded down to 224)
    codes2, e2 = q8.quantize_rows(back)
    assert np.array_equal(q8.dequantize(codes2, e2), back)
    # exact in bf16 (hence the attention oracle can take the pages as bf16 bit patterns)
    bits = q8.f64_to_bf16_bits_exact(back)
    assert np.array_equal(wl.bf16_bits_to_f64(bits), back)
    # a row scaled by a power of two keeps its codes and shifts its exponent
    codes3, e3 = q8.quantize_rows(x * 8.0)
    assert np.array_equal(codes3, codes) and np.array_equal(e3, e + 3)
    assert amax.min() > 0


def test_append_and_attention_over_fp8_pages_equal_the_definition():
    """kv_append_fp8 puts each row where the bf16 append puts it; attention over the pages (handed to the fp64
    oracle as exact bf16 bit patterns) equals dense numpy attention over the dequantised K / V."""
    rng = np.random.default_rng(3)
    Hq, Hkv, D, B, L = 4, 2, 64, 16, 70
    G = Hq // Hkv
    kb = wl.f32_to_bf16_bits(rng.standard_normal((L, Hkv, D), dtype=np.float32))
    vb = wl.f32_to_bf16_bits(rng.standard_normal((L, Hkv, D), dtype=np.float32))
    qb = wl.f32_to_bf16_bits(rng.standard_normal((L, Hq, D), dtype=np.float32))
    nb = (L + B - 1) // B
    bt = rng.permutation(nb + 3)[:nb].astype(np.int32)
    codes = np.full((nb + 3, 2, Hkv, B, D), 0x7F, np.uint8)       # NaN codes everywhere: stale slots
    scales = np.full((nb + 3, 2, Hkv, B), np.nan, np.float32)
    # append in two chunks (50 + 20): chunking cannot matter, every row is quantised on its own
    q8.kv_append_fp8(kb[:50], vb[:50], codes, scales, [50], [0], [bt])
    q8.kv_append_fp8(kb[50:], vb[50:], codes, scales, [20], [50], [bt])
    kc, ke = q8.quantize_rows(wl.bf16_bits_to_f64(kb))
    for t in (0, 17, 49, 50, 69):
        assert np.array_equal(codes[bt[t // B], 0, :, t % B], kc[t])
        assert np.array_equal(q8.scale_to_exponent(scales[bt[t // B], 0, :, t % B]), ke[t])
    nk = np.zeros(nb + 3, np.int64)
    nk[bt] = np.clip(L - np.arange(nb) * B, 0, B)
    pages = q8.pages_as_bf16_bits(codes, scales, nk)
    scale = float(np.float32(1.0) / np.sqrt(np.float32(D)))
    got = ora.attention(qb, pages, [L], [0], [bt], scale)
    K = q8.dequantize(*q8.quantize_rows(wl.bf16_bits_to_f64(kb)))
    V = q8.dequantize(*q8.quantize_rows(wl.bf16_bits_to_f64(vb)))
    Q = wl.bf16_bits_to_f64(qb)
    for h in range(Hq):
        s = (Q[:, h] @ K[:, h // G].T) * scale
        s = np.where(np.tril(np.ones((L, L), bool)), s, -np.inf)
        p = np.exp(s - s.max(axis=1, keepdims=True))
        want = (p @ V[:, h // G]) / p.sum(axis=1, keepdims=True)
        assert np.abs(got[:, h] - want).max() <= 1e-12
