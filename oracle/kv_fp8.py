"""FP8 (e4m3) KV pages: the quantisation decision and its inverse (TEST INFRASTRUCTURE, not product code).

SURVEY.md 8(f) N2, second half ("FP8 (e4m3) KV pages with per-page scales -- halves decode bytes"; the
paper only says that decode is memory-bandwidth-bound, and leaves the execution backend
untouched).  The paper defines none of it; the readings are DESIGN.md R13-R15:

  * format: OCP FP8 E4M3 ("e4m3fn"): 1 sign, 4 exponent (bias 7), 3 mantissa bits; exponent field 0 is
    subnormal (m * 2^-9); exponent 15 with mantissa 7 is NaN, there is no infinity; largest finite 448.
  * one scale per (token, KV head, K|V) row of D elements, a POWER OF TWO 2^e with
        e = the smallest integer such that 448 * 2^e >= amax(row),   clamped to [-15, 7]
    (so dequantisation is an exact exponent shift, exact in bf16 and in fp16; a row whose amax exceeds
    448 * 2^7 = 57344 saturates; an all-zero row takes e = -15);
  * code = round-to-nearest-even of x * 2^-e onto the e4m3 grid, saturating at +-448;
  * the value a page holds is code_value * 2^e, EXACTLY; attention over fp8 pages is the plain definition
    (oracle/attention_oracle.c) over those values -- they are exactly representable in bf16, so the pages are
    handed to the fp64 attention oracle as bf16 bit patterns, unchanged arithmetic.

Nothing here imports the product package.  numpy only; plain loops / table look-ups, no blocking.
"""
import numpy as np

E_MIN, E_MAX = -15, 7          # clamp of the row scale exponent (R14)
E4M3_MAX = 448.0


def e4m3_table() -> np.ndarray:
    """Value of each of the 256 codes, from the format definition (float64; NaN for 0x7F / 0xFF)."""
    out = np.empty(256, dtype=np.float64)
    for code in range(256):
        sign = -1.0 if code & 0x80 else 1.0
        exp = (code >> 3) & 0xF
        man = code & 0x7
        if exp == 0xF and man == 0x7:
            out[code] = np.nan
        elif exp == 0:
            out[code] = sign * man * 2.0 ** -9                  # subnormal: 0.mmm * 2^-6
        else:
            out[code] = sign * (1.0 + man / 8.0) * 2.0 ** (exp - 7)
    return out


_TABLE = e4m3_table()
_POS = _TABLE[:0x7F]                                            # codes 0x00..0x7E: 0 .. 448, strictly increasing


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    """Own copy of the widening (the oracle imports nothing from the product package)."""
    u = np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << 16
    return u.view(np.float32).astype(np.float64)


def f64_to_bf16_bits_exact(x: np.ndarray) -> np.ndarray:
    """float64 values that ARE bf16 numbers -> their bit patterns (asserts exactness)."""
    f = np.ascontiguousarray(x, dtype=np.float64).astype(np.float32)
    assert np.array_equal(f.astype(np.float64), x), "value is not a float32 number"
    u = f.view(np.uint32)
    assert not (u & 0xFFFF).any(), "value is not a bf16 number"
    return (u >> 16).astype(np.uint16)


def scale_exponent(amax: np.ndarray) -> np.ndarray:
    """e = smallest integer with 448 * 2^e >= amax, clamped to [E_MIN, E_MAX]; amax = 0 -> E_MIN.
    Integer arithmetic on the binary representation: amax = f * 2^k, f in [0.5, 1); 448 = 0.875 * 2^9, so
    amax / 448 = (f / 0.875) * 2^(k - 9):  f <= 0.875 -> e = k - 9, else e = k - 8."""
    amax = np.asarray(amax, dtype=np.float64)
    f, k = np.frexp(amax)
    e = np.where(f <= 0.875, k - 9, k - 8)
    e = np.where(amax == 0.0, E_MIN, e)
    return np.clip(e, E_MIN, E_MAX).astype(np.int32)


def encode_e4m3(y: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even onto the e4m3 grid, saturating at +-448.  y: float64, finite."""
    y = np.asarray(y, dtype=np.float64)
    a = np.minimum(np.abs(y), E4M3_MAX)
    hi = np.searchsorted(_POS, a, side="left")                  # first code with value >= a
    hi = np.minimum(hi, len(_POS) - 1)
    lo = np.maximum(hi - 1, 0)
    d_hi = _POS[hi] - a
    d_lo = a - _POS[lo]
    take_lo = (d_lo < d_hi) | ((d_lo == d_hi) & ((lo & 1) == 0))    # tie -> even code (even mantissa)
    code = np.where(take_lo, lo, hi).astype(np.uint8)
    code = np.where(_POS[hi] == a, hi, code).astype(np.uint8)   # exact hits
    return (code | np.where(np.signbit(y), 0x80, 0).astype(np.uint8)).astype(np.uint8)


def quantize_rows(x: np.ndarray):
    """x: float64 [..., D] (finite).  Returns (codes uint8 [..., D], e int32 [...]): one power-of-two scale per row."""
    x = np.asarray(x, dtype=np.float64)
    e = scale_exponent(np.abs(x).max(axis=-1))
    y = x * np.exp2(-e.astype(np.float64))[..., None]           # exact: a power-of-two factor
    return encode_e4m3(y), e


def dequantize(codes: np.ndarray, e: np.ndarray) -> np.ndarray:
    """Exactly code_value * 2^e (float64)."""
    return _TABLE[np.asarray(codes, dtype=np.uint8)] * np.exp2(np.asarray(e, dtype=np.float64))[..., None]


def scale_to_exponent(scale_f32: np.ndarray) -> np.ndarray:
    """The stored fp32 scale 2^e -> e (asserts it is a power of two in range)."""
    f, k = np.frexp(np.asarray(scale_f32, dtype=np.float64))
    assert np.all(f == 0.5), "scale is not a power of two"
    e = (k - 1).astype(np.int32)
    assert np.all((e >= E_MIN) & (e <= E_MAX))
    return e


def kv_append_fp8(k_new_bits, v_new_bits, codes, scales, q_len, ctx_off, block_tables):
    """H2 on fp8 pages, in place.  k_new / v_new: uint16 bf16 bit patterns [T, Hkv, D];
    codes: uint8 [num_blocks, 2, Hkv, B, D]; scales: float32 [num_blocks, 2, Hkv, B] (2^e).
    Token at absolute position p of request j goes to page bt_j[p // B], slot p % B."""
    B = codes.shape[3]
    new = (bf16_bits_to_f64(k_new_bits), bf16_bits_to_f64(v_new_bits))
    tok = 0
    for j in range(len(q_len)):
        for i in range(int(q_len[j])):
            p = int(ctx_off[j]) + i
            page, slot = int(block_tables[j][p // B]), p % B
            for kv in (0, 1):
                c, e = quantize_rows(new[kv][tok])               # [Hkv, D], [Hkv]
                codes[page, kv, :, slot, :] = c
                scales[page, kv, :, slot] = np.exp2(e.astype(np.float64)).astype(np.float32)
            tok += 1


def pages_as_bf16_bits(codes, scales, keys_per_page=None, chunk: int = 1024) -> np.ndarray:
    """The values the fp8 pages hold, as bf16 bit patterns [n, 2, Hkv, B, D] (exact; for the attention oracle).
    Slots that hold no key (keys_per_page[i] <= slot) may carry any scale bits: they are returned as zeros.
    (Converted `chunk` pages at a time: the float64 intermediate of a 40 GiB-pool batch would not fit the host.)"""
    codes = np.asarray(codes, dtype=np.uint8)
    scales = np.asarray(scales, dtype=np.float32)
    out = np.empty(codes.shape, dtype=np.uint16)
    for s0 in range(0, codes.shape[0], chunk):
        c = codes[s0:s0 + chunk]
        sc = scales[s0:s0 + chunk].astype(np.float64)
        if keys_per_page is not None:
            is_key = np.arange(c.shape[3])[None, :] < np.asarray(keys_per_page[s0:s0 + chunk])[:, None]      # [n, B]
            sc = np.where(is_key[:, None, None, :], sc, 1.0)
            c = np.where(is_key[:, None, None, :, None], c, 0).astype(np.uint8)
        out[s0:s0 + chunk] = f64_to_bf16_bits_exact(_TABLE[c] * sc[..., None])
    return out
