"""Rotary position embedding of the rows entering the attention step (TEST INFRASTRUCTURE,
not product code; imports nothing from paper_2606_09061_b200).

Where it comes from: PAPER.md is silent on positional encoding (the execution backend is
left untouched); SURVEY.md 8(f) N2 names "fused append + RoPE in the
step's producer" as the next widening of the hot path.  The definition restated here is the
textbook rotary embedding in the rotate-half pairing of the Llama-shaped configs
(reading R11): for a row x of D elements at absolute position p (= ctx_off + i
for row i of a chunk) and frequencies w_i, i in [0, D/2),

    x'[i]       = x[i] cos(p w_i) - x[i + D/2] sin(p w_i)
    x'[i + D/2] = x[i + D/2] cos(p w_i) + x[i] sin(p w_i)

applied to every head of Q and of the new K rows; V is not rotated.  The frequencies are an
INPUT (a float64 array of D/2 values); `default_inv_freq` is the usual w_i = theta^(-2i/D).

Two functions:
  rope_f64   the definition, float64 in / float64 out.
  rope_bf16  the bf16 codes that are stored in the pages / fed to the tensor cores.  Rounding
             to bf16 is a quantisation decision, so it is taken in the kernel's precision
             (R12): cos/sin evaluated in float64 and rounded to float32, the two
             products and the sum each rounded to float32 (no fused multiply-add), then
             round-to-nearest-even to bf16.

Pins (tests/test_oracle_rope.py): printed closed forms for D = 2 and D = 4 (sign and pairing
convention), the complex-multiplication form, p = 0 identity, composition, per-pair norm,
relative-position invariance of q.k, rope_bf16 within half a bf16 ulp of rope_f64.
"""
import numpy as np


def default_inv_freq(D: int, theta: float = 10000.0) -> np.ndarray:
    """w_i = theta^(-2i/D), i = 0 .. D/2 - 1, float64."""
    i = np.arange(D // 2, dtype=np.float64)
    return np.power(np.float64(theta), -2.0 * i / np.float64(D))


def token_positions(q_len, ctx_off) -> np.ndarray:
    """Absolute position of every token of the batch, descriptor order (int64 [T])."""
    pos = [int(o) + np.arange(int(n), dtype=np.int64) for n, o in zip(q_len, ctx_off)]
    return np.concatenate(pos) if pos else np.zeros(0, dtype=np.int64)


def rope_f64(x: np.ndarray, pos: np.ndarray, inv_freq: np.ndarray) -> np.ndarray:
    """x float64 [T, H, D], pos [T], inv_freq float64 [D/2] -> float64 [T, H, D]."""
    x = np.asarray(x, dtype=np.float64)
    T, H, D = x.shape
    h = D // 2
    ang = np.asarray(pos, dtype=np.float64)[:, None] * np.asarray(inv_freq, dtype=np.float64)[None, :]
    c = np.cos(ang)[:, None, :]
    s = np.sin(ang)[:, None, :]
    lo, hi = x[..., :h], x[..., h:]
    out = np.empty_like(x)
    out[..., :h] = lo * c - hi * s
    out[..., h:] = hi * c + lo * s
    return out


def _bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << 16).view(np.float32)


def _f32_to_bf16_bits_rne(x: np.ndarray) -> np.ndarray:
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    return ((u + (((u >> 16) & 1) + np.uint32(0x7FFF))) >> 16).astype(np.uint16)


def rope_bf16(x_bits: np.ndarray, pos: np.ndarray, inv_freq: np.ndarray) -> np.ndarray:
    """x_bits uint16 (bf16) [T, H, D] -> uint16 (bf16) [T, H, D]; float32 arithmetic as in the header."""
    x = _bf16_bits_to_f32(x_bits)
    T, H, D = x.shape
    h = D // 2
    ang = np.asarray(pos, dtype=np.float64)[:, None] * np.asarray(inv_freq, dtype=np.float64)[None, :]
    c = np.cos(ang).astype(np.float32)[:, None, :]
    s = np.sin(ang).astype(np.float32)[:, None, :]
    lo, hi = x[..., :h], x[..., h:]
    out = np.empty_like(x)
    # numpy float32 ufuncs round after every operation: product, product, then sum
    out[..., :h] = (lo * c) - (hi * s)
    out[..., h:] = (hi * c) + (lo * s)
    return _f32_to_bf16_bits_rne(out)
