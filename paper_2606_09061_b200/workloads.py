"""Seeded synthetic inputs shaped like the paper's mixed short/long workloads.

This module holds NONE of the method's arithmetic (no attention, no scheduling):
it only draws shapes, page assignments and values, so both the CUDA path (via the
binding) and the tests' oracle may be fed from it (task rule (3)).  numpy only at
import time; torch is imported lazily by the device helpers.

Recipe: numpy.random.default_rng(seed)
(PCG64), draws in this order: request shapes -> page assignment -> values.  The
paper measures on ShareGPT replays that are not available
here; these configs (BASELINE.json "configs") stand in for them and keep their
structure: decode-first mixed batches with heavy-tailed lengths.
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional

import numpy as np

POISON_BF16 = 0x7F7F          # +3.39e38, largest finite bf16: stale data in tails
POISON_BF16_NEG = 0xFF7F      # -3.39e38
NAN_BF16 = 0x7FC0


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit pattern, round-to-nearest-even (data conversion only)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + r) >> 16).astype(np.uint16)


def bf16_bits_to_f64(b: np.ndarray) -> np.ndarray:
    u = np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << 16
    return u.view(np.float32).astype(np.float64)


@dataclasses.dataclass
class BatchSpec:
    """Structure of one iteration: who is in the batch and where their pages are."""
    name: str
    Hq: int
    Hkv: int
    D: int
    B: int
    num_blocks: int                 # pages in the (single-layer) pool
    q_len: np.ndarray               # int32 [n]
    ctx_off: np.ndarray             # int32 [n] tokens already cached before this step
    block_tables: List[np.ndarray]  # per request: int32 pool page ids
    seed: int = 0

    @property
    def n_reqs(self) -> int:
        return len(self.q_len)

    @property
    def T(self) -> int:
        return int(self.q_len.sum())

    @property
    def sm_scale(self) -> float:
        return float(np.float32(1.0) / np.sqrt(np.float32(self.D)))

    @property
    def kv_len(self) -> np.ndarray:
        return (self.ctx_off.astype(np.int64) + self.q_len).astype(np.int64)

    def touched_pages(self) -> np.ndarray:
        return (np.concatenate(self.block_tables) if self.block_tables
                else np.zeros(0, np.int32))

    def compact_tables(self) -> List[np.ndarray]:
        """Block tables re-expressed as indices into touched_pages() order."""
        out, base = [], 0
        for bt in self.block_tables:
            out.append(np.arange(base, base + len(bt), dtype=np.int32))
            base += len(bt)
        return out

    # ---- algorithmic work (SURVEY.md 8(d) formulas; counting, not the method) ----
    def causal_pairs(self) -> int:
        q = self.q_len.astype(np.int64)
        off = self.ctx_off.astype(np.int64)
        return int((q * off + q * (q + 1) // 2).sum())

    def flops(self) -> int:
        return 4 * self.D * self.Hq * self.causal_pairs()

    def algorithmic_bytes(self, kv_dtype: str = "bf16") -> int:
        # fp8 pages: one byte per element + one fp32 scale per (token, KV head, K|V) row
        row = self.D * 2 if kv_dtype == "bf16" else self.D + 4
        kv = int(2 * self.kv_len.sum() * self.Hkv * row)
        qo = 2 * self.T * self.Hq * self.D * 2
        tables = 4 * int(sum(len(b) for b in self.block_tables))
        return kv + qo + tables


def _assign_pages(rng, q_len, ctx_off, B, num_blocks, interleave=True):
    need = [int((int(c) + int(q) + B - 1) // B) for q, c in zip(q_len, ctx_off)]
    total = sum(need)
    if total > num_blocks:
        raise ValueError(f"pool too small: need {total} pages, have {num_blocks}")
    if num_blocks <= 4 * total or num_blocks < (1 << 16):
        ids = rng.permutation(num_blocks)[:total]
    else:  # large pool: sample without replacement without a full permutation
        ids = rng.choice(num_blocks, size=total, replace=False)
    ids = ids.astype(np.int32)
    if not interleave:
        ids = np.sort(ids)
    out, base = [], 0
    for n in need:
        out.append(np.ascontiguousarray(ids[base:base + n]))
        base += n
    return out


def make_spec(name: str, Hq: int, Hkv: int, D: int, B: int, num_blocks: int,
              q_len, ctx_off, seed: int = 0, rng=None) -> BatchSpec:
    rng = np.random.default_rng(seed) if rng is None else rng
    q_len = np.asarray(q_len, dtype=np.int32)
    ctx_off = np.asarray(ctx_off, dtype=np.int32)
    bts = _assign_pages(rng, q_len, ctx_off, B, num_blocks)
    return BatchSpec(name, Hq, Hkv, D, B, num_blocks, q_len, ctx_off, bts, seed)


# ----------------------------------------------------------------------------
# BASELINE.json configs 1-4
# ----------------------------------------------------------------------------
def config_tiny(seed: int = 0) -> BatchSpec:
    """configs[0]: 4 q heads, 1 KV head, D 64, B 16; chunks (32 @0), (16 @48);
    decodes with context 40 and 100 (the context counts the decoded token:
    q_len 1, ctx_off c-1; reading R1); 16 pages randomly permuted."""
    return make_spec("tiny", 4, 1, 64, 16, 16, [32, 16, 1, 1], [0, 48, 39, 99], seed)


def config_b512(seed: int = 0) -> BatchSpec:
    """configs[1]: 8B shape, budget 512 = 64 decodes ctx ~ U[512,4096] + chunk 448 @2048."""
    rng = np.random.default_rng(seed)
    ctx = rng.integers(512, 4097, size=64)
    q_len = [1] * 64 + [448]
    ctx_off = list(ctx - 1) + [2048]
    return make_spec("b512", 32, 8, 128, 16, 32768, q_len, ctx_off, seed, rng)


def config_b2048(seed: int = 0) -> BatchSpec:
    """configs[2] (the target): 8B shape, budget 2048 = 512 decodes with lognormal
    context (median 1024, sigma 1.0, cap 32768) + 4 chunks of 384 at offsets
    0, 4096, 16384, 30720; pages scattered over a 40 GiB single-layer pool."""
    rng = np.random.default_rng(seed)
    ctx = np.rint(np.exp(np.log(1024.0) + rng.standard_normal(512)))
    ctx = np.clip(ctx, 1, 32768).astype(np.int64)
    q_len = [1] * 512 + [384] * 4
    ctx_off = list(ctx - 1) + [0, 4096, 16384, 30720]
    return make_spec("b2048", 32, 8, 128, 16, 655360, q_len, ctx_off, seed, rng)


def config_70b(seed: int = 0) -> BatchSpec:
    """configs[3]: 64 q heads, 8 KV heads, D 128; budget 8192 = 256 decodes ctx ~
    U[1024,16384] + one chunk of 7936 tokens at offset 122880."""
    rng = np.random.default_rng(seed)
    ctx = rng.integers(1024, 16385, size=256)
    q_len = [1] * 256 + [7936]
    ctx_off = list(ctx - 1) + [122880]
    return make_spec("70b", 64, 8, 128, 16, 262144, q_len, ctx_off, seed, rng)


def _subset(spec: BatchSpec, keep, name: str) -> BatchSpec:
    idx = [j for j in range(spec.n_reqs) if keep(spec.q_len[j])]
    return BatchSpec(name, spec.Hq, spec.Hkv, spec.D, spec.B, spec.num_blocks, spec.q_len[idx],
                     spec.ctx_off[idx], [spec.block_tables[j] for j in idx], spec.seed)


def config_b2048_decodes(seed: int = 0) -> BatchSpec:
    """The 512 decodes of configs[2] alone (profiling breakdown: the HBM-bound part)."""
    return _subset(config_b2048(seed), lambda q: q == 1, "b2048dec")


def config_b2048_prefill(seed: int = 0) -> BatchSpec:
    """The 4 prefill chunks of configs[2] alone (profiling breakdown: the tensor-bound part)."""
    return _subset(config_b2048(seed), lambda q: q > 1, "b2048pf")


def config_small_decode(seed: int = 0) -> BatchSpec:
    """A decode-only round as the trace run sees most of the time: 12 long-context decodes
    (context uniform in [8192, 32768]), 8B shape.  Load balance needs the key ranges split."""
    rng = np.random.default_rng(seed)
    ctx = rng.integers(8192, 32769, size=12)
    return make_spec("dec12", 32, 8, 128, 16, 65536, [1] * 12, list(ctx - 1), seed, rng)


CONFIGS = {"tiny": config_tiny, "b512": config_b512, "b2048": config_b2048,
           "70b": config_70b, "b2048dec": config_b2048_decodes, "b2048pf": config_b2048_prefill, "dec12": config_small_decode}


def random_spec(seed: int, Hq=8, Hkv=2, D=64, B=16, n_prefill=3, n_decode=5,
                max_chunk=200, max_ctx=600, slack_pages=8) -> BatchSpec:
    """Small random mixed batch for parity sweeps (ragged chunks, odd offsets)."""
    rng = np.random.default_rng(seed)
    q_len, ctx_off = [], []
    for _ in range(n_decode):
        q_len.append(1)
        ctx_off.append(int(rng.integers(0, max_ctx)))
    for _ in range(n_prefill):
        q_len.append(int(rng.integers(1, max_chunk + 1)))
        ctx_off.append(int(rng.integers(0, max_ctx)) if rng.random() < 0.7 else 0)
    order = rng.permutation(len(q_len))
    q_len = np.asarray(q_len)[order]
    ctx_off = np.asarray(ctx_off)[order]
    need = int(((q_len + ctx_off + B - 1) // B).sum())
    return make_spec(f"rand{seed}", Hq, Hkv, D, B, need + slack_pages, q_len,
                     ctx_off, seed, rng)


# ----------------------------------------------------------------------------
# Values
# ----------------------------------------------------------------------------
@dataclasses.dataclass
class HostValues:
    """bf16 bit patterns on the host.  `cache` is COMPACT: page i of `cache` is pool
    page spec.touched_pages()[i]; use spec.compact_tables() to index it."""
    q: np.ndarray        # uint16 [T, Hq, D]
    k_new: np.ndarray    # uint16 [T, Hkv, D]
    v_new: np.ndarray    # uint16 [T, Hkv, D]
    cache: np.ndarray    # uint16 [n_touched, 2, Hkv, B, D], state BEFORE this step


def _poison_unwritten(cache: np.ndarray, spec: BatchSpec, poison: int) -> None:
    """Slots at positions >= ctx_off hold stale data before the step (alternating
    +-poison so that sums of garbage do not cancel by luck)."""
    base = 0
    B = spec.B
    for bt, off in zip(spec.block_tables, spec.ctx_off):
        off = int(off)
        first = off // B
        for pi in range(first, len(bt)):
            lo = off - pi * B if pi == first else 0
            val = poison if (pi & 1) == 0 else (poison ^ 0x8000)
            cache[base + pi, :, :, lo:, :] = val
        base += len(bt)


def host_values(spec: BatchSpec, seed: Optional[int] = None,
                poison: int = POISON_BF16) -> HostValues:
    """N(0,1) values rounded RN to bf16 (BASELINE.json configs), numpy only."""
    rng = np.random.default_rng((spec.seed if seed is None else seed) + 0x5EED)
    T, Hq, Hkv, D, B = spec.T, spec.Hq, spec.Hkv, spec.D, spec.B
    q = f32_to_bf16_bits(rng.standard_normal((T, Hq, D), dtype=np.float32))
    k_new = f32_to_bf16_bits(rng.standard_normal((T, Hkv, D), dtype=np.float32))
    v_new = f32_to_bf16_bits(rng.standard_normal((T, Hkv, D), dtype=np.float32))
    n_touched = int(sum(len(b) for b in spec.block_tables))
    cache = f32_to_bf16_bits(
        rng.standard_normal((n_touched, 2, Hkv, B, D), dtype=np.float32))
    _poison_unwritten(cache, spec, poison)
    return HostValues(q, k_new, v_new, cache)


def full_pool_from_compact(spec: BatchSpec, cache: np.ndarray,
                           poison: int = POISON_BF16) -> np.ndarray:
    """Host pool [num_blocks, 2, Hkv, B, D] with untouched pages poisoned (small
    configs only)."""
    pool = np.full((spec.num_blocks, 2, spec.Hkv, spec.B, spec.D), poison,
                   dtype=np.uint16)
    pool[1::2] ^= 0x8000
    pool[spec.touched_pages()] = cache
    return pool


def device_values(spec: BatchSpec, device, seed: Optional[int] = None,
                  poison: int = POISON_BF16, pool=None):
    """Generate values ON THE GPU with a seeded torch generator (large configs).

    Returns (q, k_new, v_new, pool, compact) torch tensors: q/k_new/v_new bf16,
    pool bf16 [num_blocks, 2, Hkv, B, D] with the touched pages filled and their
    unwritten slots poisoned, compact = the touched pages in table order (a copy
    taken BEFORE the step, what the oracle starts from).  Untouched pool pages are
    poisoned only when `pool` is created here and num_blocks is small; a caller-
    provided pool is reused as is (its untouched pages keep whatever they hold).
    """
    import torch
    g = torch.Generator(device=device)
    g.manual_seed((spec.seed if seed is None else seed) + 0x5EED)
    T, Hq, Hkv, D, B = spec.T, spec.Hq, spec.Hkv, spec.D, spec.B
    q = torch.randn((T, Hq, D), generator=g, device=device, dtype=torch.float32).bfloat16()
    k_new = torch.randn((T, Hkv, D), generator=g, device=device, dtype=torch.float32).bfloat16()
    v_new = torch.randn((T, Hkv, D), generator=g, device=device, dtype=torch.float32).bfloat16()
    touched = torch.from_numpy(spec.touched_pages().astype(np.int64)).to(device)
    n_touched = int(touched.numel())
    compact = torch.empty((n_touched, 2, Hkv, B, D), device=device, dtype=torch.bfloat16)
    step = max(1, (1 << 28) // (2 * Hkv * B * D))      # <= 1 GiB of fp32 at a time
    for s in range(0, n_touched, step):
        e = min(n_touched, s + step)
        compact[s:e] = torch.randn((e - s, 2, Hkv, B, D), generator=g, device=device,
                                   dtype=torch.float32).bfloat16()
    # poison the not-yet-written slots (positions >= ctx_off) of each request
    cu16 = compact.view(torch.int16)
    pv = poison - 0x10000 if poison >= 0x8000 else poison
    base = 0
    for bt, off in zip(spec.block_tables, spec.ctx_off):
        off = int(off)
        first = off // B
        if first < len(bt):
            cu16[base + first, :, :, off - first * B:, :] = pv
            if first + 1 < len(bt):
                cu16[base + first + 1:base + len(bt)] = pv
        base += len(bt)
    if pool is None:
        pool = torch.empty((spec.num_blocks, 2, Hkv, B, D), device=device,
                           dtype=torch.bfloat16)
        if spec.num_blocks <= (1 << 16):
            pool.view(torch.int16).fill_(pv)
    pool[touched] = compact
    return q, k_new, v_new, pool, compact


def device_values_fp8(spec: BatchSpec, device, seed: Optional[int] = None):
    """FP8 (e4m3) pool for the large configs, generated ON THE GPU with a seeded torch generator: q / k_new / v_new
    bf16 N(0,1) as in device_values; the touched pages hold uniformly random finite e4m3 codes with the row scale
    2^-7 (|value| <= 3.5); slots at positions >= ctx_off and every untouched page hold NaN codes (0x7F) / whatever
    torch.empty left.  Returns (q, k_new, v_new, codes_pool u8 [num_blocks,2,Hkv,B,D], scales_pool f32
    [num_blocks,2,Hkv,B], compact_codes, compact_scales) -- the compact copies are the state BEFORE the step."""
    import torch
    g = torch.Generator(device=device)
    g.manual_seed((spec.seed if seed is None else seed) + 0xF8)
    T, Hq, Hkv, D, B = spec.T, spec.Hq, spec.Hkv, spec.D, spec.B
    q = torch.randn((T, Hq, D), generator=g, device=device, dtype=torch.float32).bfloat16()
    k_new = torch.randn((T, Hkv, D), generator=g, device=device, dtype=torch.float32).bfloat16()
    v_new = torch.randn((T, Hkv, D), generator=g, device=device, dtype=torch.float32).bfloat16()
    touched = torch.from_numpy(spec.touched_pages().astype(np.int64)).to(device)
    n_touched = int(touched.numel())
    mag = torch.randint(0, 0x7F, (n_touched, 2, Hkv, B, D), generator=g, device=device, dtype=torch.int16)
    sign = torch.randint(0, 2, (n_touched, 2, Hkv, B, D), generator=g, device=device, dtype=torch.int16)
    compact_codes = (mag | (sign << 7)).to(torch.uint8)
    del mag, sign
    compact_scales = torch.full((n_touched, 2, Hkv, B), 2.0 ** -7, device=device, dtype=torch.float32)
    base = 0
    for bt, off in zip(spec.block_tables, spec.ctx_off):
        off = int(off)
        first = off // B
        if first < len(bt):
            compact_codes[base + first, :, :, off - first * B:, :] = 0x7F
            compact_scales[base + first, :, :, off - first * B:] = float("nan")
            if first + 1 < len(bt):
                compact_codes[base + first + 1:base + len(bt)] = 0x7F
                compact_scales[base + first + 1:base + len(bt)] = float("nan")
        base += len(bt)
    codes = torch.empty((spec.num_blocks, 2, Hkv, B, D), device=device, dtype=torch.uint8)
    scales = torch.empty((spec.num_blocks, 2, Hkv, B), device=device, dtype=torch.float32)
    codes[touched] = compact_codes
    scales[touched] = compact_scales
    return q, k_new, v_new, codes, scales, compact_codes, compact_scales


# ----------------------------------------------------------------------------
# configs[4]: request trace for the scheduler-driven run
# ----------------------------------------------------------------------------
def make_trace(n_requests: int = 1000, rate_per_s: float = 8.0, seed: int = 0,
               short_median: float = 256.0, short_sigma: float = 1.0, long_lo: int = 8192,
               long_hi: int = 32768, p_long: float = 0.3, out_median: float = 128.0,
               out_sigma: float = 1.0, out_max: int = 4096):
    """Poisson arrivals; prompt lengths 70% lognormal(median 256) clipped to [1, 8191]
    + 30% uniform[8192, 32768]; output lengths lognormal(median 128) clipped to
    [1, out_max] (BASELINE.json configs[4]; sigma = 1.0 is our reading, R7).
    Returns int64 arrays (req_id, arrival_us, prompt_len, output_len)."""
    rng = np.random.default_rng(seed)
    gaps = rng.exponential(1.0 / rate_per_s, size=n_requests)
    arrival_us = np.floor(np.cumsum(gaps) * 1e6).astype(np.int64)
    is_long = rng.random(n_requests) < p_long
    short = np.clip(np.rint(np.exp(np.log(short_median) + short_sigma * rng.standard_normal(n_requests))),
                    1, long_lo - 1)
    longp = rng.integers(long_lo, long_hi + 1, size=n_requests)
    prompt = np.where(is_long, longp, short).astype(np.int64)
    out = np.clip(np.rint(np.exp(np.log(out_median) + out_sigma * rng.standard_normal(n_requests))),
                  1, out_max).astype(np.int64)
    return np.arange(n_requests, dtype=np.int64), arrival_us, prompt, out


def make_apc_trace(n_requests: int = 1000, seed: int = 0, mean_gap_us: float = 2000.0):
    """The APC-ablation shape: 49:1 short (30-50) : long (200-220) prompts,
    bursty arrivals."""
    rng = np.random.default_rng(seed)
    is_long = (np.arange(n_requests) % 50) == 49
    prompt = np.where(is_long, rng.integers(200, 221, n_requests), rng.integers(30, 51, n_requests))
    burst = rng.random(n_requests) < 0.3
    gaps = np.where(burst, 0.0, rng.exponential(mean_gap_us / 0.7, n_requests))
    arrival_us = np.floor(np.cumsum(gaps)).astype(np.int64)
    out = rng.integers(8, 65, n_requests)
    return np.arange(n_requests, dtype=np.int64), arrival_us, prompt.astype(np.int64), out.astype(np.int64)


def make_sharegpt_like_trace(n_requests: int = 200, gap_us: float = 100000.0, seed: int = 0, prompt_median: float = 19.0,
                             prompt_p90: float = 179.0, max_ctx: int = 512, max_gen: int = 512, out_median: float = 128.0,
                             out_sigma: float = 1.0):
    """The paper's short-context serving mix, as a synthetic stand-in (ShareGPT itself is not available here):
    200 requests at a FIXED inter-arrival of 0.1 s, prompt lengths with median 19 and P90 179 tokens, context clipped
    to 512, generation capped at 512.  Prompts are lognormal with that median and P90 (sigma =
    ln(179 / 19) / 1.2816), clipped to [1, max_ctx - 1]; the paper does not print the output-length distribution:
    lognormal(median 128, sigma 1) clipped to [1, min(max_gen, max_ctx - prompt)] is our reading.  `gap_us` below the
    iteration time gives the compressed variant (the queue has depth: many tiny chunks per round)."""
    rng = np.random.default_rng(seed)
    sigma = float(np.log(prompt_p90 / prompt_median) / 1.2815515655446004)
    prompt = np.clip(np.rint(np.exp(np.log(prompt_median) + sigma * rng.standard_normal(n_requests))), 1, max_ctx - 1).astype(np.int64)
    out = np.rint(np.exp(np.log(out_median) + out_sigma * rng.standard_normal(n_requests)))
    out = np.clip(out, 1, np.minimum(max_gen, max_ctx - prompt)).astype(np.int64)
    arrival_us = np.floor(np.arange(n_requests) * gap_us).astype(np.int64)
    return np.arange(n_requests, dtype=np.int64), arrival_us, prompt, out
