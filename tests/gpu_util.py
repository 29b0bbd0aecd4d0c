"""Helpers for the -m gpu parity tests: run the same seeded inputs through libcp (via the
C ABI binding) and through the fp64 oracle, and compare element by element."""
import numpy as np

from oracle import attention as ora
from paper_2606_09061_b200 import binding, build, workloads as wl

MAX_ABS_TOL = 2e-2      # BASELINE.json north_star: max-abs error on bf16 outputs
MEAN_ABS_TOL = 2e-3     # BASELINE.json north_star: mean-abs error


def torch_bf16(bits: np.ndarray, device="cuda"):
    import torch
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(device).view(torch.bfloat16)


def to_bits(t) -> np.ndarray:
    import torch
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def make_ctx(spec, variant=0, **kw):
    build.build()
    args = dict(num_q_heads=spec.Hq, num_kv_heads=spec.Hkv, head_dim=spec.D,
                num_blocks=spec.num_blocks, block_size=spec.B, sm_scale=spec.sm_scale,
                max_tokens=max(spec.T, 1), max_reqs=max(spec.n_reqs, 1),
                max_total_pages=max(int(sum(len(b) for b in spec.block_tables)), 1),
                kernel_variant=variant)
    args.update(kw)
    return binding.Context(**args)


def run_gpu_host_values(spec, hv, variant=0, append=True, ctx=None, poison=wl.POISON_BF16):
    """Small configs: host values -> full pool on the device -> one step.  Returns
    (out float64 [T,Hq,D], pool bits after the step)."""
    import torch
    own = ctx is None
    ctx = ctx or make_ctx(spec, variant)
    pool_np = wl.full_pool_from_compact(spec, hv.cache, poison)
    if not append:   # caller writes the pages itself: do it with the oracle's append on the host copy
        compact = hv.cache.copy()
        ora.kv_append(hv.k_new, hv.v_new, compact, spec.q_len, spec.ctx_off, spec.compact_tables())
        pool_np[spec.touched_pages()] = compact
    pool = torch_bf16(pool_np)
    q = torch_bf16(hv.q)
    k_new = torch_bf16(hv.k_new) if append else None
    v_new = torch_bf16(hv.v_new) if append else None
    out = torch.full((spec.T, spec.Hq, spec.D), float("nan"), device="cuda", dtype=torch.bfloat16)
    ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
    ctx.cp_attention_step(0, q, k_new, v_new, pool, out)
    torch.cuda.synchronize()
    res = wl.bf16_bits_to_f64(to_bits(out)).reshape(spec.T, spec.Hq, spec.D)
    pool_after = to_bits(pool)
    if own:
        ctx.close()
    return res, pool_after


def run_oracle_host_values(spec, hv, rows=None):
    cache = hv.cache.copy()
    tabs = spec.compact_tables()
    ora.kv_append(hv.k_new, hv.v_new, cache, spec.q_len, spec.ctx_off, tabs)
    return ora.attention(hv.q, cache, spec.q_len, spec.ctx_off, tabs, spec.sm_scale, rows=rows), cache


def assert_close(got, want, what=""):
    assert np.isfinite(got).all(), f"{what}: non-finite output"
    d = np.abs(got - want)
    assert d.max() <= MAX_ABS_TOL, f"{what}: max-abs {d.max():.4g} > {MAX_ABS_TOL}"
    assert d.mean() <= MEAN_ABS_TOL, f"{what}: mean-abs {d.mean():.4g} > {MEAN_ABS_TOL}"
    return float(d.max()), float(d.mean())


def sample_rows(spec, n, seed=0):
    """Seeded (token, head) sample that always includes each request's first and last row."""
    rng = np.random.default_rng(seed)
    cu = np.concatenate([[0], np.cumsum(spec.q_len)])
    tok = [cu[j] for j in range(spec.n_reqs)] + [cu[j + 1] - 1 for j in range(spec.n_reqs)]
    tok = np.asarray(tok, dtype=np.int64)
    if len(tok) > n // 2:
        tok = rng.choice(tok, size=n // 2, replace=False)
    extra = rng.integers(0, spec.T, size=n - len(tok))
    tok = np.concatenate([tok, extra]).astype(np.int64)
    head = rng.integers(0, spec.Hq, size=len(tok)).astype(np.int32)
    return tok, head


def keys_per_page(spec) -> np.ndarray:
    """For every page in touched_pages() order: how many of its 16 slots hold a key of its request AFTER the step."""
    out = []
    for bt, q, o in zip(spec.block_tables, spec.q_len, spec.ctx_off):
        kv_len = int(q) + int(o)
        out.append(np.clip(kv_len - np.arange(len(bt)) * spec.B, 0, spec.B))
    return np.concatenate(out).astype(np.int64) if out else np.zeros(0, np.int64)


def assert_pages(got, want, nk, what="pages"):
    """H2 parity on pages [n, 2, Hkv, B, D] (bit patterns): every slot that holds a key equals the oracle's append
    bit for bit; the slots of a request's last page past its last key are ZERO (the step clears them, include/cp.h:
    they hold no key); every other slot is untouched (= the oracle's copy, which never writes there)."""
    B = got.shape[3]
    slot = np.arange(B)[None, :]
    is_key = slot < nk[:, None]                                        # [n, B]
    is_tail = (~is_key) & (nk[:, None] > 0)                            # partly filled page = the request's last page
    k4 = is_key[:, None, None, :, None]
    t4 = is_tail[:, None, None, :, None]
    assert np.array_equal(np.where(k4, got, 0), np.where(k4, want, 0)), f"{what}: appended rows differ from the oracle's append"
    assert not np.where(t4, got, 0).any(), f"{what}: slots past the last key of a last page are not zero"
    o4 = ~(k4 | t4)
    assert np.array_equal(np.where(o4, got, 0), np.where(o4, want, 0)), f"{what}: a slot outside the batch's key range was modified"
