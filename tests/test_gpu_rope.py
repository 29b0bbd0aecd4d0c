"""-m gpu parity of the rotary-embedding step (cp_enable_rope / cp_attention_step_rope,
SURVEY.md 8(f) N2) against oracle/rope.py + the fp64 attention oracle, through the C ABI.

Pages: the K half is compared code by code with the oracle's bf16 decision (same precision on both
sides, R12); the only admissible difference is the last place of a double-precision cos / sin
(CUDA's and the host libm's differ by <= 1 ulp of fp64), which can move a bf16 code by one step for about
one element in 10^7 -- so: <= 1 bf16 step everywhere and bit-equal on >= 99.999 %.  V and everything
outside the appended rows: bit-identical.  Outputs: north_star's 2e-2 / 2e-3.
"""
import numpy as np
import pytest

from oracle import attention as ora
from oracle import rope as orope
from paper_2606_09061_b200 import binding, workloads as wl
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu


def _inv_freq(D, theta=10000.0):
    return theta ** (-np.arange(0, D, 2, dtype=np.float64) / D)


def _oracle(spec, hv, w, rows=None):
    pos = orope.token_positions(spec.q_len, spec.ctx_off)
    cache = hv.cache.copy()
    tabs = spec.compact_tables()
    ora.kv_append(orope.rope_bf16(hv.k_new, pos, w), hv.v_new, cache, spec.q_len, spec.ctx_off, tabs)
    out = ora.attention(orope.rope_bf16(hv.q, pos, w), cache, spec.q_len, spec.ctx_off, tabs, spec.sm_scale, rows=rows)
    return out, cache


def _gpu(spec, hv, w, variant=0, ctx=None):
    import torch
    own = ctx is None
    ctx = ctx or gu.make_ctx(spec, variant)
    ctx.cp_enable_rope(w)
    pool = gu.torch_bf16(wl.full_pool_from_compact(spec, hv.cache))
    q, k_new, v_new = gu.torch_bf16(hv.q), gu.torch_bf16(hv.k_new), gu.torch_bf16(hv.v_new)
    out = torch.full((spec.T, spec.Hq, spec.D), float("nan"), device="cuda", dtype=torch.bfloat16)
    ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
    ctx.cp_attention_step_rope(0, q, k_new, v_new, pool, out)
    torch.cuda.synchronize()
    assert np.array_equal(gu.to_bits(q), hv.q), "q must not be modified"
    res = wl.bf16_bits_to_f64(gu.to_bits(out)).reshape(spec.T, spec.Hq, spec.D)
    pool_after = gu.to_bits(pool)
    if own:
        ctx.close()
    return res, pool_after


def _assert_page_slice(got, want, nk):
    """V: bit-exact on keys (gu.assert_pages); K: code by code on keys, tails cleared, the rest untouched."""
    gu.assert_pages(got[:, 1:2], want[:, 1:2], nk, "V pages")
    is_key = (np.arange(got.shape[3])[None, :] < nk[:, None])[:, None, :, None]          # [n, 1, B, 1]
    is_tail = (~is_key) & (nk[:, None, None, None] > 0)
    gk, wk = got[:, 0].astype(np.int32), want[:, 0].astype(np.int32)
    diff = np.where(is_key, np.abs(gk - wk), 0)
    assert diff.max() <= 1, f"K code off by {diff.max()} steps"
    assert not np.where(is_tail, gk, 0).any(), "K slots past the last key of a last page are not zero"
    other = ~(is_key | is_tail)
    assert np.array_equal(np.where(other, gk, 0), np.where(other, wk, 0)), "a K slot outside the batch's key range was modified"
    return int((diff != 0).sum())


def _assert_pages(pool_after, cache_after, spec):
    n_diff = _assert_page_slice(pool_after[spec.touched_pages()], cache_after, gu.keys_per_page(spec))
    assert n_diff <= 1e-5 * cache_after[:, 0].size + 1, f"{n_diff} K codes differ"


@pytest.mark.parametrize("variant", [0])
def test_tiny_config_with_rope(variant):
    spec = wl.config_tiny()
    hv = wl.host_values(spec)
    w = _inv_freq(spec.D)
    got, pool_after = _gpu(spec, hv, w, variant)
    want, cache_after = _oracle(spec, hv, w)
    gu.assert_close(got, want, "tiny+rope")
    _assert_pages(pool_after, cache_after, spec)
    # rotation really happened: the unrotated oracle is far away
    plain, _ = gu.run_oracle_host_values(spec, hv)
    assert np.abs(got - plain).max() > 0.1


@pytest.mark.parametrize("seed,Hq,Hkv,D,theta", [(1, 8, 2, 64, 10000.0), (2, 8, 8, 128, 500000.0),
                                                 (3, 16, 2, 128, 10000.0), (4, 32, 8, 128, 500000.0)])
def test_random_mixed_batches_with_rope(seed, Hq, Hkv, D, theta):
    spec = wl.random_spec(seed, Hq=Hq, Hkv=Hkv, D=D, n_prefill=4, n_decode=6, max_chunk=300, max_ctx=700)
    hv = wl.host_values(spec)
    w = _inv_freq(D, theta)
    got, pool_after = _gpu(spec, hv, w)
    want, cache_after = _oracle(spec, hv, w)
    gu.assert_close(got, want, spec.name)
    _assert_pages(pool_after, cache_after, spec)


def test_long_positions_and_edges_with_rope():
    # positions up to 131071: an fp32 angle would be off by 1e-2 rad there (the table is fp64)
    q_len = [1, 1, 127, 129, 16, 1, 33]
    ctx_off = [0, 131071 - 1, 0, 127, 65536 - 8, 32767, 100000]
    spec = wl.make_spec("rope_edges", 8, 2, 128, 16, 24000, q_len, ctx_off, seed=5)
    hv = wl.host_values(spec)
    w = _inv_freq(spec.D)
    got, pool_after = _gpu(spec, hv, w)
    tok, head = gu.sample_rows(spec, 64, seed=1)
    want, cache_after = _oracle(spec, hv, w, rows=(tok, head))
    d = np.abs(got[tok, head] - want)
    assert d.max() <= gu.MAX_ABS_TOL and d.mean() <= gu.MEAN_ABS_TOL
    _assert_pages(pool_after, cache_after, spec)


def test_chunked_equals_unchunked_with_rope_and_state_errors():
    """One context: a 200-token prompt in chunks of 64/64/72 (pages carried from step to step) equals
    the oracle's unchunked run; and the call-order errors of include/cp.h."""
    import torch
    L, Hq, Hkv, D, B = 200, 8, 2, 128, 16
    w = _inv_freq(D)
    whole = wl.make_spec("whole", Hq, Hkv, D, B, 64, [L], [0], seed=9)
    hv = wl.host_values(whole)
    want, _ = _oracle(whole, hv, w)
    ctx = gu.make_ctx(whole)
    pool = gu.torch_bf16(wl.full_pool_from_compact(whole, hv.cache))
    q, k_new, v_new = gu.torch_bf16(hv.q), gu.torch_bf16(hv.k_new), gu.torch_bf16(hv.v_new)
    out = torch.full((L, Hq, D), float("nan"), device="cuda", dtype=torch.bfloat16)
    ctx.cp_build_batch([64], [0], whole.block_tables)
    with pytest.raises(binding.CpError):                      # rope not enabled
        ctx.cp_attention_step_rope(0, q[:64], k_new[:64], v_new[:64], pool, out[:64])
    ctx.cp_enable_rope(w)
    with pytest.raises(binding.CpError):                      # batch built before cp_enable_rope
        ctx.cp_attention_step_rope(0, q[:64], k_new[:64], v_new[:64], pool, out[:64])
    off = 0
    for n in (64, 64, 72):
        ctx.cp_build_batch([n], [off], whole.block_tables)
        with pytest.raises(binding.CpError):                  # k_new must be given
            ctx.cp_attention_step_rope(0, q[off:off + n], None, None, pool, out[off:off + n])
        ctx.cp_attention_step_rope(0, q[off:off + n], k_new[off:off + n], v_new[off:off + n], pool, out[off:off + n])
        off += n
    torch.cuda.synchronize()
    got = wl.bf16_bits_to_f64(gu.to_bits(out)).reshape(L, Hq, D)
    gu.assert_close(got, want, "chunked+rope")
    with pytest.raises(binding.CpError):
        ctx.cp_enable_rope(np.full(D // 2, np.nan))
    with pytest.raises(ValueError):
        ctx.cp_enable_rope(np.ones(3))
    ctx.close()


def test_b2048_with_rope_all_rows():
    """BASELINE.json configs[2] in the launch configuration bench.py --rope times: all 65,536 (token, head) rows."""
    import torch
    spec = wl.config_b2048()
    q, k_new, v_new, pool, compact = wl.device_values(spec, "cuda")
    w = _inv_freq(spec.D)
    ctx = gu.make_ctx(spec)
    ctx.cp_enable_rope(w)
    out = torch.full((spec.T, spec.Hq, spec.D), float("nan"), device="cuda", dtype=torch.bfloat16)
    ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
    ctx.cp_attention_step_rope(0, q, k_new, v_new, pool, out)
    torch.cuda.synchronize()
    hv = wl.HostValues(gu.to_bits(q), gu.to_bits(k_new), gu.to_bits(v_new), gu.to_bits(compact))
    want, cache_after = _oracle(spec, hv, w)
    got = wl.bf16_bits_to_f64(gu.to_bits(out)).reshape(spec.T, spec.Hq, spec.D)
    d = np.abs(got - want)
    assert np.isfinite(got).all() and d.max() <= gu.MAX_ABS_TOL and d.mean() <= gu.MEAN_ABS_TOL
    touched = torch.from_numpy(spec.touched_pages().astype(np.int64)).to("cuda")
    n_diff = 0
    nk = gu.keys_per_page(spec)
    for s in range(0, len(touched), 8192):
        n_diff += _assert_page_slice(gu.to_bits(pool[touched[s:s + 8192]]), cache_after[s:s + 8192], nk[s:s + 8192])
    assert n_diff <= 1e-5 * spec.T * spec.Hkv * spec.D + 2
    ctx.close()
