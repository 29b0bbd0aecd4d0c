"""-m gpu parity at BASELINE.json's full sizes, in the launch configuration bench.py times.
configs[1] (budget 512) and configs[2] (budget 2048, the bench workload) are compared in FULL, every
(token, head) row against the oracle; configs[3] (70B-shaped, 33 TFLOP of fp64) on a seeded sample of rows
the oracle computes one by one."""
import numpy as np
import pytest

from oracle import attention as ora
from paper_2606_09061_b200 import workloads as wl
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu


def _run_device_config(spec, variant, n_sample):
    import torch
    dev = torch.device("cuda:0")
    q, k_new, v_new, pool, compact = wl.device_values(spec, dev)
    ctx = gu.make_ctx(spec, variant)
    out = torch.full((spec.T, spec.Hq, spec.D), float("nan"), device=dev, dtype=torch.bfloat16)
    ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
    ctx.cp_attention_step(0, q, k_new, v_new, pool, out)
    torch.cuda.synchronize()
    got = wl.bf16_bits_to_f64(gu.to_bits(out)).reshape(spec.T, spec.Hq, spec.D)
    assert np.isfinite(got).all()
    # oracle: same bits, its own append, sampled rows
    cache = gu.to_bits(compact)
    tabs = spec.compact_tables()
    ora.kv_append(gu.to_bits(k_new), gu.to_bits(v_new), cache, spec.q_len, spec.ctx_off, tabs)
    # H2 parity: the pages the step wrote equal the oracle's append, bit for bit
    touched = torch.from_numpy(spec.touched_pages().astype(np.int64)).to(dev)
    step = 8192
    nk = gu.keys_per_page(spec)
    for s in range(0, len(touched), step):
        gu.assert_pages(gu.to_bits(pool[touched[s:s + step]]), cache[s:s + step], nk[s:s + step])
    if n_sample is None:
        want = ora.attention(gu.to_bits(q), cache, spec.q_len, spec.ctx_off, tabs, spec.sm_scale)
        stats = gu.assert_close(got, want, spec.name)
    else:
        tok, head = gu.sample_rows(spec, n_sample)
        want = ora.attention(gu.to_bits(q), cache, spec.q_len, spec.ctx_off, tabs, spec.sm_scale,
                             rows=(tok, head))
        stats = gu.assert_close(got[tok, head], want, spec.name)
    info = ctx.cp_get_batch_info()
    ctx.close()
    del pool, compact
    torch.cuda.empty_cache()
    return stats, info


def test_config_b512_full():
    _run_device_config(wl.config_b512(), 0, None)


def test_config_b2048_full():
    """All 65,536 (token, head) rows of the bench workload (the oracle takes ~7 s on 16 cores)."""
    stats, info = _run_device_config(wl.config_b2048(), 0, None)
    assert info.n_tokens == 2048 and info.n_reqs == 516


def test_config_70b_sampled():
    _run_device_config(wl.config_70b(), 0, 1024)


def test_config_b2048_fp8_sampled():
    """configs[2] on FP8 (e4m3) KV pages in the launch configuration `bench.py --kv-dtype e4m3` times: appended
    codes / scales bit-exact against oracle/kv_fp8.py on every touched page, outputs on a seeded sample of rows
    (first and last row of every request + random rows) against the fp64 oracle over the dequantised pages."""
    import torch
    from oracle import kv_fp8 as q8
    from paper_2606_09061_b200 import binding
    spec = wl.config_b2048()
    dev = torch.device("cuda:0")
    q, k_new, v_new, codes, scales, ccodes, cscales = wl.device_values_fp8(spec, dev)
    chunk_pages = int(sum(len(b) for b, ql in zip(spec.block_tables, spec.q_len) if ql * (spec.Hq // spec.Hkv) > 8))
    ctx = gu.make_ctx(spec, kv_dtype=binding.CP_KV_E4M3, max_scratch_pages=chunk_pages)
    out = torch.full((spec.T, spec.Hq, spec.D), float("nan"), device=dev, dtype=torch.bfloat16)
    ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
    ctx.cp_attention_step_fp8(0, q, k_new, v_new, codes, scales, out)
    torch.cuda.synchronize()
    got = wl.bf16_bits_to_f64(gu.to_bits(out)).reshape(spec.T, spec.Hq, spec.D)
    assert np.isfinite(got).all()
    want_codes, want_scales = ccodes.cpu().numpy(), cscales.cpu().numpy()
    tabs = spec.compact_tables()
    q8.kv_append_fp8(gu.to_bits(k_new), gu.to_bits(v_new), want_codes, want_scales, spec.q_len, spec.ctx_off, tabs)
    nk = gu.keys_per_page(spec)
    touched = torch.from_numpy(spec.touched_pages().astype(np.int64)).to(dev)
    slot = np.arange(spec.B)[None, :]
    for s in range(0, len(touched), 8192):
        gc, gs = codes[touched[s:s + 8192]].cpu().numpy(), scales[touched[s:s + 8192]].cpu().numpy()
        is_key = (slot < nk[s:s + 8192, None])[:, None, None, :]
        is_tail = ((slot >= nk[s:s + 8192, None]) & (nk[s:s + 8192, None] > 0))[:, None, None, :]
        assert np.array_equal(np.where(is_key[..., None], gc, 0), np.where(is_key[..., None], want_codes[s:s + 8192], 0))
        assert np.array_equal(np.where(is_key, gs, 0).view(np.uint32), np.where(is_key, want_scales[s:s + 8192], 0).view(np.uint32))
        assert not np.where(is_tail[..., None], gc, 0).any() and np.all(np.where(is_tail, gs, 1.0) == 1.0)
    pages = q8.pages_as_bf16_bits(want_codes, want_scales, nk)
    tok, head = gu.sample_rows(spec, 2048)
    want = ora.attention(gu.to_bits(q), pages, spec.q_len, spec.ctx_off, tabs, spec.sm_scale, rows=(tok, head))
    gu.assert_close(got[tok, head], want, "b2048 fp8")
    ctx.close()
