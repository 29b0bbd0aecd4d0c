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
