"""-m gpu parity of FP8 (e4m3) KV pages (cp_attention_step_fp8, SURVEY.md 8(f) N2 second half) against
oracle/kv_fp8.py + the fp64 attention oracle, through the C ABI.

Pages: codes and scales of every slot that holds a key equal the oracle's quantisation BIT FOR BIT (the decision is
integer / exact arithmetic on both sides); the unused slots of a last page are cleared (code 0, scale 1); nothing
else is written.  Outputs: north_star's 2e-2 / 2e-3 against the oracle over the DEQUANTISED pages (R15).
"""
import numpy as np
import pytest

from oracle import attention as ora
from oracle import kv_fp8 as q8
from paper_2606_09061_b200 import binding, workloads as wl
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu

NAN_CODE = 0x7F


def _initial_pool(spec, hv):
    """fp8 state BEFORE the step: keys already cached (positions < ctx_off) hold the oracle's quantisation of the
    seeded bf16 values; every other slot of every page holds NaN codes and NaN scales."""
    n = spec.num_blocks
    codes = np.full((n, 2, spec.Hkv, spec.B, spec.D), NAN_CODE, np.uint8)
    scales = np.full((n, 2, spec.Hkv, spec.B), np.nan, np.float32)
    base = 0
    for bt, off in zip(spec.block_tables, spec.ctx_off):
        for pi in range(len(bt)):
            nv = int(np.clip(int(off) - pi * spec.B, 0, spec.B))
            if nv:
                c, e = q8.quantize_rows(wl.bf16_bits_to_f64(hv.cache[base + pi, :, :, :nv]))
                codes[bt[pi], :, :, :nv] = c
                scales[bt[pi], :, :, :nv] = np.exp2(e.astype(np.float64)).astype(np.float32)
        base += len(bt)
    return codes, scales


def _run(spec, hv, append=True, ctx=None):
    import torch
    codes, scales = _initial_pool(spec, hv)
    want_codes, want_scales = codes.copy(), scales.copy()
    q8.kv_append_fp8(hv.k_new, hv.v_new, want_codes, want_scales, spec.q_len, spec.ctx_off, spec.block_tables)
    if not append:
        codes, scales = want_codes.copy(), want_scales.copy()
    own = ctx is None
    ctx = ctx or gu.make_ctx(spec, kv_dtype=binding.CP_KV_E4M3)
    d_codes = torch.from_numpy(codes).cuda()
    d_scales = torch.from_numpy(scales).cuda()
    out = torch.full((spec.T, spec.Hq, spec.D), float("nan"), device="cuda", dtype=torch.bfloat16)
    ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
    ctx.cp_attention_step_fp8(0, gu.torch_bf16(hv.q), gu.torch_bf16(hv.k_new) if append else None,
                              gu.torch_bf16(hv.v_new) if append else None, d_codes, d_scales, out)
    torch.cuda.synchronize()
    got = wl.bf16_bits_to_f64(gu.to_bits(out)).reshape(spec.T, spec.Hq, spec.D)
    info = ctx.cp_get_batch_info()
    if own:
        ctx.close()
    return got, d_codes.cpu().numpy(), d_scales.cpu().numpy(), want_codes, want_scales, info


def _oracle_out(spec, hv, want_codes, want_scales, rows=None):
    touched = spec.touched_pages()
    pages = q8.pages_as_bf16_bits(want_codes[touched], want_scales[touched], gu.keys_per_page(spec))
    return ora.attention(hv.q, pages, spec.q_len, spec.ctx_off, spec.compact_tables(), spec.sm_scale, rows=rows)


def _assert_fp8_pages(spec, codes, scales, want_codes, want_scales, codes0_untouched=True):
    touched = spec.touched_pages()
    nk = gu.keys_per_page(spec)
    slot = np.arange(spec.B)[None, :]
    is_key = (slot < nk[:, None])[:, None, None, :]                 # [n, 1, 1, B]
    is_tail = ((slot >= nk[:, None]) & (nk[:, None] > 0))[:, None, None, :]
    gc, gs = codes[touched], scales[touched]
    wc, ws = want_codes[touched], want_scales[touched]
    assert np.array_equal(np.where(is_key[..., None], gc, 0), np.where(is_key[..., None], wc, 0)), "codes of key slots differ"
    assert np.array_equal(np.where(is_key, gs, 0).view(np.uint32), np.where(is_key, ws, 0).view(np.uint32)), "scales of key slots differ"
    assert not np.where(is_tail[..., None], gc, 0).any(), "tail codes are not cleared"
    assert np.all(np.where(is_tail, gs, 1.0) == 1.0), "tail scales are not 1"
    other = ~(is_key | is_tail)
    assert np.all(np.where(other[..., None], gc, NAN_CODE) == NAN_CODE), "a slot outside the batch's key range was modified"
    untouched = np.setdiff1d(np.arange(spec.num_blocks), touched)
    assert np.all(codes[untouched] == NAN_CODE) and np.all(np.isnan(scales[untouched]))


@pytest.mark.parametrize("Hq,Hkv,q_len,ctx_off", [
    (8, 2, [1, 1, 1, 1, 1], [0, 15, 16, 700, 2047]),               # decodes only (4 rows per KV head)
    (16, 2, [1, 1, 1], [5, 300, 1999]),                            # G = 8: 8 rows per KV head
    (8, 8, [1] * 6, [0, 1, 127, 128, 129, 1000]),                  # G = 1
    (8, 2, [40, 1, 1, 200, 1], [77, 14, 130, 300, 1000]),          # mixed: chunks go through the scratch pool
    (32, 8, [333, 1, 1, 17, 2], [5, 2047, 15, 250, 31]),           # 8B shape: ragged chunk, 2-token chunk (8 rows)
    (32, 2, [1, 3], [500, 100]),                                   # G = 16: decode rows > 8 -> tile kind on fp8 pages
])
def test_fp8_pages_against_oracle(Hq, Hkv, q_len, ctx_off):
    pages = sum((q + o + 15) // 16 for q, o in zip(q_len, ctx_off)) + 9
    spec = wl.make_spec("fp8", Hq, Hkv, 128, 16, pages, q_len, ctx_off, seed=51)
    hv = wl.host_values(spec)
    for append in (True, False):
        got, codes, scales, want_codes, want_scales, info = _run(spec, hv, append=append)
        want = _oracle_out(spec, hv, want_codes, want_scales)
        gu.assert_close(got, want, f"fp8 pages, append={append}")
        _assert_fp8_pages(spec, codes, scales, want_codes, want_scales)
    # really fp8: the bf16-page result of the same batch differs from the fp8 one by the quantisation error
    plain, _ = gu.run_oracle_host_values(spec, hv)
    assert np.abs(plain - want).max() > 1e-3


def test_fp8_long_decodes_split_and_combine():
    """Long contexts: key ranges are split over the SMs, partials merged by the combine kernel."""
    spec = wl.make_spec("fp8_long", 32, 8, 128, 16, 9000, [1, 1, 1, 1], [30000, 12, 7000, 65535], seed=52)
    hv = wl.host_values(spec)
    got, codes, scales, want_codes, want_scales, info = _run(spec, hv)
    assert info.n_combine_items > 0
    want = _oracle_out(spec, hv, want_codes, want_scales)
    gu.assert_close(got, want, "fp8 long decodes")


def test_fp8_state_errors():
    spec = wl.config_tiny()
    with pytest.raises(binding.CpError):                            # e4m3 pools need head_dim 128
        gu.make_ctx(spec, kv_dtype=binding.CP_KV_E4M3)
    spec = wl.make_spec("e", 8, 2, 128, 16, 40, [1, 200], [100, 0], seed=1)
    import torch
    ctx = gu.make_ctx(spec, kv_dtype=binding.CP_KV_E4M3, max_scratch_pages=4)
    with pytest.raises(binding.CpError) as e:                       # the 200-token chunk needs 13 scratch pages
        ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
    assert e.value.code == binding.CP_ECAPACITY
    ctx.cp_build_batch([1], [100], [spec.block_tables[0]])
    d = torch.zeros(4096, device="cuda", dtype=torch.bfloat16)
    with pytest.raises(binding.CpError) as e:                       # bf16 entry point on an e4m3 context
        ctx.cp_attention_step(0, d, None, None, d, d)
    assert e.value.code == binding.CP_ESTATE
    ctx.close()
    ctx = gu.make_ctx(spec)
    ctx.cp_build_batch([1], [100], [spec.block_tables[0]])
    with pytest.raises(binding.CpError) as e:
        ctx.cp_attention_step_fp8(0, d, None, None, d, d, d)
    assert e.value.code == binding.CP_ESTATE
    ctx.close()
