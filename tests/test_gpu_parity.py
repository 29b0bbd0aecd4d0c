"""-m gpu parity tests: libcp (through the C ABI) vs the fp64 oracle on the same seeded
inputs.  Tolerance: max-abs 2e-2 and mean-abs 2e-3 on bf16 outputs (BASELINE.json)."""
import numpy as np
import pytest

from oracle import attention as ora
from paper_2606_09061_b200 import binding, workloads as wl
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu

VARIANTS = [0]          # the shipped library holds ONE attention kernel (a -DCP_DEBUG_VARIANTS build adds 1 = SIMT cross-check)


@pytest.mark.parametrize("variant", VARIANTS)
def test_tiny_config_full(variant):
    spec = wl.config_tiny()
    hv = wl.host_values(spec)
    got, pool_after = gu.run_gpu_host_values(spec, hv, variant)
    want, cache_after = gu.run_oracle_host_values(spec, hv)
    gu.assert_close(got, want, "tiny")
    # H2: the appended rows are bit-identical to the oracle's append; last-page tails are cleared; nothing else moved
    gu.assert_pages(pool_after[spec.touched_pages()], cache_after, gu.keys_per_page(spec))
    untouched = np.setdiff1d(np.arange(spec.num_blocks), spec.touched_pages())
    assert np.array_equal(pool_after[untouched], wl.full_pool_from_compact(spec, hv.cache)[untouched])


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("seed,Hq,Hkv,D", [(1, 8, 2, 64), (2, 8, 8, 128), (3, 16, 2, 128),
                                           (4, 16, 1, 64), (5, 4, 2, 128), (6, 32, 8, 128)])
def test_random_mixed_batches(variant, seed, Hq, Hkv, D):
    spec = wl.random_spec(seed, Hq=Hq, Hkv=Hkv, D=D, n_prefill=4, n_decode=6, max_chunk=300,
                          max_ctx=700)
    hv = wl.host_values(spec)
    got, _ = gu.run_gpu_host_values(spec, hv, variant)
    want, _ = gu.run_oracle_host_values(spec, hv)
    gu.assert_close(got, want, spec.name)


@pytest.mark.parametrize("variant", VARIANTS)
def test_edge_shapes(variant):
    # single key; chunk lengths around the tile sizes; offsets around tile/page boundaries
    q_len = [1, 1, 1, 127, 128, 129, 33, 16, 1, 257]
    ctx_off = [0, 15, 16, 0, 1, 127, 128, 255, 511, 3]
    spec = wl.make_spec("edges", 8, 2, 128, 16, 400, q_len, ctx_off, seed=3)
    hv = wl.host_values(spec)
    got, _ = gu.run_gpu_host_values(spec, hv, variant)
    want, _ = gu.run_oracle_host_values(spec, hv)
    gu.assert_close(got, want, "edges")


@pytest.mark.parametrize("variant", VARIANTS)
def test_caller_wrote_pages_path_and_stale_tails(variant):
    spec = wl.random_spec(11, Hq=8, Hkv=2, D=128)
    hv = wl.host_values(spec)
    want, _ = gu.run_oracle_host_values(spec, hv)
    got, _ = gu.run_gpu_host_values(spec, hv, variant, append=False)
    gu.assert_close(got, want, "k_new=NULL")
    # different stale data in tails / untouched pages must not change a single output bit
    got2, _ = gu.run_gpu_host_values(spec, hv, variant, append=False, poison=wl.POISON_BF16_NEG)
    assert np.array_equal(got, got2)


@pytest.mark.parametrize("q_len,ctx_off", [([1, 1, 1, 1, 40, 200], [0, 14, 130, 1000, 77, 300]),
                                           ([333, 1, 1, 17], [5, 2047, 15, 250])])
@pytest.mark.parametrize("Hq,Hkv,D", [(8, 2, 128), (8, 2, 64), (16, 1, 128)])
def test_stale_tails_nan_strict(Hq, Hkv, D, q_len, ctx_off):
    """SURVEY.md 8(c) reading table, "Stale data in page tails / unused pool pages ... NaN in a strict mode":
    every slot that is not a key of its request -- the tails of last pages, every untouched page of the pool --
    holds NaN.  The output must be finite, within tolerance of the oracle, and bit-identical to the run with
    finite poison.  Both append paths: k_new given (the step appends) and k_new = NULL (caller wrote the pages)."""
    pages = sum((q + o + 15) // 16 for q, o in zip(q_len, ctx_off)) + 9
    spec = wl.make_spec("nan_strict", Hq, Hkv, D, 16, pages, q_len, ctx_off, seed=31)
    hv_nan = wl.host_values(spec, poison=wl.NAN_BF16)
    hv_fin = wl.host_values(spec)
    want, _ = gu.run_oracle_host_values(spec, hv_fin)
    for append in (True, False):
        got_fin, _ = gu.run_gpu_host_values(spec, hv_fin, 0, append=append)
        got_nan, pool_after = gu.run_gpu_host_values(spec, hv_nan, 0, append=append, poison=wl.NAN_BF16)
        gu.assert_close(got_nan, want, f"NaN tails, append={append}")
        assert np.array_equal(got_nan, got_fin)
    # the NaN really was there: the pool's untouched pages still hold it after the step; the tails of the requests'
    # last pages were cleared by the step (they hold no key)
    untouched = np.setdiff1d(np.arange(spec.num_blocks), spec.touched_pages())
    assert ((pool_after[untouched] & 0x7FFF) == wl.NAN_BF16).all()
    _, cache_after = gu.run_oracle_host_values(spec, hv_nan)
    gu.assert_pages(pool_after[spec.touched_pages()], cache_after, gu.keys_per_page(spec))


@pytest.mark.parametrize("variant", VARIANTS)
def test_chunking_invariance_and_decode_consistency_on_gpu(variant):
    """A prompt processed as chunks equals the unchunked prompt (within 2x tolerance GPU vs
    GPU, within tolerance vs the oracle); a decode equals the last row of full attention."""
    import torch
    rng = np.random.default_rng(5)
    L, Hq, Hkv, D, B = 300, 8, 2, 128, 16
    Kb = wl.f32_to_bf16_bits(rng.standard_normal((L, Hkv, D), dtype=np.float32))
    Vb = wl.f32_to_bf16_bits(rng.standard_normal((L, Hkv, D), dtype=np.float32))
    Qb = wl.f32_to_bf16_bits(rng.standard_normal((L, Hq, D), dtype=np.float32))
    nb = (L + B - 1) // B
    bt = rng.permutation(nb + 6)[:nb].astype(np.int32)
    spec1 = wl.BatchSpec("whole", Hq, Hkv, D, B, nb + 6, np.array([L], np.int32), np.array([0], np.int32), [bt])
    ctx = gu.make_ctx(spec1, variant, max_tokens=L, max_reqs=4)

    def run(cuts):
        pool = gu.torch_bf16(np.full((nb + 6, 2, Hkv, B, D), wl.POISON_BF16, np.uint16))
        outs = []
        for a, b in zip(cuts[:-1], cuts[1:]):
            out = torch.empty((b - a, Hq, D), device="cuda", dtype=torch.bfloat16)
            ctx.cp_build_batch([b - a], [a], [bt])
            ctx.cp_attention_step(0, gu.torch_bf16(Qb[a:b]), gu.torch_bf16(Kb[a:b]), gu.torch_bf16(Vb[a:b]), pool, out)
            outs.append(wl.bf16_bits_to_f64(gu.to_bits(out)))
        return np.concatenate(outs), pool

    whole, pool = run([0, L])
    chunked, _ = run([0, 1, 2, 50, 128, 129, 177, 290, L])
    cache = np.full((nb + 6, 2, Hkv, B, D), wl.POISON_BF16, np.uint16)
    ora.kv_append(Kb, Vb, cache, [L], [0], [bt])
    want = ora.attention(Qb, cache, [L], [0], [bt], spec1.sm_scale)
    gu.assert_close(whole, want, "unchunked")
    gu.assert_close(chunked, want, "chunked")
    assert np.abs(whole - chunked).max() <= 2 * gu.MAX_ABS_TOL
    # decode consistency: q of the last token as a decode over the full cache
    out = torch.empty((1, Hq, D), device="cuda", dtype=torch.bfloat16)
    ctx.cp_build_batch([1], [L - 1], [bt])
    ctx.cp_attention_step(0, gu.torch_bf16(Qb[L - 1:]), None, None, pool, out)
    dec = wl.bf16_bits_to_f64(gu.to_bits(out))
    gu.assert_close(dec, want[L - 1:], "decode = last row")
    ctx.close()


@pytest.mark.parametrize("variant", VARIANTS)
def test_closed_form_constant_v(variant):
    spec = wl.random_spec(21, Hq=8, Hkv=2, D=64)
    hv = wl.host_values(spec)
    vrow = wl.f32_to_bf16_bits(np.random.default_rng(0).standard_normal((1, spec.Hkv, spec.D), dtype=np.float32))
    hv.v_new[:] = vrow
    base = 0
    for bt, off in zip(spec.block_tables, spec.ctx_off):
        for pi in range(len(bt)):
            n_valid = min(max(int(off) - pi * spec.B, 0), spec.B)
            hv.cache[base + pi, 1, :, :n_valid, :] = vrow[0][:, None, :]
        base += len(bt)
    got, _ = gu.run_gpu_host_values(spec, hv, variant)
    G = spec.Hq // spec.Hkv
    want = np.repeat(wl.bf16_bits_to_f64(vrow)[0], G, axis=0)[None]
    assert np.abs(got - want).max() <= 2 ** -8 * np.abs(want).max()      # one bf16 rounding


def test_empty_batch_and_errors():
    import torch
    spec = wl.config_tiny()
    with pytest.raises(binding.CpError) as e:           # one attention kernel: no variant dispatch in the shipped library
        gu.make_ctx(spec, 1)
    assert e.value.code == binding.CP_EINVAL
    with pytest.raises(binding.CpError) as e:
        gu.make_ctx(spec, 0, sm_scale=0.0)
    assert e.value.code == binding.CP_EINVAL
    ctx = gu.make_ctx(spec, 0, max_tokens=64, max_reqs=4, max_total_pages=16)
    with pytest.raises(binding.CpError) as e:
        ctx.cp_attention_step(0, 16, None, None, 16, 16)
    assert e.value.code == binding.CP_ESTATE
    ctx.cp_build_batch([], [], [])
    dummy = torch.zeros(64, device="cuda", dtype=torch.bfloat16)
    ctx.cp_attention_step(0, dummy, None, None, dummy, dummy)           # no-op, still timed
    torch.cuda.synchronize()
    for q, o, bt, code in [([0], [0], [[0]], binding.CP_EINVAL), ([1], [-1], [[0]], binding.CP_EINVAL),
                           ([17], [0], [[0]], binding.CP_EINVAL), ([1], [0], [[16]], binding.CP_EINVAL),
                           ([65], [0], [[0, 1, 2, 3, 4]], binding.CP_ECAPACITY),
                           ([1] * 5, [0] * 5, [[i] for i in range(5)], binding.CP_ECAPACITY)]:
        with pytest.raises(binding.CpError) as e:
            ctx.cp_build_batch(q, o, [np.asarray(b, np.int32) for b in bt])
        assert e.value.code == code
    assert ctx.cp_get_batch_info().n_reqs == 0          # failed builds kept the previous batch
    ctx.close()


def test_latency_table_rows():
    import torch
    spec = wl.config_tiny()
    hv = wl.host_values(spec)
    ctx = gu.make_ctx(spec, 0, num_layers=3)
    ctx.cp_set_memory_stats(10.0, 20.0, 5.0, 8.0)
    pool = gu.torch_bf16(wl.full_pool_from_compact(spec, hv.cache))
    out = torch.empty((spec.T, spec.Hq, spec.D), device="cuda", dtype=torch.bfloat16)
    ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
    for layer in range(3):
        ctx.cp_attention_step(layer, gu.torch_bf16(hv.q), None if layer else gu.torch_bf16(hv.k_new),
                              None if layer else gu.torch_bf16(hv.v_new), pool, out)
    rows = ctx.cp_latency_table()
    assert [r.layer for r in rows] == [0, 1, 2] and all(r.us > 0 for r in rows)
    r = rows[0]
    # Table 1 features of this batch: chunks (32 @0), (16 @48); decodes ctx 40, 100
    assert list(r.feat) == [48.0, 2.0, 4.0, 140.0, 100.0, 48.0, 48.0, 10.0, 20.0, 5.0, 8.0]
    assert (r.n_prefill, r.n_decode, r.iter) == (2, 2, 0)
    assert ctx.cp_latency_table() == []
    # a 1-token prefill chunk (Eq. 8's candidate c = 1, the last token of a prompt) is flagged by the scheduler and
    # counts as prefill in the Table-1 features, as in the scheduler's own feature vector; unflagged it is a decode
    ctx.cp_build_batch([1, 1], [7, 99], [spec.block_tables[0], spec.block_tables[3]], flags=[binding.CP_REQ_PREFILL, 0])
    ctx.cp_attention_step(0, gu.torch_bf16(hv.q[:2]), None, None, pool, out)
    r = ctx.cp_latency_table()[0]
    assert list(r.feat[:7]) == [1.0, 1.0, 2.0, 100.0, 100.0, 7.0, 7.0] and (r.n_prefill, r.n_decode) == (1, 1)
    # all layers in one submission: one row for the iteration, layer = -n
    pa = binding.Context.pointer_array
    q2 = gu.torch_bf16(hv.q[:2])
    ctx.cp_attention_layers(pa([q2] * 3), None, None, pa([pool] * 3), pa([out] * 3))
    rows = ctx.cp_latency_table()
    assert len(rows) == 1 and rows[0].layer == -3 and rows[0].us > 0
    ctx.close()


def test_stress_long_decodes_with_chunk_no_deadlock():
    """Regression: swap-kind (decode) items used to let the softmax warps run a full p_full phase
    ahead of the MMA issuer (mbarrier parity aliasing -> rare deadlock, seen in the trace run).
    Many back-to-back launches of the batch shape that triggered it; result checked on a sample."""
    import torch
    rng = np.random.default_rng(7)
    ctx_dec = rng.integers(17000, 23500, size=13)
    spec = wl.make_spec("stress", 32, 8, 128, 16, 24000, [1] * 13 + [1, 530],
                        list(ctx_dec - 1) + [1992, 1500], seed=7)
    dev = torch.device("cuda:0")
    q, k_new, v_new, pool, compact = wl.device_values(spec, dev)
    ctx = gu.make_ctx(spec, 0)
    out = torch.empty((spec.T, spec.Hq, spec.D), device=dev, dtype=torch.bfloat16)
    ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
    for i in range(1500):
        ctx.cp_attention_step(0, q, k_new if i == 0 else None, v_new if i == 0 else None, pool, out)
        if i % 500 == 499:
            torch.cuda.synchronize()
            ctx.cp_latency_table()
    torch.cuda.synchronize()
    cache = gu.to_bits(compact)
    tabs = spec.compact_tables()
    ora.kv_append(gu.to_bits(k_new), gu.to_bits(v_new), cache, spec.q_len, spec.ctx_off, tabs)
    tok, head = gu.sample_rows(spec, 96)
    want = ora.attention(gu.to_bits(q), cache, spec.q_len, spec.ctx_off, tabs, spec.sm_scale, rows=(tok, head))
    got = wl.bf16_bits_to_f64(gu.to_bits(out)).reshape(spec.T, spec.Hq, spec.D)[tok, head]
    gu.assert_close(got, want, "stress")
    ctx.close()


def test_split_decode_groups_are_merged_inside_the_attention_kernel():
    """H5 without a launch: the split-KV groups of decodes (swap-kind items) are merged by the split that arrives
    last, inside the attention kernel; a decode-only batch is two launches (append, attention).  Three steps in a row
    on one batch with different Q, then another batch on the same context: the groups' arrival counters re-arm
    themselves, stale partial rows of an earlier step never reach a result (out starts as NaN every time)."""
    import torch
    rng = np.random.default_rng(5)
    ctx_a = list(rng.integers(3000, 20000, size=6)) + [1, 17, 300, 129]
    spec = wl.make_spec("fused", 32, 8, 128, 16, 6000, [1] * len(ctx_a), [c - 1 for c in ctx_a], seed=51)
    dev = torch.device("cuda:0")
    ctx = gu.make_ctx(spec)
    tabs = spec.compact_tables()
    q, k_new, v_new, pool, compact = wl.device_values(spec, dev)
    cache = gu.to_bits(compact)
    ora.kv_append(gu.to_bits(k_new), gu.to_bits(v_new), cache, spec.q_len, spec.ctx_off, tabs)
    ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
    info = ctx.cp_get_batch_info()
    assert info.n_combine_items > 0
    for step in range(3):
        if step:
            q = (torch.randn(q.shape, device=dev, dtype=torch.float32, generator=torch.Generator(device=dev).manual_seed(step)) * 1.5).bfloat16()
        out = torch.full((spec.T, spec.Hq, spec.D), float("nan"), device=dev, dtype=torch.bfloat16)
        ctx.cp_attention_step(0, q, k_new if step == 0 else None, v_new if step == 0 else None, pool, out)
        torch.cuda.synchronize()
        want = ora.attention(gu.to_bits(q), cache, spec.q_len, spec.ctx_off, tabs, spec.sm_scale)
        got = wl.bf16_bits_to_f64(gu.to_bits(out)).reshape(spec.T, spec.Hq, spec.D)
        gu.assert_close(got, want, f"fused merge, step {step}")
    info = ctx.cp_get_batch_info()
    assert info.grid_combine == 0 and info.kernels_per_step == 1          # no combine launch, no append launch (H2 inside the attention kernel)
    # another batch on the same context: fewer, differently split groups reuse the counters and the workspace
    sub = [0, 3, 6, 8]
    spec2 = wl.BatchSpec("fused2", spec.Hq, spec.Hkv, spec.D, spec.B, spec.num_blocks, spec.q_len[sub], spec.ctx_off[sub],
                         [spec.block_tables[j] for j in sub], spec.seed)
    q2 = q[sub].contiguous()
    out2 = torch.full((len(sub), spec.Hq, spec.D), float("nan"), device=dev, dtype=torch.bfloat16)
    ctx.cp_build_batch(spec2.q_len, spec2.ctx_off, spec2.block_tables)
    ctx.cp_attention_step(0, q2, None, None, pool, out2)
    torch.cuda.synchronize()
    want_all = ora.attention(gu.to_bits(q), cache, spec.q_len, spec.ctx_off, tabs, spec.sm_scale)
    got2 = wl.bf16_bits_to_f64(gu.to_bits(out2)).reshape(len(sub), spec.Hq, spec.D)
    gu.assert_close(got2, want_all[sub], "fused merge, second batch")
    ctx.close()


def test_few_long_decodes_fit_one_round_of_the_lanes():
    """A decode-only round with few long requests (what the configs[4] trace runs most of the time): cp_build_batch
    picks the split length by the number of ROUNDS the lanes need, not by the mean load alone, so the
    work list has at most one item per lane (2 lanes x SMs) and at most as many as the mean-load rule would give;
    every row against the oracle (the merge of the split groups runs inside the attention kernel)."""
    import torch
    spec = wl.config_small_decode(seed=3)
    dev = torch.device("cuda:0")
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    ctx = gu.make_ctx(spec)
    q, k_new, v_new, pool, compact = wl.device_values(spec, dev)
    cache = gu.to_bits(compact)
    tabs = spec.compact_tables()
    ora.kv_append(gu.to_bits(k_new), gu.to_bits(v_new), cache, spec.q_len, spec.ctx_off, tabs)
    ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
    info = ctx.cp_get_batch_info()
    tiles = [(int(c) + 1 + 127) // 128 for c in spec.ctx_off]
    mean_load = -(-sum(tiles) * spec.Hkv // (2 * n_sm))
    by_mean_load = sum(-(-t // mean_load) for t in tiles) * spec.Hkv
    assert by_mean_load > 2 * n_sm                      # the case the rule exists for: slightly more items than lanes
    assert info.n_work_items <= 2 * n_sm and info.n_work_items <= by_mean_load
    assert info.n_combine_items > 0 and info.n_work_items >= n_sm
    out = torch.full((spec.T, spec.Hq, spec.D), float("nan"), device=dev, dtype=torch.bfloat16)
    ctx.cp_attention_step(0, q, k_new, v_new, pool, out)
    torch.cuda.synchronize()
    assert ctx.cp_get_batch_info().kernels_per_step == 1          # decode-only: the append runs inside the attention kernel
    want = ora.attention(gu.to_bits(q), cache, spec.q_len, spec.ctx_off, tabs, spec.sm_scale)
    got = wl.bf16_bits_to_f64(gu.to_bits(out)).reshape(spec.T, spec.Hq, spec.D)
    gu.assert_close(got, want, "12 long decodes")
    # H2 parity of the fused append: every appended row bit for bit, the tail of each last page zero, nothing else touched
    gu.assert_pages(gu.to_bits(pool)[spec.touched_pages()], cache, gu.keys_per_page(spec), "fused append")
    ctx.close()


@pytest.mark.parametrize("Hq,Hkv", [(8, 2), (4, 4), (16, 1)])
def test_fused_append_of_small_decode_only_batches(Hq, Hkv):
    """Small batches without a tile-kind item run ONE kernel: the attention kernel's producers append the step's rows and
    clear the page tails (include/cp.h).  Requests of 1..4 tokens (as many as still make a swap-kind item) whose new rows
    start a request, straddle page and tile boundaries, end exactly on them, and sit behind long split contexts; NaN in
    every stale slot; outputs against the oracle on every row, pages bit for bit; then a second step with k_new = NULL
    (the caller wrote the pages: only the tails are cleared)."""
    import torch
    G = Hq // Hkv
    qmax = 16 // G                                           # tokens of a swap-kind q tile
    ctx_off = [0, 13, 14, 15, 16, 125, 126, 127, 128, 255, 1023, 5000, 20001]
    q_len = [min(qmax, 1 + (i % 4)) for i in range(len(ctx_off))]
    pages = sum((q + o + 15) // 16 for q, o in zip(q_len, ctx_off)) + 9
    spec = wl.make_spec("fused_append", Hq, Hkv, 128, 16, pages, q_len, ctx_off, seed=77)
    hv = wl.host_values(spec, poison=wl.NAN_BF16)
    ctx = gu.make_ctx(spec)
    got, pool_after = gu.run_gpu_host_values(spec, hv, 0, ctx=ctx, poison=wl.NAN_BF16)
    info = ctx.cp_get_batch_info()
    assert info.kernels_per_step == 1 and info.n_combine_items > 0
    want, _ = gu.run_oracle_host_values(spec, wl.host_values(spec))
    gu.assert_close(got, want, "fused append")
    _, cache_nan = gu.run_oracle_host_values(spec, hv)
    gu.assert_pages(pool_after[spec.touched_pages()], cache_nan, gu.keys_per_page(spec), "fused append")
    got2, pool_after2 = gu.run_gpu_host_values(spec, hv, 0, append=False, ctx=ctx, poison=wl.NAN_BF16)
    assert ctx.cp_get_batch_info().kernels_per_step == 1
    gu.assert_close(got2, want, "fused tail clearing, caller-written pages")
    gu.assert_pages(pool_after2[spec.touched_pages()], cache_nan, gu.keys_per_page(spec), "fused tail clearing")
    ctx.close()


@pytest.mark.parametrize("seed", range(100, 112))
def test_fuzz_shapes_against_oracle(seed):
    """Randomised shapes: every supported group size, both head dims, ragged chunks, contexts long enough
    for split key ranges and several tiles per item, decodes and chunks in random order."""
    rng = np.random.default_rng(seed)
    G = int(rng.choice([1, 2, 4, 8, 16]))
    Hkv = int(rng.choice([1, 2, 4]))
    D = int(rng.choice([64, 128]))
    spec = wl.random_spec(seed, Hq=G * Hkv, Hkv=Hkv, D=D, n_prefill=int(rng.integers(0, 5)), n_decode=int(rng.integers(0, 24)),
                          max_chunk=int(rng.choice([40, 300, 900])), max_ctx=int(rng.choice([100, 1500, 6000])))
    if spec.T == 0:
        pytest.skip("empty draw")
    hv = wl.host_values(spec)
    got, pool_after = gu.run_gpu_host_values(spec, hv, 0)
    want, cache_after = gu.run_oracle_host_values(spec, hv)
    gu.assert_close(got, want, spec.name)
    gu.assert_pages(pool_after[spec.touched_pages()], cache_after, gu.keys_per_page(spec))


def test_repeated_launches_mixed_shapes_no_deadlock():
    """Back-to-back launches over alternating batch shapes (tile-heavy, decode-heavy, mixed, split and
    unsplit items): the persistent kernel's counters, rings and barrier phases must re-arm every time."""
    import torch
    dev = torch.device("cuda:0")
    shapes = [([1] * 40 + [700, 333], list(range(500, 4500, 100)) + [2500, 0]),
              ([1] * 3, [30000, 12, 7000]),
              ([129, 1, 64, 1, 1, 2047], [0, 999, 4096, 1, 127, 9000]),
              ([1] * 200, [int(x) for x in np.random.default_rng(3).integers(1, 3000, 200)])]
    runs = []
    for k, (q_len, ctx_off) in enumerate(shapes):
        spec = wl.make_spec(f"rep{k}", 32, 8, 128, 16, 24000, q_len, ctx_off, seed=k)
        q, k_new, v_new, pool, compact = wl.device_values(spec, dev)
        out = torch.empty((spec.T, spec.Hq, spec.D), device=dev, dtype=torch.bfloat16)
        runs.append((spec, q, k_new, v_new, pool, compact, out))
    ctx = binding.Context(32, 8, 128, 24000, 16, max_tokens=4096, max_reqs=256, max_total_pages=24000)
    for it in range(300):
        spec, q, k_new, v_new, pool, compact, out = runs[it % len(runs)]
        ctx.cp_build_batch(spec.q_len, spec.ctx_off, spec.block_tables)
        ctx.cp_attention_step(0, q, k_new if it < len(runs) else None, v_new if it < len(runs) else None, pool, out)
    torch.cuda.synchronize()
    ctx.cp_latency_table()
    for spec, q, k_new, v_new, pool, compact, out in runs:
        cache = gu.to_bits(compact)
        tabs = spec.compact_tables()
        ora.kv_append(gu.to_bits(k_new), gu.to_bits(v_new), cache, spec.q_len, spec.ctx_off, tabs)
        tok, head = gu.sample_rows(spec, 64)
        want = ora.attention(gu.to_bits(q), cache, spec.q_len, spec.ctx_off, tabs, spec.sm_scale, rows=(tok, head))
        got = wl.bf16_bits_to_f64(gu.to_bits(out)).reshape(spec.T, spec.Hq, spec.D)[tok, head]
        gu.assert_close(got, want, spec.name)
    ctx.close()


@pytest.mark.parametrize("Hq,Hkv,D,q_len,ctx_off", [(8, 2, 128, [300, 129], [517, 0]), (8, 2, 64, [257], [1000]),
                                                    (32, 8, 128, [384], [2048])])
def test_tensor_bound_batches_take_the_fma_pipe_share_kernel(Hq, Hkv, D, q_len, ctx_off):
    """Chunk-only batches are tensor-bound by the SURVEY.md 8(d) formulas, so cp_attention_step launches the
    instantiation that evaluates every fourth exponential of a score row with a polynomial on the FMA pipe
    (DESIGN.md 6.1); same tolerance, full oracle.  The same chunks next to long decodes form an HBM-bound batch
    and take the MUFU-only instantiation: also within tolerance."""
    pages = sum((q + o + 15) // 16 for q, o in zip(q_len, ctx_off)) + 40
    spec = wl.make_spec("tensor_bound", Hq, Hkv, D, 16, pages, q_len, ctx_off, seed=21)
    hv = wl.host_values(spec)
    got, _ = gu.run_gpu_host_values(spec, hv, 0)
    want, _ = gu.run_oracle_host_values(spec, hv)
    gu.assert_close(got, want, "tensor-bound batch")
    # the same chunks next to enough long decodes to make the batch HBM-bound: the MUFU-only instantiation
    dec_ctx = [6000] * 24
    spec2 = wl.make_spec("hbm_bound", Hq, Hkv, D, 16, pages + 24 * 376 + 40, q_len + [1] * 24,
                         ctx_off + [c - 1 for c in dec_ctx], seed=21)
    hv2 = wl.host_values(spec2)
    got2, _ = gu.run_gpu_host_values(spec2, hv2, 0)
    tok, head = gu.sample_rows(spec2, 256, seed=3)
    want2, _ = gu.run_oracle_host_values(spec2, hv2, rows=(tok, head))
    gu.assert_close(got2[tok, head], want2, "hbm-bound batch")


SPLIT_CASES = [
    # (Hq, Hkv, D, q_len, ctx_off): every batch is tensor-bound by the SURVEY.md 8(d) formulas -> SPLIT instantiation
    (8, 2, 128, [1200], [0]),                      # G = 4: a pair is 2 x 32 tokens; 18.75 pairs -> last pair's second tile empty
    (8, 2, 128, [1376, 673], [200, 1000]),         # odd numbers of Q tiles, ragged key ranges
    (8, 2, 128, [579, 769], [5, 777]),             # remainders: a 3-token tail (12 rows -> swap-kind item on the TWIN kernel)
    (2, 2, 128, [2600], [100]),                    # G = 1: a pair is 256 tokens
    (16, 1, 128, [700, 663], [0, 3000]),           # G = 16: a pair is 16 tokens
    (16, 2, 64, [1300, 900], [1000, 0]),           # D = 64 (tile kind only), G = 8
    (8, 2, 128, [100], [30000]),                   # long context: the pair's key range is split over the SMs + combine
    (32, 8, 128, [384, 1, 1, 1], [2048, 300, 17, 4000]),   # 8B shape with a few short decodes (swap items after the tiles)
    (64, 8, 128, [200, 1], [5000, 12000]),         # 70B shape, G = 8
    (8, 2, 128, [1000, 65], [64, 0]),              # last tile of <= 64 keys (phantom second half), 1-token remainder
]


@pytest.mark.parametrize("Hq,Hkv,D,q_len,ctx_off", SPLIT_CASES)
def test_split_mode_tensor_bound_batches(Hq, Hkv, D, q_len, ctx_off):
    """Tensor-bound batches run the SPLIT instantiation (both softmax warpgroups on every chunk tile):
    full oracle comparison, NaN in every stale slot, pages bit-exact; cp_get_batch_info confirms the mode."""
    pages = sum((q + o + 15) // 16 for q, o in zip(q_len, ctx_off)) + 11
    spec = wl.make_spec("split", Hq, Hkv, D, 16, pages, q_len, ctx_off, seed=41)
    hv = wl.host_values(spec, poison=wl.NAN_BF16)
    ctx = gu.make_ctx(spec)
    got, pool_after = gu.run_gpu_host_values(spec, hv, 0, ctx=ctx, poison=wl.NAN_BF16)
    assert ctx.cp_get_batch_info().split == 1
    ctx.close()
    want, cache_after = gu.run_oracle_host_values(spec, wl.host_values(spec))
    gu.assert_close(got, want, "split")
    _, cache_nan = gu.run_oracle_host_values(spec, hv)
    gu.assert_pages(pool_after[spec.touched_pages()], cache_nan, gu.keys_per_page(spec))
