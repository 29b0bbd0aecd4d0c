"""cp_decode_attention_static (include/cp.h): the entry point that allocates nothing -- its split-KV partials live
in a file-scope static device array.  Checked against the EXISTING path (cp_build_batch + cp_attention_step on the
same decode batch) within the tolerance of the parity tests, on two calls in a row with different shapes, split
counts and context lengths (the array keeps the first call's contents; the second must not see them).

Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest

from paper_2606_09061_b200 import binding, workloads as wl
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu


def _run_both(spec, n_splits, seed):
    """Returns (existing path's out, static entry point's out, oracle's out), float64 [n_reqs, Hq, D]."""
    import torch
    hv = wl.host_values(spec, seed=seed)
    ref, pool_after = gu.run_gpu_host_values(spec, hv)              # existing path; the pool now holds the new rows
    pool = gu.torch_bf16(pool_after)
    q = gu.torch_bf16(hv.q)
    n = spec.n_reqs
    max_pages = max(len(b) for b in spec.block_tables)
    bt = np.zeros((n, max_pages), dtype=np.int32)
    for j, b in enumerate(spec.block_tables):
        bt[j, :len(b)] = b
    bt_d = torch.from_numpy(bt).cuda()
    kv_len_d = torch.from_numpy((spec.ctx_off + 1).astype(np.int32)).cuda()
    out = torch.full((n, spec.Hq, spec.D), float("nan"), device="cuda", dtype=torch.bfloat16)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    binding.cp_decode_attention_static(q, pool, bt_d, kv_len_d, n, max_pages, spec.Hq, spec.Hkv, spec.D, spec.B,
                                       spec.sm_scale, n_splits, out)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    got = wl.bf16_bits_to_f64(gu.to_bits(out)).reshape(n, spec.Hq, spec.D)
    want, _ = gu.run_oracle_host_values(spec, hv)
    return ref, got, want, free_before - free_after


def test_static_entry_point_matches_the_existing_path_twice_in_a_row():
    rng = np.random.default_rng(7)
    # call 1: 8B shape, 12 decodes with contexts up to 3000 keys, 8 splits (3072 of the 4096 partial rows)
    ctx1 = rng.integers(1, 3001, size=12)
    ctx1[0], ctx1[1] = 1, 17                                       # one key only; one key past a page boundary
    spec1 = wl.make_spec("static1", 32, 8, 128, 16, 4096, [1] * 12, list(ctx1 - 1), seed=11)
    # call 2: other shape, fewer rows, short contexts, 3 splits (more splits than keys for some requests: empty splits)
    spec2 = wl.make_spec("static2", 8, 2, 64, 16, 64, [1] * 5, [0, 1, 15, 16, 40], seed=12)
    used = []
    for spec, n_splits, seed in ((spec1, 8, 21), (spec2, 3, 22)):
        ref, got, want, used_bytes = _run_both(spec, n_splits, seed)
        gu.assert_close(got, ref, f"{spec.name}: static entry point vs cp_attention_step")
        gu.assert_close(got, want, f"{spec.name}: static entry point vs the fp64 oracle")
        used.append(used_bytes)
    # the second call (module loaded, symbol address known) takes no device memory at all
    assert used[1] == 0, f"device memory in use grew by {used[1]} bytes across a call that must not allocate"


def test_static_entry_point_rejects_what_does_not_fit():
    import torch
    lib = binding.load()
    t = torch.zeros(64, device="cuda", dtype=torch.int32)
    p = int(t.data_ptr())
    # 33 requests x 32 heads x 4 splits = 4224 > CP_STATIC_MAX_PARTIAL_ROWS: refused before anything is launched
    rc = lib.cp_decode_attention_static(p, p, p, p, 33, 1, 32, 8, 128, 16, 0.1, 4, p, None)
    assert rc == binding.CP_ECAPACITY
    msg = lib.cp_last_error().decode()
    assert "CP_STATIC_MAX_PARTIAL_ROWS" in msg and "4224" in msg
    assert 32 * 32 * 4 == binding.CP_STATIC_MAX_PARTIAL_ROWS
    assert lib.cp_decode_attention_static(p, p, p, p, 1, 1, 32, 8, 96, 16, 0.1, 1, p, None) == binding.CP_EINVAL
    assert lib.cp_decode_attention_static(None, p, p, p, 1, 1, 32, 8, 128, 16, 0.1, 1, p, None) == binding.CP_EINVAL
    torch.cuda.synchronize()
