"""Pins for the fp64 attention oracle (oracle/attention_oracle.c), CPU only.

Each test checks the oracle against something OTHER than itself (SURVEY.md 8(c)
pins 1-7): a dense brute-force softmax written here in numpy, torch's fp64 SDPA,
closed forms, and invariants.  A dropped term, wrong sign/index, transposed
operand, off-by-one diagonal or wrong GQA mapping fails at least one of them.
"""
import numpy as np
import pytest
import torch

from oracle import attention as ora
from paper_2606_09061_b200 import workloads as wl

TOL = 1e-12


# ---- independent helpers (no oracle code) -----------------------------------
def rand_bf16(rng, shape):
    return wl.f32_to_bf16_bits(rng.standard_normal(shape, dtype=np.float32))


def page_out(K, V, B, rng, extra_pages=3, poison=wl.POISON_BF16):
    """Scatter contiguous K,V [L,Hkv,D] (uint16) through a random block table."""
    L, Hkv, D = K.shape
    nb = (L + B - 1) // B
    num_blocks = nb + extra_pages
    cache = np.full((num_blocks, 2, Hkv, B, D), poison, dtype=np.uint16)
    bt = rng.permutation(num_blocks)[:nb].astype(np.int32)
    for t in range(L):
        cache[bt[t // B], 0, :, t % B, :] = K[t]
        cache[bt[t // B], 1, :, t % B, :] = V[t]
    return cache, bt


def brute_force(Q, K, V, scale, offset=0):
    """Dense masked softmax, fp64.  Q [Lq,Hq,D], K,V [L,Hkv,D] as float64;
    row i sees keys 0..offset+i."""
    Lq, Hq, D = Q.shape
    L, Hkv, _ = K.shape
    G = Hq // Hkv
    out = np.zeros((Lq, Hq, D))
    for h in range(Hq):
        S = scale * (Q[:, h, :] @ K[:, h // G, :].T)            # [Lq, L]
        mask = np.arange(L)[None, :] <= (offset + np.arange(Lq))[:, None]
        S = np.where(mask, S, -np.inf)
        P = np.exp(S - S.max(axis=1, keepdims=True))
        out[:, h, :] = (P / P.sum(axis=1, keepdims=True)) @ V[:, h // G, :]
    return out


def f64(bits):
    return wl.bf16_bits_to_f64(bits)


def run_oracle_full(Qb, Kb, Vb, B, rng, scale):
    """Oracle on an unchunked offset-0 prompt whose K/V are already in the cache."""
    L = Kb.shape[0]
    cache, bt = page_out(Kb, Vb, B, rng)
    return ora.attention(Qb, cache, [L], [0], [bt], scale)


# ---- pin 1: brute force ------------------------------------------------------
@pytest.mark.parametrize("L,Hq,Hkv,D,B", [(1, 2, 1, 8, 16), (17, 4, 1, 64, 16),
                                          (128, 8, 2, 32, 16), (75, 6, 3, 16, 8)])
def test_brute_force_unpaged(L, Hq, Hkv, D, B):
    rng = np.random.default_rng(L * 7 + D)
    Qb, Kb, Vb = rand_bf16(rng, (L, Hq, D)), rand_bf16(rng, (L, Hkv, D)), rand_bf16(rng, (L, Hkv, D))
    scale = float(np.float32(1 / np.sqrt(D)))
    got = run_oracle_full(Qb, Kb, Vb, B, rng, scale)
    want = brute_force(f64(Qb), f64(Kb), f64(Vb), scale)
    assert np.abs(got - want).max() <= TOL


def test_brute_force_chunk_with_prefix_and_append():
    """A chunk at offset 48 whose own K/V arrive as k_new/v_new (H2 then attend)."""
    rng = np.random.default_rng(5)
    Hq, Hkv, D, B, off, qn = 4, 2, 32, 16, 48, 21
    L = off + qn
    Kb, Vb = rand_bf16(rng, (L, Hkv, D)), rand_bf16(rng, (L, Hkv, D))
    Qb = rand_bf16(rng, (qn, Hq, D))
    # cache holds only the prefix; the rest is poison until the append
    Kpre, Vpre = Kb.copy(), Vb.copy()
    Kpre[off:] = wl.POISON_BF16
    Vpre[off:] = wl.POISON_BF16
    cache, bt = page_out(Kpre, Vpre, B, rng)
    ora.kv_append(Kb[off:], Vb[off:], cache, [qn], [off], [bt])
    scale = 0.2
    got = ora.attention(Qb, cache, [qn], [off], [bt], scale)
    want = brute_force(f64(Qb), f64(Kb), f64(Vb), float(np.float32(scale)), offset=off)
    assert np.abs(got - want).max() <= TOL


# ---- pin 2: library special case ---------------------------------------------
def test_matches_torch_sdpa_fp64():
    rng = np.random.default_rng(11)
    L, Hq, Hkv, D, B = 96, 8, 2, 64, 16
    Qb, Kb, Vb = rand_bf16(rng, (L, Hq, D)), rand_bf16(rng, (L, Hkv, D)), rand_bf16(rng, (L, Hkv, D))
    scale = float(np.float32(1 / np.sqrt(D)))
    got = run_oracle_full(Qb, Kb, Vb, B, rng, scale)
    G = Hq // Hkv
    q = torch.from_numpy(f64(Qb)).permute(1, 0, 2)[None]
    k = torch.from_numpy(f64(Kb)).permute(1, 0, 2).repeat_interleave(G, dim=0)[None]
    v = torch.from_numpy(f64(Vb)).permute(1, 0, 2).repeat_interleave(G, dim=0)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(q, k, v, is_causal=True, scale=scale)
    ref = ref[0].permute(1, 0, 2).numpy()
    assert np.abs(got - ref).max() <= 1e-11


# ---- pin 3: chunking invariance ------------------------------------------------
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_chunking_invariance(seed):
    rng = np.random.default_rng(100 + seed)
    L, Hq, Hkv, D, B = 90, 4, 2, 32, 16
    Qb, Kb, Vb = rand_bf16(rng, (L, Hq, D)), rand_bf16(rng, (L, Hkv, D)), rand_bf16(rng, (L, Hkv, D))
    scale = float(np.float32(1 / np.sqrt(D)))
    whole = run_oracle_full(Qb, Kb, Vb, B, rng, scale)
    cuts = np.sort(rng.choice(np.arange(1, L), size=6, replace=False))
    cuts = [0, *cuts.tolist(), L]
    if seed == 2:                      # chunks of one token
        cuts = list(range(L + 1))
    empty = np.full_like(Kb, wl.POISON_BF16)
    cache, bt = page_out(empty, empty, B, rng)
    rows = []
    for a, b in zip(cuts[:-1], cuts[1:]):
        ora.kv_append(Kb[a:b], Vb[a:b], cache, [b - a], [a], [bt])
        rows.append(ora.attention(Qb[a:b], cache, [b - a], [a], [bt], scale))
    assert np.abs(np.concatenate(rows) - whole).max() <= TOL


# ---- pin 4: decode consistency ---------------------------------------------------
def test_decode_equals_last_row_of_full_attention():
    rng = np.random.default_rng(21)
    c, Hq, Hkv, D, B = 100, 4, 1, 64, 16
    Qb, Kb, Vb = rand_bf16(rng, (c, Hq, D)), rand_bf16(rng, (c, Hkv, D)), rand_bf16(rng, (c, Hkv, D))
    scale = float(np.float32(1 / np.sqrt(D)))
    cache, bt = page_out(Kb, Vb, B, rng)
    full = ora.attention(Qb, cache, [c], [0], [bt], scale)
    dec = ora.attention(Qb[c - 1:c], cache, [1], [c - 1], [bt], scale)
    assert np.array_equal(dec[0], full[c - 1])
    want = brute_force(f64(Qb), f64(Kb), f64(Vb), scale)[c - 1]
    assert np.abs(dec[0] - want).max() <= TOL


# ---- pin 5: closed forms ----------------------------------------------------------
def test_closed_form_identical_keys_running_mean():
    rng = np.random.default_rng(31)
    L, Hq, Hkv, D, B, off = 40, 2, 1, 16, 16, 13
    Kb = np.repeat(rand_bf16(rng, (1, Hkv, D)), L, axis=0)
    Vb = rand_bf16(rng, (L, Hkv, D))
    Qb = rand_bf16(rng, (L - off, Hq, D))
    cache, bt = page_out(Kb, Vb, B, rng)
    got = ora.attention(Qb, cache, [L - off], [off], [bt], 0.3)
    V = f64(Vb)[:, 0, :]
    for i in range(L - off):
        want = V[: off + i + 1].mean(axis=0)
        for h in range(Hq):
            assert np.abs(got[i, h] - want).max() <= 1e-13
    # (v) Q = 0 gives the same uniform weights for arbitrary K
    Kb2 = rand_bf16(rng, (L, Hkv, D))
    cache2, bt2 = page_out(Kb2, Vb, B, rng)
    got0 = ora.attention(np.zeros_like(Qb), cache2, [L - off], [off], [bt2], 0.3)
    assert np.abs(got0 - got).max() <= 1e-13


def test_closed_form_constant_v_and_first_row():
    rng = np.random.default_rng(32)
    L, Hq, Hkv, D, B = 50, 4, 2, 32, 16
    Qb, Kb = rand_bf16(rng, (L, Hq, D)), rand_bf16(rng, (L, Hkv, D))
    vrow = rand_bf16(rng, (1, Hkv, D))
    Vb = np.repeat(vrow, L, axis=0)
    got = run_oracle_full(Qb, Kb, Vb, B, rng, 0.25)
    G = Hq // Hkv
    for h in range(Hq):
        assert np.abs(got[:, h, :] - f64(vrow)[0, h // G][None, :]).max() <= 1e-13
    # (iii) row 0 at offset 0 returns v_0 exactly
    Vb2 = rand_bf16(rng, (L, Hkv, D))
    got2 = run_oracle_full(Qb, Kb, Vb2, B, rng, 0.25)
    for h in range(Hq):
        assert np.array_equal(got2[0, h], f64(Vb2)[0, h // G])


def test_closed_form_dominant_key():
    """One key with logit ~ +64 above the rest: output = its V row to ~1e-20."""
    rng = np.random.default_rng(33)
    L, D, B = 30, 16, 16
    Kb = np.zeros((L, 1, D), dtype=np.uint16)
    Qb = np.zeros((1, 1, D), dtype=np.uint16)
    one8 = wl.f32_to_bf16_bits(np.array([8.0], dtype=np.float32))[0]
    Qb[0, 0, 0] = one8
    Kb[7, 0, 0] = one8                     # s_7 = 64, all other s = 0
    Vb = rand_bf16(rng, (L, 1, D))
    cache, bt = page_out(Kb, Vb, B, rng)
    got = ora.attention(Qb, cache, [1], [L - 1], [bt], 1.0)
    assert np.abs(got[0, 0] - f64(Vb)[7, 0]).max() <= 1e-20 * 1e3 + 30 * np.exp(-64.0) * 8


# ---- pin 6: invariants --------------------------------------------------------------
def test_block_table_permutation_is_bit_identical_and_poison_free():
    spec = wl.random_spec(3, Hq=4, Hkv=2, D=32)
    hv = wl.host_values(spec)
    tabs = spec.compact_tables()
    c1 = hv.cache.copy()
    ora.kv_append(hv.k_new, hv.v_new, c1, spec.q_len, spec.ctx_off, tabs)
    out1 = ora.attention(hv.q, c1, spec.q_len, spec.ctx_off, tabs, spec.sm_scale)
    assert np.isfinite(out1).all() and np.abs(out1).max() < 10.0   # no poison leaked
    # move pages: same logical content under a permuted table, different poison
    n = hv.cache.shape[0]
    perm = np.random.default_rng(9).permutation(n + 5)[:n]
    c2 = np.full((n + 5,) + hv.cache.shape[1:], wl.POISON_BF16_NEG, dtype=np.uint16)
    before = hv.cache.copy()
    before[before == wl.POISON_BF16] = wl.POISON_BF16_NEG
    before[before == (wl.POISON_BF16 ^ 0x8000)] = wl.NAN_BF16     # strict poison too
    c2[perm] = before
    tabs2 = [perm[t].astype(np.int32) for t in tabs]
    ora.kv_append(hv.k_new, hv.v_new, c2, spec.q_len, spec.ctx_off, tabs2)
    out2 = ora.attention(hv.q, c2, spec.q_len, spec.ctx_off, tabs2, spec.sm_scale)
    assert np.array_equal(out1, out2)


def test_gqa_equals_replicated_mha_and_convexity():
    rng = np.random.default_rng(41)
    L, Hq, Hkv, D, B = 64, 6, 2, 16, 16
    G = Hq // Hkv
    Qb, Kb, Vb = rand_bf16(rng, (L, Hq, D)), rand_bf16(rng, (L, Hkv, D)), rand_bf16(rng, (L, Hkv, D))
    gqa = run_oracle_full(Qb, Kb, Vb, B, rng, 0.25)
    mha = run_oracle_full(Qb, np.repeat(Kb, G, axis=1), np.repeat(Vb, G, axis=1), B, rng, 0.25)
    assert np.array_equal(gqa, mha)
    V = f64(Vb)
    for i in range(L):
        for h in range(Hq):
            lo = V[: i + 1, h // G].min(axis=0) - 1e-12
            hi = V[: i + 1, h // G].max(axis=0) + 1e-12
            assert (gqa[i, h] >= lo).all() and (gqa[i, h] <= hi).all()


def test_sampled_rows_match_full():
    spec = wl.random_spec(4, Hq=4, Hkv=1, D=32)
    hv = wl.host_values(spec)
    tabs = spec.compact_tables()
    c = hv.cache.copy()
    ora.kv_append(hv.k_new, hv.v_new, c, spec.q_len, spec.ctx_off, tabs)
    full = ora.attention(hv.q, c, spec.q_len, spec.ctx_off, tabs, spec.sm_scale)
    rng = np.random.default_rng(0)
    tok = rng.integers(0, spec.T, size=20)
    head = rng.integers(0, spec.Hq, size=20)
    part = ora.attention(hv.q, c, spec.q_len, spec.ctx_off, tabs, spec.sm_scale, rows=(tok, head))
    assert np.array_equal(part, full[tok, head])


def test_bad_table_is_rejected():
    spec = wl.config_tiny()
    hv = wl.host_values(spec)
    tabs = spec.compact_tables()
    short = [t[:-1] if i == 0 else t for i, t in enumerate(tabs)]
    with pytest.raises(ValueError):
        ora.attention(hv.q, hv.cache, spec.q_len, spec.ctx_off, short, spec.sm_scale)


# ---- pin 7: split / combine identity (H5) ---------------------------------------------
@pytest.mark.parametrize("seed", range(4))
def test_split_combine_identity(seed):
    rng = np.random.default_rng(200 + seed)
    n, D = 77, 8
    s = rng.standard_normal(n) * 3
    V = rng.standard_normal((n, D))
    p = np.exp(s - s.max())
    want = (p[:, None] * V).sum(0) / p.sum()
    cuts = np.sort(rng.integers(0, n + 1, size=5))          # may repeat -> empty ranges
    cuts = [0, *cuts.tolist(), n]
    if seed == 3:
        cuts = [0, 1, 2, n]                                   # 1-key ranges
    ms, ls, os_ = [], [], []
    for a, b in zip(cuts[:-1], cuts[1:]):
        if a == b:
            ms.append(-np.inf); ls.append(0.0); os_.append(np.zeros(D)); continue
        m = s[a:b].max()
        e = np.exp(s[a:b] - m)
        ms.append(m); ls.append(e.sum()); os_.append((e[:, None] * V[a:b]).sum(0))
    got = ora.combine_partials(ms, ls, np.stack(os_))
    assert np.abs(got - want).max() <= 1e-13
