"""Pins for the reference scheduler (oracle/ref_scheduler.py), CPU only.

The paper prints no worked numeric example of its scheduler, so
the pins are what the paper and the mathematics fix: Eq. 3 order equivalence, the
FCFS / shortest-remaining-first limits, the closed-form overtake
time from Eq. 1, conservation laws (Eq. 2, Eq. 6, decode-first PAPER.md:87), Alg. 1
against a brute-force argmin and a closed form, Eq. 12-14 against a literal
transcription over an exhaustive grid.  Each expected value is computed here,
independently of the scheduler's own code.
"""
import itertools
import math

import numpy as np
import pytest

from oracle import ref_scheduler as rs


def drain(s, iter_us=1000, max_iters=100000):
    """Run to completion with a constant iteration time; return all batches."""
    t, batches = 0, []
    for _ in range(max_iters):
        if not s.has_work():
            return batches
        b = s.next(t)
        if not b:
            nxt = s.next_arrival_us()
            assert nxt > t, "nothing runnable and nothing arriving: deadlock"
            t = nxt
            continue
        batches.append((t, b))
        s.commit(iter_us)
        t += iter_us
    raise AssertionError("did not drain")


# ---- (1) Eq. 3: ordering by K equals ordering by P_i(t) for any t --------------------
@pytest.mark.parametrize("seed", range(3))
def test_key_order_equals_priority_order(seed):
    rng = np.random.default_rng(seed)
    alpha, beta = 100.0, -1.0
    s = rs.RefScheduler(rs.SchedConfig(alpha=alpha, beta=beta, B_max=64, S_max=0, num_blocks=4096))
    reqs = [(i, int(rng.integers(0, 5_000_000)), int(rng.integers(1, 3000))) for i in range(40)]
    for i, a, r in reqs:
        s.add_request(i, a, r, 1)
    assert s.next(10_000_000) == []     # S_max = 0: arrivals are queued, nothing is scheduled
    popped = [e[2] for e in sorted(s.heap)]          # heap pop order (total order)
    for t in (5.0, 77.7, 1e4):
        P = {i: alpha * (t - a * 1e-6) + beta * r for i, a, r in reqs}     # Eq. 1
        order = sorted(P, key=lambda i: -P[i])
        gaps = np.diff(sorted(P.values()))
        assert gaps.min() > 1e-6          # keys well separated: rounding cannot reorder
        assert order == popped


# ---- (2) limits: beta = 0 -> FCFS, alpha = 0 -> shortest remaining first -------------
def _first_service_order(alpha, beta, reqs, B_max=64):
    s = rs.RefScheduler(rs.SchedConfig(alpha=alpha, beta=beta, B_max=B_max, num_blocks=8192))
    for i, a, p in reqs:
        s.add_request(i, a, p, 1)
    order = []
    for _, b in drain(s):
        for rid, q_len, off, _ in b:
            if rid not in order:
                order.append(rid)
    return order


def test_beta_zero_is_fcfs_and_alpha_zero_is_srpt():
    rng = np.random.default_rng(7)
    reqs = [(i, 0 if i < 30 else 1, int(rng.integers(65, 900))) for i in range(30)]
    arr = rng.permutation(30)
    reqs = [(i, int(arr[i]), p) for i, _, p in reqs]           # distinct arrivals, all <= 29 us
    # all have arrived before the 2nd round; service order after the first round is the policy's
    fcfs = _first_service_order(1.0, 0.0, reqs)
    assert fcfs == [i for i, a, p in sorted(reqs, key=lambda x: x[1])]
    srpt = _first_service_order(0.0, -1.0, [(i, 0, p) for i, a, p in reqs])
    assert srpt == [i for i, a, p in sorted(reqs, key=lambda x: (x[2], x[0]))]


# ---- (3) closed-form overtake time (from Eq. 1) ---------------------------------------
@pytest.mark.parametrize("extra_wait_us,old_first", [(1_900_000, False), (2_100_000, True)])
def test_overtake_threshold(extra_wait_us, old_first):
    # old: r = 300, newcomer: r' = 100 -> old wins iff alpha * extra_wait > |beta| (r - r')
    # alpha = 100 /s, beta = -1: threshold = 200 / 100 = 2.0 s
    s = rs.RefScheduler(rs.SchedConfig(alpha=100.0, beta=-1.0, B_max=50, num_blocks=1024))
    s.add_request(1, 0, 300, 1)
    s.add_request(2, extra_wait_us, 100, 1)
    b = s.next(extra_wait_us)
    assert b[0][0] == (1 if old_first else 2)


def test_tie_break_earlier_arrival_then_smaller_id():
    s = rs.RefScheduler(rs.SchedConfig(alpha=0.0, beta=-1.0, B_max=10, num_blocks=1024))
    s.add_request(9, 5, 100, 1)
    s.add_request(3, 5, 100, 1)
    s.add_request(4, 2, 100, 1)
    assert s.next(10)[0][0] == 4
    s.commit(1)
    # req 4 now has r = 90 -> best key; after it the tie (3 vs 9) goes to the smaller id
    s2 = rs.RefScheduler(rs.SchedConfig(alpha=0.0, beta=-1.0, B_max=10, num_blocks=1024))
    s2.add_request(9, 5, 100, 1)
    s2.add_request(3, 5, 100, 1)
    assert s2.next(10)[0][0] == 3


# ---- (4) conservation laws on random traces -------------------------------------------
@pytest.mark.parametrize("mode,apc", [(rs.MODE_TOKEN_BUDGET, False), (rs.MODE_LPRS, False),
                                      (rs.MODE_LPRS, True), (rs.MODE_TOKEN_BUDGET, True)])
def test_conservation(mode, apc):
    rng = np.random.default_rng(11)
    w = [0.0] * 16
    w[11], w[12], w[14], w[15] = 50.0, 0.4, 0.002, 1e-5      # bias, tokens, decode ctx, prefill
    cfg = rs.SchedConfig(B_max=256, S_max=24, mode=mode, apc=apc, Delta=32, T_star=120.0,
                         C_max=3, L_min=16, num_blocks=600, pred_weights=w)
    s = rs.RefScheduler(cfg)
    meta = {}
    t = 0
    for i in range(120):
        t += int(rng.exponential(3000))
        p, o = int(rng.integers(1, 1200)), int(rng.integers(1, 40))
        s.add_request(i, t, p, o)
        meta[i] = (t, p, o)
    batches = drain(s, iter_us=2500)
    got_prefill = {i: 0 for i in meta}
    got_decode = {i: 0 for i in meta}
    live_decodes = set()
    for now, b in batches:
        assert sum(q for _, q, _, _ in b) <= cfg.B_max                 # hard token budget
        assert len(b) <= cfg.S_max
        kinds = [got_prefill[rid] >= meta[rid][1] for rid, _, _, _ in b]
        assert kinds == sorted(kinds, reverse=True)                     # decodes first
        dec_in_batch = [rid for rid, *_ in b if got_prefill[rid] >= meta[rid][1]]
        assert dec_in_batch == sorted(dec_in_batch, key=lambda r: (meta[r][0], r))
        if len(live_decodes) <= min(cfg.B_max, cfg.S_max):
            assert set(dec_in_batch) == live_decodes                    # every runnable decode
        pages_seen = set()
        for rid, q_len, off, pages in b:
            a, p, o = meta[rid]
            assert a <= now
            assert len(pages) * cfg.block_size >= off + q_len
            assert not (pages_seen & set(pages))
            pages_seen |= set(pages)
            if got_prefill[rid] < p:
                assert off == got_prefill[rid] and 1 <= q_len <= p - off   # Eq. 2 / Eq. 6
                got_prefill[rid] += q_len
                if got_prefill[rid] == p and o > 1:
                    live_decodes.add(rid)
            else:
                assert q_len == 1 and off == p + got_decode[rid]
                got_decode[rid] += 1
                if got_decode[rid] == o - 1:
                    live_decodes.discard(rid)
    for i, (a, p, o) in meta.items():
        assert got_prefill[i] == p and got_decode[i] == o - 1
        assert s.reqs[i].phase == "done" and s.reqs[i].ttft_us >= a
    assert s.used_pages == 0 and sorted(s.free_pages) == list(range(cfg.num_blocks))
    if not apc:
        assert s.blocked_by_activity_cap == 0 and s.blocked_by_min_chunk == 0


# ---- (5) Algorithm 1 ------------------------------------------------------------------
def _lprs(T_star, w_bias, w_tok, lam_u=1.0, lam_o=2.0, Delta=64, B_max=2048):
    w = [0.0] * 16
    w[11], w[0] = w_bias, w_tok          # T_hat = u + w * prefill_tokens
    return rs.RefScheduler(rs.SchedConfig(mode=rs.MODE_LPRS, T_star=T_star, lambda_u=lam_u,
                                          lambda_o=lam_o, Delta=Delta, B_max=B_max,
                                          pred_weights=w, num_blocks=64))


EMPTY = (0, 0, 0, 0, 0, 0, 0)


def test_candidate_set_is_eq8():
    s = _lprs(0, 0, 0, Delta=64)
    assert s.candidates(1) == [1]
    assert s.candidates(63) == [1, 63]
    assert s.candidates(64) == [1, 64]
    assert s.candidates(200) == [1, 64, 128, 192, 200]
    assert rs.RefScheduler(rs.SchedConfig(Delta=1, num_blocks=4)).candidates(5) == [1, 2, 3, 4, 5]


@pytest.mark.parametrize("seed", range(5))
def test_alg1_equals_bruteforce_argmin(seed):
    rng = np.random.default_rng(seed)
    u, w = float(rng.uniform(10, 60)), float(rng.uniform(0.05, 0.4))
    T_star = float(rng.uniform(20, 200))
    lam_u, lam_o = 1.0, float(rng.uniform(1.1, 4))
    Delta = int(rng.integers(1, 100))
    s = _lprs(T_star, u, w, lam_u, lam_o, Delta)
    for r_i, U_t in [(5000, 0), (300, 1900), (77, 10), (1, 0), (2048, 2047)]:
        h = min(r_i, 2048 - U_t)
        cands = sorted({1, h} | {k * Delta for k in range(1, h // Delta + 1)})

        def score(c):
            T = 0.0 + u * 1.0
            T = u + w * c            # only bias and prefill_tokens carry weight
            return lam_u * (T_star - T) if T <= T_star else lam_o * (T - T_star)
        best = min(score(c) for c in cands)
        # allow for the fixed-order fp64 sum of the 16-term dot product
        want = max(c for c in cands if abs(score(c) - best) <= 1e-9)
        got = s.select_chunk(r_i, 0, U_t, EMPTY)
        assert abs(score(got) - best) <= 1e-9 and got == want


def test_alg1_closed_form_linear_symmetric_delta1():
    """f(c) = u + w c, lambda_u = lambda_o, Delta = 1: c* = clamp(nearest int to
    (T* - u)/w, 1, h), exact ties to the larger c.  Dyadic numbers keep fp64 exact."""
    u, w = 16.0, 0.25
    for T_star, h, want in [(48.0, 500, 128), (48.125, 500, 129), (48.0625, 500, 128),
                            (48.1875, 500, 129), (1000.0, 500, 500), (3.0, 500, 1),
                            (48.0, 100, 100)]:
        s = _lprs(T_star, u, w, 1.0, 1.0, Delta=1)
        assert s.select_chunk(h, 0, 0, EMPTY) == want
    # exact tie between 128 and 129 -> larger
    s = _lprs(16.0 + 0.25 * 128.5, u, w, 1.0, 1.0, Delta=1)
    assert s.select_chunk(500, 0, 0, EMPTY) == 129


def test_alg1_overflow_penalised_not_forbidden_and_guard():
    # every candidate overflows: the smallest overflow (c = 1) wins
    s = _lprs(5.0, 10.0, 1.0)
    assert s.select_chunk(500, 0, 0, EMPTY) == 1
    # NaN predictor: no finite score -> c* = 0 -> starvation guard returns 1 on an empty batch
    s = _lprs(5.0, float("nan"), 1.0)
    assert s.select_chunk(500, 0, 0, EMPTY) == 1
    assert s.select_chunk(500, 0, 7, EMPTY) == 0          # batch not empty: skipped
    assert s.select_chunk(500, 0, 2048, EMPTY) == 0       # h <= 0


def test_features_tables_1_and_2():
    s = rs.RefScheduler(rs.SchedConfig(num_blocks=100, page_mb=2.0))
    s.used_pages = 30
    x = s.features(n_dec=4, sum_ctx=1000, max_ctx=400, pf_tokens=96, n_pf=2, pf_proc=640,
                   pf_proc_max=512)
    want = dict(prefill_tokens=96, decode_tokens=4, batch_request_count=6,
                sum_decode_context_len=1000, max_decode_context_len=400,
                prefill_processed_tokens=640, max_prefill_processed_tokens=512,
                gpu_mem_used_mb=60, gpu_mem_free_mb=140, cuda_allocated_mb=60,
                cuda_reserved_mb=200, bias=1, scheduled_tokens=100, avg_decode_ctx=250,
                decode_ctx_interaction=1000, prefill_interaction=96 * 640)
    assert x == [float(want[n]) for n in rs.FEATURE_NAMES]
    assert s.features(0, 0, 0, 5, 1, 0, 0)[13] == 0.0        # max(decode_tokens, 1)


def test_mlp_predictor_matches_numpy():
    rng = np.random.default_rng(3)
    n = rs.mlp_num_weights()
    w = rng.standard_normal(n) * 0.2
    mu, inv = rng.standard_normal(16), rng.uniform(0.5, 2, 16)
    s = rs.RefScheduler(rs.SchedConfig(pred_kind=rs.PRED_MLP, pred_weights=list(w),
                                       feat_mu=list(mu), feat_inv_sigma=list(inv), num_blocks=4))
    x = rng.standard_normal(16) * 3
    z, pos = (x - mu) * inv, 0
    for li in range(4):
        i, o = rs.MLP_DIMS[li], rs.MLP_DIMS[li + 1]
        W = w[pos:pos + o * i].reshape(o, i); b = w[pos + o * i:pos + o * i + o]; pos += o * i + o
        z = W @ z + b
        if li < 3:
            z = np.maximum(z, 0)
    assert abs(s.predict(list(x)) - z[0]) <= 1e-12 * max(1, abs(z[0]))


# ---- (6) Eq. 12-14 against a literal transcription, exhaustive grid ---------------------
def test_apc_exhaustive():
    C_max, S_max, B_max, L_min = 3, 6, 40, 8
    s = rs.RefScheduler(rs.SchedConfig(apc=True, C_max=C_max, S_max=S_max, B_max=B_max,
                                       L_min=L_min, num_blocks=4))
    for D_t, U_extra in itertools.product(range(0, 7), range(0, 34, 3)):
        U_t = D_t + U_extra
        if U_t > B_max:
            continue
        C_t = min(C_max, S_max - D_t, math.floor((B_max - U_t) / L_min))      # Eq. 12
        assert s.activity_cap(D_t, U_t) == C_t
        for r_i, P_size in itertools.product([1, 3, 8, 9, 30, 100], range(0, 5)):
            h_i = min(r_i, B_max - U_t)
            if h_i <= 0:
                continue
            for c_star in range(0, h_i + 1):
                m_i = min(r_i, L_min)                                          # Eq. 13
                if P_size < C_t and c_star >= m_i:                             # Eq. 14
                    want = c_star
                elif c_star < m_i and P_size == 0:
                    want = min(h_i, m_i)
                else:
                    want = 0
                got = s.apc_decision(c_star, r_i, h_i, P_size, C_t)
                assert got == want and got in (0, c_star, min(h_i, m_i))


def test_apc_counters_and_fragmentation_control():
    """Many short prompts, tiny residual budget: APC keeps few meaningful prefills active
    (fewer scheduled prefill sequences, larger chunks) and counts blocks."""
    def run(apc):
        cfg = rs.SchedConfig(B_max=64, S_max=64, apc=apc, C_max=2, L_min=16, num_blocks=4096)
        s = rs.RefScheduler(cfg)
        for i in range(60):
            s.add_request(i, i * 10, 40, 30)
        b = drain(s, iter_us=500)
        n_pf = [sum(1 for rid, q, off, _ in bb if off < 40) for _, bb in b]
        return s, float(np.mean(n_pf))
    s_off, mean_off = run(False)
    s_on, mean_on = run(True)
    assert s_off.blocked_by_activity_cap == 0 and s_off.blocked_by_min_chunk == 0
    assert s_on.blocked_by_activity_cap + s_on.blocked_by_min_chunk > 0
    assert mean_on <= mean_off


def test_pool_exhaustion_sets_requests_aside_without_deadlock():
    cfg = rs.SchedConfig(B_max=128, num_blocks=20, block_size=16)     # 320 token slots
    s = rs.RefScheduler(cfg)
    for i in range(6):
        s.add_request(i, 0, 100, 50)            # 10 pages each: only two fit at a time
    b = drain(s, iter_us=100)
    live = set()
    for _, bb in b:
        assert len({rid for rid, *_ in bb}) <= 2
    assert all(r.phase == "done" for r in s.reqs.values())
    with pytest.raises(ValueError):
        s.add_request(99, 0, 400, 1)            # can never fit


def test_edge_prompts_of_one_token_and_output_len_one():
    s = rs.RefScheduler(rs.SchedConfig(B_max=8, num_blocks=64))
    s.add_request(1, 0, 1, 1)
    s.add_request(2, 0, 1, 3)
    s.add_request(3, 0, 20, 1)
    b = drain(s, iter_us=10)
    assert s.reqs[1].finish_us == s.reqs[1].ttft_us == 10
    assert s.reqs[2].finish_us == 30
    assert [x[:3] for x in b[0][1]] == [(1, 1, 0), (2, 1, 0), (3, 6, 0)]
