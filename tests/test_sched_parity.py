"""libcp's C++ scheduler vs the independent Python reference: batch composition must be
bit-exact on every iteration (BASELINE.json north_star; SURVEY.md 8(c2) pin 7)."""
import hashlib

import numpy as np
import pytest

from oracle import ref_scheduler as rs
from paper_2606_09061_b200 import binding, build, workloads as wl


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()


def iter_us_model(batch):
    """Deterministic stand-in for the measured iteration time (integer us)."""
    tokens = sum(b[1] for b in batch)
    ctx = sum(b[2] + b[1] for b in batch)
    return 40 + (tokens * 3) // 10 + ctx // 700


def run_both(trace, max_iters=400000, **kw):
    ref = rs.RefScheduler(rs.SchedConfig(**kw))
    cpp = binding.Scheduler(**{**kw, "max_batch": max(kw.get("S_max", 1024), 1)})
    for rid, a, p, o in zip(*trace):
        ref.add_request(int(rid), int(a), int(p), int(o))
        cpp.cp_sched_add_request(int(rid), int(a), int(p), int(o))
    t, n_it = 0, 0
    h_ref, h_cpp = hashlib.sha256(), hashlib.sha256()
    while ref.has_work():
        assert cpp.cp_sched_has_work()
        b_ref = ref.next(t)
        n = cpp.cp_sched_next(t)
        b_cpp = cpp.batch()
        assert b_cpp == b_ref, f"iteration {n_it} at t={t} differs"
        h_ref.update(rs.pack_record(b_ref))
        h_cpp.update(rs.pack_record(b_cpp))
        if not b_ref:
            nxt = ref.next_arrival_us()
            assert nxt == cpp.cp_sched_next_arrival() and nxt > t
            t = nxt
            continue
        dt = iter_us_model(b_ref)
        ref.commit(dt)
        cpp.cp_sched_commit(dt)
        t += dt
        n_it += 1
        assert n_it < max_iters
    assert not cpp.cp_sched_has_work()
    assert h_ref.digest() == h_cpp.digest()
    st = cpp.cp_sched_get_stats()
    assert st.n_iters == ref.n_iters == n_it
    assert st.blocked_by_activity_cap == ref.blocked_by_activity_cap
    assert st.blocked_by_min_chunk == ref.blocked_by_min_chunk
    assert st.used_pages == ref.used_pages == 0
    for rid in trace[0]:
        assert cpp.cp_sched_request_times(int(rid)) == (ref.reqs[int(rid)].ttft_us, ref.reqs[int(rid)].finish_us)
    return ref, n_it


LIN_W = [0.0] * 16
LIN_W[11], LIN_W[12], LIN_W[14], LIN_W[15], LIN_W[7] = 37.5, 0.31, 0.0021, 1.3e-5, 0.01


def small_trace(seed, n=150, rate=400.0):
    return wl.make_trace(n, rate_per_s=rate, seed=seed, short_median=120, long_lo=600, long_hi=2500,
                         out_median=12, out_max=60)


@pytest.mark.parametrize("seed", range(3))
def test_token_budget_aging(seed):
    run_both(small_trace(seed), alpha=100.0, beta=-1.0, B_max=256, S_max=32, num_blocks=2000)


@pytest.mark.parametrize("alpha,beta", [(1.0, 0.0), (0.0, -1.0), (500.0, -1.0), (0.37, -0.011)])
def test_policy_limits(alpha, beta):
    run_both(small_trace(5), alpha=alpha, beta=beta, B_max=128, S_max=16, num_blocks=1500)


@pytest.mark.parametrize("apc", [False, True])
def test_lprs_linear(apc):
    ref, _ = run_both(small_trace(7), B_max=512, S_max=48, mode=rs.MODE_LPRS, apc=apc, Delta=32,
                      T_star=120.0, lambda_u=1.0, lambda_o=2.5, C_max=3, L_min=24, num_blocks=2500,
                      page_mb=0.0625, pred_weights=LIN_W)
    if apc:
        assert ref.blocked_by_activity_cap + ref.blocked_by_min_chunk > 0


def test_lprs_mlp_with_normalisation():
    rng = np.random.default_rng(0)
    w = (rng.standard_normal(rs.mlp_num_weights()) * 0.15).tolist()
    mu = [100, 8, 10, 4000, 900, 500, 400, 30, 90, 30, 120, 0, 110, 500, 4000, 50000]
    inv = [1 / 120, 1 / 8, 1 / 9, 1 / 3000, 1 / 700, 1 / 600, 1 / 500, 1 / 20, 1 / 40, 1 / 20, 1.0, 1.0,
           1 / 100, 1 / 300, 1 / 3000, 1 / 60000]
    run_both(small_trace(9, n=60), B_max=256, S_max=32, mode=rs.MODE_LPRS, apc=True, Delta=16,
             T_star=0.4, C_max=2, L_min=16, num_blocks=1200, pred_kind=rs.PRED_MLP,
             pred_weights=w, feat_mu=mu, feat_inv_sigma=inv)


def test_predictor_and_alg1_pure_functions_agree():
    rng = np.random.default_rng(1)
    kw = dict(B_max=2048, mode=rs.MODE_LPRS, Delta=64, T_star=300.0, lambda_o=3.0, num_blocks=512,
              pred_weights=LIN_W)
    ref = rs.RefScheduler(rs.SchedConfig(**kw))
    cpp = binding.Scheduler(**kw)
    for _ in range(200):
        x = (rng.standard_normal(16) * rng.choice([1.0, 100.0, 1e4])).tolist()
        assert cpp.cp_sched_predict(x) == ref.predict(x)           # bit-exact fp64
        r_i, U_t = int(rng.integers(1, 5000)), int(rng.integers(0, 2048))
        st = (int(rng.integers(0, 200)), int(rng.integers(0, 10 ** 6)), int(rng.integers(0, 40000)),
              int(rng.integers(0, 600)), int(rng.integers(0, 5)), int(rng.integers(0, 60000)),
              int(rng.integers(0, 30000)))
        ctx_i = int(rng.integers(0, 30000))
        assert cpp.cp_sched_select_chunk(r_i, ctx_i, U_t, *st) == ref.select_chunk(r_i, ctx_i, U_t, st)


def test_adversarial_traces():
    ids = np.arange(40, dtype=np.int64)
    same = (ids, np.zeros(40, np.int64), np.full(40, 77, np.int64), np.full(40, 5, np.int64))
    run_both(same, B_max=100, S_max=12, num_blocks=400)                      # simultaneous, equal
    ones = (ids, ids * 3, np.ones(40, np.int64), np.ones(40, np.int64))
    run_both(ones, B_max=4, S_max=4, num_blocks=64)                          # 1-token prompts, output 1
    tight = (ids, ids * 10, np.full(40, 300, np.int64), np.full(40, 40, np.int64))
    run_both(tight, B_max=128, S_max=64, num_blocks=50)                      # pool exhaustion
    many_dec = (ids, np.zeros(40, np.int64), np.full(40, 3, np.int64), np.full(40, 30, np.int64))
    run_both(many_dec, B_max=16, S_max=8, num_blocks=400)                    # decodes exceed the limits


def test_apc_ablation_shape():
    tr = wl.make_apc_trace(400, seed=2)
    run_both(tr, B_max=96, S_max=64, mode=rs.MODE_LPRS, apc=True, Delta=8, T_star=70.0, C_max=2,
             L_min=16, num_blocks=4000, pred_weights=LIN_W)


def test_config5_trace_bit_exact():
    """configs[4]: 1000 requests, Poisson 8 req/s, aging with budget 2048, alpha 100, beta -1."""
    tr = wl.make_trace(1000, rate_per_s=8.0, seed=0)
    _, n_it = run_both(tr, alpha=100.0, beta=-1.0, B_max=2048, S_max=1024, num_blocks=20480,
                       max_iters=2_000_000)
    assert n_it > 10000


def test_trace_run_record_packing_matches_reference_packing():
    """trace_run hashes the C descriptors directly (pack_batch); the reference replay hashes
    pack_record of Python tuples: the two encodings must be byte-identical."""
    from paper_2606_09061_b200 import trace_run
    kw = dict(alpha=100.0, beta=-1.0, B_max=64, S_max=8, num_blocks=256)
    cpp = binding.Scheduler(**{**kw, "max_batch": 8})
    for rid, (a, p, o) in enumerate([(0, 70, 3), (5, 9, 2), (9, 130, 4)]):
        cpp.cp_sched_add_request(rid, a, p, o)
    t = 0
    for _ in range(6):
        n = cpp.cp_sched_next(t)
        assert trace_run.pack_batch(cpp.descs, n) == rs.pack_record(cpp.batch())
        if n == 0:
            break
        cpp.cp_sched_commit(50)
        t += 50
