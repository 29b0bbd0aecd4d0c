"""-m gpu: the trace-driven run (BASELINE.json configs[4], reduced) -- the C++ scheduler forms
every iteration, libcp runs it on the GPU for every layer, and
  * sampled iterations are checked against the fp64 oracle (layers 0 and last),
  * the KV pages the step wrote equal the oracle's append,
  * the schedule is bit-identical to the reference scheduler replayed on the measured times.
configs[4] at its full shape (1000-request trace, 32 layers, 20,480 pages per layer = 40 GiB, budget 2048) runs
un-gated for its first 400 iterations with an oracle sample every 50th iteration on layers 0 and 31 (SURVEY.md
8(d)); CP_FULL_TRACE=1 additionally runs it to the end.  The LPRS / APC loop (harvest -> train -> schedule) runs
un-gated on a reduced model with the whole-forward-pass clock; CP_FULL_TRACE=1 runs the long version."""
import hashlib
import json
import os

import numpy as np
import pytest

from oracle import attention as ora
from oracle import ref_scheduler as rs
from oracle import rope as orope
from paper_2606_09061_b200 import binding, build, trace_run, workloads as wl
from tests import gpu_util as gu

pytestmark = pytest.mark.gpu


def replay_reference(trace, iter_us_log, truncated=False, **kw):
    """Reference scheduler fed the SAME measured iteration times; returns its schedule digest.
    truncated: the run stopped after len(iter_us_log) iterations (max_iters) -- stop at the same point."""
    ref = rs.RefScheduler(rs.SchedConfig(**kw))
    for rid, a, p, o in zip(*trace):
        ref.add_request(int(rid), int(a), int(p), int(o))
    h, t, i = hashlib.sha256(), 0, 0
    while ref.has_work() and i <= len(iter_us_log):
        if truncated and i == len(iter_us_log):
            break
        b = ref.next(t)
        h.update(rs.pack_record(b))
        if not b:
            t = ref.next_arrival_us()
            continue
        if i == len(iter_us_log):
            break
        ref.commit(iter_us_log[i])
        t += iter_us_log[i]
        i += 1
    return h.hexdigest(), i


def make_parity_hook(Hq, Hkv, D, B, layers, every, n_rows, stats, scale, inv_freq=None, max_reqs=None):
    """max_reqs: check only a seeded subset of the iteration's requests (their pages and rows) -- what makes an oracle
    sample every 50th iteration affordable on the full configs[4] trace (a long-context batch touches > 1 GB of pages
    per layer)."""
    def hook(it, batch, layer_tensors):
        if it % every:
            return
        import torch
        q_all = np.array([b[1] for b in batch], np.int64)
        cu = np.concatenate([[0], np.cumsum(q_all)])
        sel = np.arange(len(batch))
        if max_reqs is not None and len(batch) > max_reqs:
            sel = np.sort(np.random.default_rng(it).choice(len(batch), size=max_reqs, replace=False))
        q_len = np.array([batch[j][1] for j in sel], np.int32)
        ctx_off = np.array([batch[j][2] for j in sel], np.int32)
        used = [(int(c) + int(q) + B - 1) // B for q, c in zip(q_len, ctx_off)]
        tables = [np.asarray(batch[j][3][:u], np.int32) for j, u in zip(sel, used)]
        spec = wl.BatchSpec(f"it{it}", Hq, Hkv, D, B, 0, q_len, ctx_off, tables)
        rows_of = np.concatenate([np.arange(cu[j], cu[j + 1]) for j in sel])          # token rows of the selected requests
        touched = torch.from_numpy(spec.touched_pages().astype(np.int64)).cuda()
        tok, head = gu.sample_rows(spec, n_rows, seed=it)
        for l in sorted({0, layers - 1}):
            q, k_new, v_new, pool_l, out_l = layer_tensors(l)
            cache = gu.to_bits(pool_l[touched])                       # AFTER the step's append
            before = cache.copy()
            q_bits, k_bits, v_bits = gu.to_bits(q)[rows_of], gu.to_bits(k_new)[rows_of], gu.to_bits(v_new)[rows_of]
            if inv_freq is not None:                                  # the step rotated Q and the new K rows
                pos = orope.token_positions(q_len, ctx_off)
                q_bits, k_bits = orope.rope_bf16(q_bits, pos, inv_freq), orope.rope_bf16(k_bits, pos, inv_freq)
            ora.kv_append(k_bits, v_bits, cache, q_len, ctx_off, spec.compact_tables())
            if inv_freq is None:
                assert np.array_equal(cache, before), "H2: GPU append differs from the oracle's"
            else:                                                     # DESIGN.md R12: fp64 cos / sin last place
                dk = np.abs(cache.astype(np.int32) - before.astype(np.int32))
                assert dk.max() <= 1 and (dk != 0).sum() <= 2 + 1e-5 * spec.T * Hkv * D
            want = ora.attention(q_bits, cache, q_len, ctx_off, spec.compact_tables(), scale, rows=(tok, head))
            got = wl.bf16_bits_to_f64(gu.to_bits(out_l)[rows_of]).reshape(spec.T, Hq, D)[tok, head]
            mx, mean = gu.assert_close(got, want, f"iteration {it} layer {l}")
            stats.append((it, l, mx, mean))
    return hook


def test_reduced_trace_parity_and_schedule_identity():
    build.build()
    Hq, Hkv, D, B, layers = 32, 8, 128, 16, 4
    trace = wl.make_trace(80, rate_per_s=2000.0, seed=3, short_median=200, long_lo=1500, long_hi=6000,
                          out_median=24, out_max=96)
    kw = dict(alpha=100.0, beta=-1.0, B_max=512, S_max=128, num_blocks=6144, block_size=B)
    stats = []
    scale = float(np.float32(1.0) / np.sqrt(np.float32(D)))
    hook = make_parity_hook(Hq, Hkv, D, B, layers, 9, 256, stats, scale)
    report, log = trace_run.run_trace(trace, Hq=Hq, Hkv=Hkv, D=D, B=B, layers=layers, pages_per_layer=6144,
                                      sched_kw=kw, seed=3, hook=hook)
    assert report["e2e_s"]["finished"] == 80 and report["ttft_s"]["started"] == 80
    assert report["iterations"] == len(log) > 100 and len(stats) >= 20
    assert report["iteration_us_by_class"]["mixed"]["iterations"] > 0
    kw_ref = dict(kw, page_mb=2 * Hkv * B * D * 2 * layers / 2**20)
    digest, n = replay_reference(trace, log, **kw_ref)
    assert n == len(log) and digest == report["schedule_sha256"]


def test_reduced_trace_with_rope():
    """The serving loop through cp_attention_step_rope: same schedule identity, parity against the
    rotated oracle on sampled iterations (pages carry rotated K from step to step)."""
    build.build()
    Hq, Hkv, D, B, layers = 32, 8, 128, 16, 2
    trace = wl.make_trace(40, rate_per_s=2000.0, seed=5, short_median=200, long_lo=1500, long_hi=6000,
                          out_median=24, out_max=96)
    kw = dict(alpha=100.0, beta=-1.0, B_max=512, S_max=128, num_blocks=6144, block_size=B)
    stats = []
    scale = float(np.float32(1.0) / np.sqrt(np.float32(D)))
    w = binding.rope_inv_freq(D, 500000.0)
    hook = make_parity_hook(Hq, Hkv, D, B, layers, 7, 256, stats, scale, inv_freq=w)
    report, log = trace_run.run_trace(trace, Hq=Hq, Hkv=Hkv, D=D, B=B, layers=layers, pages_per_layer=6144,
                                      sched_kw=kw, seed=5, hook=hook, rope_inv_freq=w)
    assert report["e2e_s"]["finished"] == 40 and len(stats) >= 10
    kw_ref = dict(kw, page_mb=2 * Hkv * B * D * 2 * layers / 2**20)
    digest, n = replay_reference(trace, log, **kw_ref)
    assert n == len(log) and digest == report["schedule_sha256"]


@pytest.mark.skipif(os.environ.get("CP_FULL_TRACE") != "1", reason="set CP_FULL_TRACE=1 (minutes, 40 GiB pool)")
def test_full_config5_trace():
    build.build()
    rate = float(os.environ.get("CP_TRACE_RATE", "8"))
    trace = wl.make_trace(1000, rate_per_s=rate, seed=0)
    stats = []
    scale = float(np.float32(1.0) / np.sqrt(np.float32(128)))
    # an oracle sample every 50th iteration, layers 0 and 31 (on up to 6 requests of the iteration)
    hook = make_parity_hook(32, 8, 128, 16, 32, int(os.environ.get("CP_TRACE_EVERY", "50")), 128, stats, scale, max_reqs=6)
    report, log = trace_run.run_trace(trace, hook=hook)
    kw = dict(alpha=100.0, beta=-1.0, B_max=2048, S_max=1024, num_blocks=20480, block_size=16,
              page_mb=2 * 8 * 16 * 128 * 2 * 32 / 2**20)
    digest, n = replay_reference(trace, log, **kw)
    report["arrival_rate_per_s"] = rate
    report["oracle_parity_samples"] = [{"iteration": s[0], "layer": s[1], "max_abs": s[2], "mean_abs": s[3]} for s in stats]
    report["reference_schedule_sha256"] = digest
    os.makedirs("gpurun_out", exist_ok=True)
    with open(f"gpurun_out/trace_config5_rate{int(rate)}.json", "w") as f:
        json.dump(report, f)
    assert report["e2e_s"]["finished"] == 1000
    assert n == len(log) and digest == report["schedule_sha256"]


def test_apc_ablation_shape_trace_on_gpu():
    """the APC ablation workload shape (49:1 short (30-50) : long (200-220)
    prompts, bursty arrivals) -- many tiny chunks per iteration -- through the whole path with LPRS + APC on,
    oracle parity on sampled iterations and schedule identity with the reference."""
    build.build()
    Hq, Hkv, D, B, layers = 32, 8, 128, 16, 2
    trace = wl.make_apc_trace(300, seed=2, mean_gap_us=8.0)          # arrivals faster than iterations: the queue has depth
    lin_w = [0.0] * 16
    lin_w[11], lin_w[12], lin_w[14], lin_w[15] = 8.0, 0.02, 0.0004, 1e-6          # us per layer: bias, tokens, decode ctx, prefill interaction
    kw = dict(alpha=100.0, beta=-1.0, B_max=96, S_max=64, mode=rs.MODE_LPRS, apc=True, Delta=8, T_star=11.0, C_max=2, L_min=16,
              num_blocks=4096, block_size=B, pred_weights=lin_w)
    stats = []
    scale = float(np.float32(1.0) / np.sqrt(np.float32(D)))
    hook = make_parity_hook(Hq, Hkv, D, B, layers, 25, 128, stats, scale)
    report, log = trace_run.run_trace(trace, Hq=Hq, Hkv=Hkv, D=D, B=B, layers=layers, pages_per_layer=4096,
                                      sched_kw=kw, seed=2, hook=hook)
    assert report["e2e_s"]["finished"] == 300 and len(stats) >= 10
    assert report["blocked_by_activity_cap"] + report["blocked_by_min_chunk"] > 0      # APC intervened (Table 10 counters)
    kw_ref = dict(kw, page_mb=2 * Hkv * B * D * 2 * layers / 2**20)
    digest, n = replay_reference(trace, log, **kw_ref)
    assert n == len(log) and digest == report["schedule_sha256"]


def test_reduced_trace_with_layer_gemms():
    """the same loop with the dense projections of every layer (library GEMMs on seeded random
    weights) inside the timed iteration; the schedule must still equal the reference replay on the measured times,
    and iterations must take longer than the attention steps alone."""
    build.build()
    Hq, Hkv, D, B, layers = 32, 8, 128, 16, 2
    trace = wl.make_trace(40, rate_per_s=2000.0, seed=4, short_median=200, long_lo=1500, long_hi=4000, out_median=16, out_max=48)
    kw = dict(alpha=100.0, beta=-1.0, B_max=512, S_max=128, num_blocks=4096, block_size=B)
    rep0, log0 = trace_run.run_trace(trace, Hq=Hq, Hkv=Hkv, D=D, B=B, layers=layers, pages_per_layer=4096, sched_kw=kw, seed=4)
    rep1, log1 = trace_run.run_trace(trace, Hq=Hq, Hkv=Hkv, D=D, B=B, layers=layers, pages_per_layer=4096, sched_kw=kw, seed=4,
                                     layer_gemms=True)
    assert rep1["e2e_s"]["finished"] == 40
    assert np.mean(log1) > np.mean(log0)
    digest, n = replay_reference(trace, log1, **dict(kw, page_mb=2 * Hkv * B * D * 2 * layers / 2**20))
    assert n == len(log1) and digest == rep1["schedule_sha256"]


def test_config5_full_shape_first_iterations():
    """BASELINE.json configs[4] at full shape -- 8B attention shape x 32 layers, 20,480 pages per layer (40 GiB
    pool), 1000-request trace at 8 req/s, aging scheduler with budget 2048 -- for its first 400 iterations: oracle
    parity every 50th iteration on layers 0 and 31, schedule identity with the reference replay,
    and the trace-level roofline fields of the report."""
    build.build()
    trace = wl.make_trace(1000, rate_per_s=8.0, seed=0)
    stats = []
    scale = float(np.float32(1.0) / np.sqrt(np.float32(128)))
    hook = make_parity_hook(32, 8, 128, 16, 32, 50, 128, stats, scale)
    report, log = trace_run.run_trace(trace, hook=hook, max_iters=400)
    assert len(log) == 400 and len(stats) == 2 * 8 and {s[1] for s in stats} == {0, 31}
    kw = dict(alpha=100.0, beta=-1.0, B_max=2048, S_max=1024, num_blocks=20480, block_size=16,
              page_mb=2 * 8 * 16 * 128 * 2 * 32 / 2**20)
    digest, n = replay_reference(trace, log, truncated=True, **kw)
    assert n == 400 and digest == report["schedule_sha256"]
    roof = report["attention_roofline_by_class"]
    assert roof["all"]["algorithmic_bytes"] > 0 and 0 < roof["all"]["frac_of_hbm_peak"] < 1.2
    os.makedirs("gpurun_out", exist_ok=True)
    report["oracle_parity_samples"] = [{"iteration": s[0], "layer": s[1], "max_abs": s[2], "mean_abs": s[3]} for s in stats]
    with open("gpurun_out/trace_config5_first400.json", "w") as f:
        json.dump(report, f)


def _lprs_loop(n_harvest, epochs, layers, n_requests, rate, max_iters, pages_per_layer, out_name):
    """SURVEY.md 8(f) N1 on the N3 clock: harvest whole-forward-pass times (attention of every layer + dense GEMM
    filler) through the serving loop's own IterationRunner, train the Table-7 MLP, take T* = the median time of the
    full-budget rounds, then run the trace under token budget / LPRS / LPRS + APC with that predictor; every schedule
    must equal the reference scheduler's replay on the measured times (same predictor data on both sides)."""
    from paper_2606_09061_b200 import predictor as pr
    build.build()
    raw, us = pr.harvest(n_harvest, seed=0, layers=layers, layer_gemms=True, pages_per_layer=65536, repeats=2)
    rep, lin, mlp = pr.train_and_report(raw, us, seed=0, epochs=epochs)
    X = pr.features16(raw)
    t_star = float(np.median(us[X[:, 12] >= 2000]))           # a typical full-budget round (T* is a whole-iteration time)
    trace = wl.make_trace(n_requests, rate_per_s=rate, seed=0)
    kind, w, mu, inv = pr.export_mlp(mlp)
    base = dict(alpha=100.0, beta=-1.0, B_max=2048, S_max=1024, num_blocks=pages_per_layer, block_size=16,
                page_mb=2 * 8 * 16 * 128 * 2 * layers / 2**20)
    lprs = dict(base, mode=rs.MODE_LPRS, Delta=64, T_star=t_star, lambda_u=1.0, lambda_o=2.0, C_max=4, L_min=64,
                pred_kind=kind, pred_weights=w, feat_mu=mu, feat_inv_sigma=inv)
    out = {"predictor": rep, "T_star_us": t_star, "arrival_rate_per_s": rate, "layers": layers,
           "clock": "whole forward pass (attention + dense GEMM filler)", "runs": {}}
    for name, kw in [("token_budget", base), ("lprs", lprs), ("lprs_apc", dict(lprs, apc=True))]:
        report, log = trace_run.run_trace(trace, layers=layers, pages_per_layer=pages_per_layer, sched_kw=kw,
                                          layer_gemms=True, max_iters=max_iters)
        digest, n = replay_reference(trace, log, truncated=max_iters is not None, **kw)
        assert n == len(log) and digest == report["schedule_sha256"], name
        it = np.asarray(log, np.float64)
        report["iteration_us"] = {"mean": float(it.mean()), "p50": float(np.percentile(it, 50)), "p95": float(np.percentile(it, 95)),
                                  "p99": float(np.percentile(it, 99)), "max": float(it.max()), "frac_over_T_star": float((it > t_star).mean()),
                                  "mean_abs_dev_from_T_star_of_mixed": None}
        report.pop("sched", None)
        out["runs"][name] = report
    os.makedirs("gpurun_out", exist_ok=True)
    with open(f"gpurun_out/{out_name}", "w") as f:
        json.dump(out, f)
    return out


def test_lprs_apc_loop_on_the_whole_iteration_clock():
    """Bounded version for every run: 300 harvested rounds, 30 epochs, a 4-layer model, 120 requests at 200 req/s, 500
    iterations per mode.  Latency control ("minimizing deviation from a target latency budget"): LPRS
    pulls the tail of the iteration time towards T*."""
    out = _lprs_loop(300, 30, 4, 120, 200.0, 500, 20480, "lprs_report_bounded.json")
    tb, lp = out["runs"]["token_budget"]["iteration_us"], out["runs"]["lprs"]["iteration_us"]
    # (measured margins are thin on this bounded run -- p95 6793 against 6852 us -- and iteration times jitter by a few
    # per cent from box to box: the tail must not get worse by more than that jitter, and fewer rounds may exceed T*)
    assert lp["p95"] <= tb["p95"] * 1.05 and lp["max"] <= tb["max"] * 1.10
    assert lp["frac_over_T_star"] <= tb["frac_over_T_star"] + 0.02
    assert out["predictor"]["mlp_test"]["mape_pct"] < 30.0


@pytest.mark.skipif(os.environ.get("CP_FULL_TRACE") != "1", reason="set CP_FULL_TRACE=1 (long: 32 layers with GEMM filler)")
def test_lprs_apc_loop_long():
    out = _lprs_loop(int(os.environ.get("CP_HARVEST", "2500")), int(os.environ.get("CP_EPOCHS", "300")), 32, 1000,
                     float(os.environ.get("CP_TRACE_RATE", "8")), None, 20480, "lprs_report.json")
    assert out["predictor"]["mlp_test"]["mape_pct"] < 10.0


def test_sharegpt_like_short_context_trace():
    """the paper's short-context mix (prompt median 19, P90 179, max context 512,
    generation <= 512) as a synthetic trace, in the compressed-arrival variant so that rounds carry many tiny chunks
    (PAPER.md:488-497), aging scheduler with chunk budget 256 as in Table 4: oracle parity on sampled iterations,
    schedule identity, and the per-iteration time against the small-batch floor."""
    build.build()
    Hq, Hkv, D, B, layers = 32, 8, 128, 16, 2
    trace = wl.make_sharegpt_like_trace(200, gap_us=150.0, seed=6)
    kw = dict(alpha=100.0, beta=-1.0, B_max=256, S_max=64, num_blocks=8192, block_size=B)
    stats = []
    scale = float(np.float32(1.0) / np.sqrt(np.float32(D)))
    hook = make_parity_hook(Hq, Hkv, D, B, layers, 40, 192, stats, scale)
    report, log = trace_run.run_trace(trace, Hq=Hq, Hkv=Hkv, D=D, B=B, layers=layers, pages_per_layer=8192,
                                      sched_kw=kw, seed=6, hook=hook)
    assert report["e2e_s"]["finished"] == 200 and len(stats) >= 10
    digest, n = replay_reference(trace, log, **dict(kw, page_mb=2 * Hkv * B * D * 2 * layers / 2**20))
    assert n == len(log) and digest == report["schedule_sha256"]
    per_layer = np.asarray(log, np.float64) / layers
    report["us_per_layer"] = {"p50": float(np.percentile(per_layer, 50)), "p95": float(np.percentile(per_layer, 95)), "min": float(per_layer.min())}
    assert report["us_per_layer"]["p50"] < 60.0            # short contexts: a round is a few times the launch floor, not more
    os.makedirs("gpurun_out", exist_ok=True)
    with open("gpurun_out/trace_sharegpt_like.json", "w") as f:
        json.dump(report, f)
