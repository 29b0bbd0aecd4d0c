#!/usr/bin/env python
"""bench.py -- mixed-batch paged-attention iteration on B200 (libcp), one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload b2048] [--impl reference]

A "step" is one pass of the hot path over one synthetic batch:
H1 cp_build_batch (pack + one H2D of metadata) -> H2 KV append -> H3/H4 attention ->
H5 combine -> H6 event pair, for one layer.  `value` = tokens/s with Q/K/V and the KV
pool already resident in HBM; `e2e` = the same through the C ABI with HOST buffers
(pinned Q/K_new/V_new copied in, `out` copied back, every step; copies of neighbouring
steps overlap the attention of the current one on their own streams).  The workload is
BASELINE.json configs[2] (token budget 2048, the config the north-star target is quoted
on); inputs are seeded and synthetic (paper_2606_09061_b200/workloads.py).
N > 1: replicas only (the path does not shard in scope): each rank
runs an independent replica, no data-path collective, scaling = weak.
`--impl reference` times the fp64 CPU oracle (test infrastructure) on the host cores.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2606_09061_b200 import workloads as wl  # noqa: E402

METRIC = "mixed-batch attention tokens/s (iteration us = 1000*ms_per_step; % of HBM/tensor roofline in roofline.frac)"
UNIT = "tokens/s"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                    "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    "source": "measured"}
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0,
            "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks + throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=lambda: [self.lines.append(l) for l in self.proc.stdout], daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, pw, mx, reasons = [], [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in self.lines:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx = float(f[1])
            except ValueError:
                continue
            try:
                pw.append(float(f[2]))
            except ValueError:
                pass
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        # power.draw is a running average that lags the load by ~1 s: the last quarter of the samples is
        # the steady state of a long run (--steps 4000), the start of a short one
        tail = pw[-max(1, len(pw) // 4):]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx,
                "reasons": sorted(reasons), "samples": len(sm),
                "sm_mhz_last_quarter": float(np.median(sm[-max(1, len(sm) // 4):])) if sm else None,
                "power_w_last_quarter": float(np.mean(tail)) if tail else None,
                "power_w_max": float(max(pw)) if pw else None}


def oracle_sample_rate(spec, q_bits, cache_bits, target_s, seed=0):
    """Time the fp64 oracle, as it stands, on a bounded seeded sample of (token, head) rows.
    Returns (equivalent tokens/s for the whole batch, threads, description)."""
    from oracle import attention as ora
    rng = np.random.default_rng(seed)
    tabs = spec.compact_tables()
    cu = np.concatenate([[0], np.cumsum(spec.q_len)])
    tok_req = np.repeat(np.arange(spec.n_reqs), spec.q_len)
    keys_of_tok = spec.ctx_off[tok_req].astype(np.int64) + (np.arange(spec.T) - cu[tok_req]) + 1

    def run(n):
        if n >= spec.T * spec.Hq:                          # the whole batch fits the time budget
            tok = np.repeat(np.arange(spec.T, dtype=np.int64), spec.Hq)
            head = np.tile(np.arange(spec.Hq, dtype=np.int32), spec.T)
        else:
            tok = rng.integers(0, spec.T, size=n).astype(np.int64)
            head = rng.integers(0, spec.Hq, size=n).astype(np.int32)
        t0 = time.perf_counter()
        ora.attention(q_bits, cache_bits, spec.q_len, spec.ctx_off, tabs, spec.sm_scale, rows=(tok, head))
        return time.perf_counter() - t0, int(keys_of_tok[tok].sum())

    threads = ora.num_threads()
    dt, pairs = run(64 * threads)                         # calibration (also warms the pages)
    n = int(max(64 * threads, min(2_000_000, 64 * threads * target_s / max(dt, 1e-3))))
    dt, pairs = run(n)
    total_pairs = spec.causal_pairs() * spec.Hq
    full_s = dt * total_pairs / max(pairs, 1)
    n = min(n, spec.T * spec.Hq)
    desc = (f"{n} seeded (token,head) rows of {spec.T * spec.Hq} ({pairs} of {total_pairs} causal "
            f"pairs) in {dt:.2f} s" + ("; the whole batch" if n == spec.T * spec.Hq else
                                       "; full-batch time extrapolated by the causal-pair ratio"))
    return spec.T / full_s, threads, desc


def ncu_traffic(workload):
    """DRAM bytes per launch of the attention kernel from the committed `ncu --set full` capture of this
    workload (profiles/traffic.json: a STATIC figure copied from the capture named there, not measured in
    this run -- it goes stale when the kernel or the work-list order changes, hence the source string that
    travels with it).  Returns (bytes or None, source or None)."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        e = json.load(open(p)).get(workload, {})
        if "dram_bytes_per_launch" not in e:
            return None, None
        return e["dram_bytes_per_launch"], f"profiles/traffic.json (static; {e.get('capture', 'capture unnamed')}; kernel at commit {e.get('commit', '?')})"
    except Exception:
        return None, None


def config_dict(spec, kv_dtype="bf16"):
    """The workload description, identical in both arms (ours and --impl reference)."""
    return {"workload": f"BASELINE.json configs[2] '{spec.name}'" if spec.name == "b2048" else spec.name,
            "tokens": spec.T, "requests": spec.n_reqs, "decodes": int((spec.q_len == 1).sum()),
            "prefill_chunks": int((spec.q_len > 1).sum()), "sum_kv_len": int(spec.kv_len.sum()),
            "pages": int(sum(len(b) for b in spec.block_tables)), "pool_pages": spec.num_blocks,
            "Hq": spec.Hq, "Hkv": spec.Hkv, "D": spec.D, "block": spec.B, "layers_per_step": 1,
            "kv_dtype": kv_dtype, "l2": "inputs_exceed_l2 (KV >> 126 MB), no flush"}


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def max_over_ranks(ms: float, device="cpu") -> float:
    """Device time of the slowest replica (the contract's max-over-ranks); identity at N = 1."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank_step: int, steps: int, world: int, ms_max: float) -> float:
    """Replicas only, weak scaling: every rank processes the same number of units per step."""
    return world * units_per_rank_step * steps / (ms_max * 1e-3)


def run_ours(args):
    import torch
    from paper_2606_09061_b200 import binding, build
    rank, local_rank, world = dist_env()
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    torch.cuda.set_device(local_rank)
    dev = torch.device(f"cuda:{local_rank}")
    build.build()
    spec = wl.CONFIGS[args.workload](seed=rank)           # replicas: same shape, own seed
    fp8 = args.kv_dtype == "e4m3"                          # a separate workload, the headline stays bf16
    n_pages = int(sum(len(b) for b in spec.block_tables))
    if fp8:
        q, k_new, v_new, pool, scales, compact, compact_scales = wl.device_values_fp8(spec, dev)
        chunk_pages = int(sum(len(b) for b, ql in zip(spec.block_tables, spec.q_len) if ql * (spec.Hq // spec.Hkv) > 8))
    else:
        q, k_new, v_new, pool, compact = wl.device_values(spec, dev)
    ctx = binding.Context(spec.Hq, spec.Hkv, spec.D, spec.num_blocks, spec.B, sm_scale=spec.sm_scale,
                          max_tokens=spec.T, max_reqs=spec.n_reqs, max_total_pages=n_pages,
                          device=local_rank, kv_dtype=binding.CP_KV_E4M3 if fp8 else binding.CP_KV_BF16,
                          max_scratch_pages=max(chunk_pages, 1) if fp8 else 0)
    descs, keep = binding.make_descs(spec.q_len, spec.ctx_off, spec.block_tables)
    out = torch.empty((spec.T, spec.Hq, spec.D), device=dev, dtype=torch.bfloat16)
    free_b, total_b = torch.cuda.mem_get_info(dev)
    ctx.cp_set_memory_stats((total_b - free_b) / 2**20, free_b / 2**20,
                            torch.cuda.memory_allocated(dev) / 2**20, torch.cuda.memory_reserved(dev) / 2**20)

    if args.rope:                                          # rotary embedding fused into the append
        ctx.cp_enable_rope(binding.rope_inv_freq(spec.D))
    attention_step = ctx.cp_attention_step_rope if args.rope else ctx.cp_attention_step
    if fp8:
        attention_step = lambda layer, q_, k_, v_, pool_, out_, stream=None: ctx.cp_attention_step_fp8(
            layer, q_, k_, v_, pool_, scales, out_, stream=stream)

    def step():
        ctx.cp_build_batch(descs=descs, n=spec.n_reqs)
        attention_step(0, q, k_new, v_new, pool, out)

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    ctx.cp_latency_table()                                 # drop warm-up rows
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_host0 = time.perf_counter()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    t_host_issue = time.perf_counter() - t_host0
    barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop()
    ms_total = max_over_ranks(ms_total, dev)
    rows = ctx.cp_latency_table()
    step_us = np.array([r.us for r in rows], dtype=np.float64)
    info = ctx.cp_get_batch_info()
    # H1 on its own ("cp_build_batch timed and reported separately"): host time of the call
    # (validate + plan + pack + enqueue one H2D), median of 20, queue drained between calls
    bb = []
    for _ in range(20):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.cp_build_batch(descs=descs, n=spec.n_reqs)
        bb.append((time.perf_counter() - t0) * 1e6)
    torch.cuda.synchronize()
    build_batch_us = float(np.median(bb))

    # ---- e2e: same metric through the C ABI with HOST buffers ------------------------------
    # Every step copies its Q / new K / new V from pinned host memory and reads its output back.  The
    # copies of step i+1 and the read-back of step i-1 run on their own streams under the attention
    # of step i (two sets of device buffers; the C ABI takes the stream), as a serving engine would
    # pipeline layers: the step time is the slowest of the three legs, not their sum.
    hq, hk, hv_ = (t.cpu().pin_memory() for t in (q, k_new, v_new))
    s_h2d, s_cmp, s_d2h = torch.cuda.Stream(dev), torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    sets = []
    for _ in range(2):
        sets.append({"q": torch.empty_like(q), "k": torch.empty_like(k_new), "v": torch.empty_like(v_new),
                     "out": torch.empty_like(out), "hout": torch.empty_like(out, device="cpu").pin_memory(),
                     "h2d": torch.cuda.Event(), "cmp": torch.cuda.Event(), "d2h": torch.cuda.Event()})
    hout = sets[0]["hout"]
    torch.cuda.synchronize()

    def e2e_step(i):
        b = sets[i % 2]
        s_h2d.wait_event(b["cmp"])                      # the step that last used these inputs has run
        with torch.cuda.stream(s_h2d):
            b["q"].copy_(hq, non_blocking=True); b["k"].copy_(hk, non_blocking=True); b["v"].copy_(hv_, non_blocking=True)
            b["h2d"].record(s_h2d)
        s_cmp.wait_event(b["h2d"])
        s_cmp.wait_event(b["d2h"])                      # its previous output has been read back
        ctx.cp_build_batch(descs=descs, n=spec.n_reqs, stream=s_cmp.cuda_stream)
        attention_step(0, b["q"], b["k"], b["v"], pool, b["out"], stream=s_cmp.cuda_stream)
        b["cmp"].record(s_cmp)
        s_d2h.wait_event(b["cmp"])
        with torch.cuda.stream(s_d2h):
            b["hout"].copy_(b["out"], non_blocking=True)
            b["d2h"].record(s_d2h)

    def e2e_join():                                     # everything issued so far, on all three streams
        for b in sets:
            s_cmp.wait_event(b["h2d"]); s_cmp.wait_event(b["d2h"])

    for i in range(4):
        e2e_step(i)
    e2e_join()
    barrier()
    e0.record(s_cmp)
    for i in range(args.steps):
        e2e_step(i)
    e2e_join()
    e1.record(s_cmp)
    barrier()
    e2e_ms = e0.elapsed_time(e1)
    e2e_ms = max_over_ranks(e2e_ms, dev)
    ctx.cp_latency_table()
    meta_bytes = 4 * (4 * spec.n_reqs + 2 + n_pages + spec.T) + 36 * info.n_work_items + 32 * info.n_combine_items
    h2d = int(hq.numel() * 2 + hk.numel() * 2 + hv_.numel() * 2 + meta_bytes)
    d2h = int(hout.numel() * 2)

    if rank != 0:
        ctx.close()
        return
    peaks = measured_peaks()
    ms_per_step = ms_total / args.steps
    tokens_per_s = whole_job_rate(spec.T, args.steps, world, ms_total)
    # roofline for the step's kernels (append + attention + combine), CUDA events on the launch stream
    attn_us = float(np.mean(step_us)) if len(step_us) else ms_per_step * 1e3
    bytes_alg, flops_alg = spec.algorithmic_bytes(args.kv_dtype), spec.flops()
    t_hbm = bytes_alg / (peaks["hbm_gbs"] * 1e9)
    # the tensor peak that applies (B200_PROFILING.md): the burst figure for a kernel timed alone for a short while,
    # the sustained one when the timed region is long enough for the power cap to engage (>= 1 s, or sw_power_cap seen)
    sustained = ms_total >= 1000.0 or "sw_power_cap" in (clocks.get("reasons") or [])
    tc_peak = peaks["bf16_tflops_sustained"] if sustained else peaks["bf16_tflops"]
    t_tc = flops_alg / (tc_peak * 1e12)
    bound = "hbm" if t_hbm >= t_tc else "tensor"
    if bound == "hbm":
        achieved, peak, runit = bytes_alg / (attn_us * 1e-6) / 1e9, peaks["hbm_gbs"], "GB/s"
    else:
        achieved, peak, runit = flops_alg / (attn_us * 1e-6) / 1e12, tc_peak, "TFLOP/s"
    traffic, traffic_source = ncu_traffic(spec.name + ("_e4m3" if fp8 else ""))
    res = {
        "metric": METRIC, "value": tokens_per_s, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "bf16" if not fp8 else "bf16 (fp8 e4m3 KV pages)", "data": "synthetic",
        "config": config_dict(spec, args.kv_dtype),
        "launch": {"parallelism": "replicas" if world > 1 else "single", "rope": bool(args.rope),
                   "work_items": info.n_work_items, "combine_items": info.n_combine_items,
                   "grid_attn": info.grid_attn, "kernels_per_step": info.kernels_per_step},
        "clocks": clocks,
        "e2e": {"value": whole_job_rate(spec.T, args.steps, world, e2e_ms), "unit": UNIT,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms / args.steps},
        "gpu_launches": int((info.kernels_per_step + (1 if args.rope else 0)) * args.steps),   # + rope_table_kernel of cp_build_batch
        "iteration_us": {"step_incl_build_batch": ms_per_step * 1e3, "attention_step_mean": attn_us,
                         "attention_step_median": float(np.median(step_us)) if len(step_us) else None,
                         "attention_step_min": float(step_us.min()) if len(step_us) else None,
                         "attention_step_p10": float(np.percentile(step_us, 10)) if len(step_us) else None,
                         "attention_step_p90": float(np.percentile(step_us, 90)) if len(step_us) else None,
                         "attention_step_last_quarter": float(step_us[-max(1, len(step_us) // 4):].mean()) if len(step_us) else None,
                         "host_issue_per_step": t_host_issue / args.steps * 1e6,
                         "build_batch_host_median": build_batch_us, "build_batch_h2d_bytes": int(meta_bytes)},
        "tflops": flops_alg / (attn_us * 1e-6) / 1e12, "gbs": bytes_alg / (attn_us * 1e-6) / 1e9,
        "roofline": {"bound": bound, "achieved": achieved, "peak": peak, "unit": runit,
                     "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_source,
                     "peak_source": peaks["source"] + (" (sustained)" if bound == "tensor" and sustained else " (burst)" if bound == "tensor" else ""),
                     "frac_of_tensor_burst": flops_alg / (attn_us * 1e-6) / 1e12 / peaks["bf16_tflops"],
                     "frac_of_tensor_sustained": flops_alg / (attn_us * 1e-6) / 1e12 / peaks["bf16_tflops_sustained"],
                     "frac_of_hbm": bytes_alg / (attn_us * 1e-6) / 1e9 / peaks["hbm_gbs"],
                     "kernel": "cp_attention_step kernels (append + attention + combine), mean of CUDA-event pairs",
                     "algorithmic_bytes": bytes_alg, "algorithmic_flops": flops_alg,
                     "t_hbm_us": t_hbm * 1e6, "t_tensor_us": t_tc * 1e6,
                     "frac_nominal_8TBs_2250TF": max(bytes_alg / 8e12, flops_alg / 2.25e15) / (attn_us * 1e-6)},
    }
    if bound == "hbm" and achieved > peak:
        # the peak is a COPY (half reads, half writes); a read-only stream runs above it on this part
        res["roofline"]["note"] = "achieved > peak: the measured peak is a read+write copy, this batch is a read-only stream"
    if world == 1 and not args.no_cpu_baseline and not fp8:
        from oracle import attention as ora
        cache = compact.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
        kb = k_new.view(torch.int16).cpu().numpy().view(np.uint16)
        vb = v_new.view(torch.int16).cpu().numpy().view(np.uint16)
        qb = q.view(torch.int16).cpu().numpy().view(np.uint16)
        ora.kv_append(kb, vb, cache, spec.q_len, spec.ctx_off, spec.compact_tables())
        v, threads, desc = oracle_sample_rate(spec, qb, cache, args.cpu_seconds)
        res["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc}
    ctx.close()
    print(json.dumps(res), flush=True)


def run_reference(args):
    """The reference arm for this tier = the fp64 oracle on the host cores (rank 0 only)."""
    rank, _, world = dist_env()
    if rank != 0:
        return
    from oracle import attention as ora
    spec = wl.CONFIGS[args.workload](seed=0)
    try:
        import torch
        assert torch.cuda.is_available()
        q, k_new, v_new, pool, compact = wl.device_values(spec, torch.device("cuda:0"))
        b = lambda t: t.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
        qb, kb, vb, cache = b(q), b(k_new), b(v_new), b(compact)
        del pool, compact
        torch.cuda.empty_cache()
    except Exception:
        hv = wl.host_values(spec)
        qb, kb, vb, cache = hv.q, hv.k_new, hv.v_new, hv.cache
    ora.kv_append(kb, vb, cache, spec.q_len, spec.ctx_off, spec.compact_tables())
    # A step = the oracle over the WHOLE batch when warm-up + steps of that fit ~5 minutes on this host (configs[2]:
    # ~7 s per step on 16 cores); otherwise a bounded seeded row sample per step, the full-batch rate extrapolated by
    # the causal-pair ratio and the line says so ("extrapolated": true; ms_per_step stays the measured wall time).
    n_steps = args.warmup + args.steps
    v0, threads, _ = oracle_sample_rate(spec, qb, cache, 1.0, seed=10_000)
    full_s = spec.T / v0
    whole = full_s * n_steps <= 300.0
    per_step_s = 1e9 if whole else max(1.0, min(20.0, 150.0 / n_steps))
    vals, descs, walls = [], [], []
    for i in range(n_steps):
        t0 = time.perf_counter()
        v, threads, desc = oracle_sample_rate(spec, qb, cache, per_step_s, seed=i)
        if i >= args.warmup:
            vals.append(v); descs.append(desc); walls.append(time.perf_counter() - t0)
    v = float(np.mean(vals))
    res = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": world,
           "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": spec.T / v * 1e3 if whole else float(np.mean(walls)) * 1e3, "extrapolated": not whole,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
           "data": "synthetic", "config": config_dict(spec),
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": descs[-1]},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(res), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="b2048", choices=sorted(wl.CONFIGS))
    ap.add_argument("--rope", action="store_true",
                    help="time cp_attention_step_rope (rotary embedding of Q / new K fused into the append)")
    ap.add_argument("--kv-dtype", default="bf16", choices=["bf16", "e4m3"],
                    help="e4m3: FP8 KV pages through cp_attention_step_fp8 (its own algorithmic-bytes roofline)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.gpus > 1 and "RANK" not in os.environ:
        # `python bench.py --gpus N` without a launcher: re-exec under torch.distributed.run, one replica per GPU
        # (rendezvous on 127.0.0.1; "replicas only")
        port = 29500 + os.getpid() % 2000
        os.execvp(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
                                   f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
                                   "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]])
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
