"""Trace-driven serving loop (BASELINE.json configs[4]): the C++ aging / LPRS / APC scheduler
forms every iteration, libcp runs that iteration's attention on the GPU for every layer, the
measured device time advances the scheduler's clock (PAPER.md:87 round structure, PAPER.md:155
"ground-truth batch latency measured by a high-resolution timer").

  python -m paper_2606_09061_b200.trace_run [--requests 1000] [--rate 8] [--layers 32] ...

Everything on the path goes through the C ABI (binding.Scheduler, binding.Context); PyTorch
only owns the device buffers.  The model around the attention step does not exist here (no
weights): Q and the new K/V rows of a layer are seeded N(0,1) bf16 rows from a bank, so the KV
cache content is a deterministic function of (seed, schedule).  The clock is virtual: `now`
advances by the measured device microseconds of the iteration's attention steps, so host
overhead of this Python loop does not distort the schedule.

All layers of an iteration go down in ONE cp_attention_layers submission with one CUDA-event pair
(kernel launch latency is a fixed per-round overhead; most rounds are a few decodes).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import struct
import time
from typing import Callable, Optional

import numpy as np

from . import binding, workloads as wl


def pack_batch(descs, n) -> bytes:
    """Canonical little-endian record of one iteration's composition:
    (req_id i64, q_len i32, ctx_off i32, n_pages i32, pages i32[n_pages]) per request."""
    b = bytearray()
    for i in range(n):
        d = descs[i]
        b += struct.pack("<qiii", d.req_id, d.q_len, d.ctx_off, d.n_blocks)
        b += bytes(memoryview((binding.C.c_int32 * d.n_blocks).from_address(
            binding.C.addressof(d.block_table.contents))))
    return bytes(b)


def percentile(x, p):
    return float(np.percentile(np.asarray(x, dtype=np.float64), p)) if len(x) else None


class IterationRunner:
    """One scheduled iteration over all layers, as the scheduler's clock sees it.  Owns the seeded Q / K / V banks,
    the paged pool and the libcp context.  `run(descs, n)` packs the batch (cp_build_batch), runs every layer and
    returns (device microseconds, latency row, batch info).

    Plain attention: ONE cp_attention_layers submission, one CUDA-event pair (H6).
    layer_gemms=True: per layer the attention step plus the dense projections of a Llama-shaped
    block -- QKV, O, gate/up, down as plain library GEMMs (torch.matmul = cuBLAS) on seeded random bf16 weights shared
    by all layers -- timed with one event pair around the whole iteration: the whole-forward-pass clock that the LPRS
    target T* and predictor are about.  The GEMMs are filler for the clock, not part of libcp.
    rope_inv_freq: every step goes through cp_attention_step_rope."""

    def __init__(self, Hq=32, Hkv=8, D=128, B=16, layers=32, pages_per_layer=20480, B_max=2048, S_max=1024, seed=0,
                 device=0, layer_gemms=False, d_model=4096, d_ff=14336, rope_inv_freq=None, random_pool=False):
        import torch
        self.torch = torch
        dev = self.dev = torch.device(f"cuda:{device}")
        torch.cuda.set_device(dev)
        self.layers, self.B_max, self.Hq, self.D, self.d_ff = layers, B_max, Hq, D, d_ff
        g = torch.Generator(device=dev)
        g.manual_seed(seed + 0x7ACE)
        bank = lambda h: torch.randn((layers, B_max, h, D), generator=g, device=dev, dtype=torch.float32).bfloat16()
        self.q_bank, self.k_bank, self.v_bank = bank(Hq), bank(Hkv), bank(Hkv)
        # torch.empty would do (include/cp.h: the pool needs no initialisation); zeros keep reruns reproducible
        self.pool = torch.zeros((layers, pages_per_layer, 2, Hkv, B, D), device=dev, dtype=torch.bfloat16)
        if random_pool:                                        # harvesting: decodes attend to pages nobody appended
            step = 8192
            for l in range(layers):
                for s0 in range(0, pages_per_layer, step):
                    n = min(step, pages_per_layer - s0)
                    self.pool[l, s0:s0 + n] = torch.randn((n, 2, Hkv, B, D), generator=g, device=dev, dtype=torch.float32).bfloat16()
        self.out = torch.empty((layers, B_max, Hq, D), device=dev, dtype=torch.bfloat16)
        ptr = lambda t: [int(t[l].data_ptr()) for l in range(layers)]
        self.q_p, self.k_p, self.v_p, self.pool_p, self.out_p = ptr(self.q_bank), ptr(self.k_bank), ptr(self.v_bank), ptr(self.pool), ptr(self.out)
        pa = binding.Context.pointer_array
        self.q_a, self.k_a, self.v_a, self.pool_a, self.out_a = pa(self.q_p), pa(self.k_p), pa(self.v_p), pa(self.pool_p), pa(self.out_p)
        self.ctx = binding.Context(Hq, Hkv, D, pages_per_layer, B, num_layers=layers, max_tokens=B_max, max_reqs=S_max,
                                   max_total_pages=pages_per_layer, device=device)
        self.rope = rope_inv_freq is not None
        if self.rope:
            self.ctx.cp_enable_rope(rope_inv_freq)
        free_b, total_b = torch.cuda.mem_get_info(dev)
        self.ctx.cp_set_memory_stats((total_b - free_b) / 2**20, free_b / 2**20,
                                     torch.cuda.memory_allocated(dev) / 2**20, torch.cuda.memory_reserved(dev) / 2**20)
        self.layer_gemms = layer_gemms
        if layer_gemms:
            gw = lambda k, n: (torch.randn((k, n), generator=g, device=dev, dtype=torch.float32) * 0.02).bfloat16()
            self.w_qkv, self.w_o = gw(d_model, (Hq + 2 * Hkv) * D), gw(Hq * D, d_model)
            self.w_gu, self.w_dn = gw(d_model, 2 * d_ff), gw(d_ff, d_model)
            self.x_buf = torch.randn((B_max, d_model), generator=g, device=dev, dtype=torch.float32).bfloat16()
        self.ev0, self.ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def _dense_part(self, T):
        torch, d_ff = self.torch, self.d_ff
        x = self.x_buf[:T]
        qkv = x @ self.w_qkv                                   # the attention inputs stay the seeded banks
        h = (x @ self.w_gu)
        y = (torch.nn.functional.silu(h[:, :d_ff]) * h[:, d_ff:]) @ self.w_dn
        return qkv, y, self.out[0, :T].reshape(T, self.Hq * self.D) @ self.w_o

    def run(self, descs, n, q_len=None, ctx_off=None, block_tables=None):
        ctx = self.ctx
        if descs is not None:
            ctx.cp_build_batch(descs=descs, n=n)
        else:
            ctx.cp_build_batch(q_len, ctx_off, block_tables)
        info = ctx.cp_get_batch_info()
        if not self.layer_gemms and not self.rope:
            ctx.cp_attention_layers(self.q_a, self.k_a, self.v_a, self.pool_a, self.out_a)
            row = ctx.cp_latency_table(cap=2)[0]               # waits for the iteration (H6)
            return float(row.us), row, info
        step = ctx.cp_attention_step_rope if self.rope else ctx.cp_attention_step
        self.ev0.record()
        for l in range(self.layers):
            step(l, self.q_p[l], self.k_p[l], self.v_p[l], self.pool_p[l], self.out_p[l])
            if self.layer_gemms:
                self._dense_part(info.n_tokens)
        self.ev1.record()
        rows = ctx.cp_latency_table(cap=self.layers)
        self.ev1.synchronize()
        us = self.ev0.elapsed_time(self.ev1) * 1e3 if self.layer_gemms else float(sum(r.us for r in rows))
        return us, rows[0], info

    def layer_tensors(self, l, T):
        return self.q_bank[l, :T], self.k_bank[l, :T], self.v_bank[l, :T], self.pool[l], self.out[l, :T]

    def close(self):
        self.ctx.close()


def _peaks():
    """Measured B200 peaks for the trace roofline (MEASURED_PEAKS.json at the repo root when present, else the
    fallback of B200_PROFILING.md)."""
    import os
    p = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")
    try:
        d = json.load(open(p))
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]), "source": "measured"}
    except Exception:
        return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "source": "fallback"}


def run_trace(trace, *, Hq=32, Hkv=8, D=128, B=16, layers=32, pages_per_layer=20480,
              sched_kw: Optional[dict] = None, seed=0, device=0,
              hook: Optional[Callable] = None, max_iters: Optional[int] = None,
              overhead_us: int = 0, layer_gemms: bool = False, d_model: int = 4096, d_ff: int = 14336,
              rope_inv_freq=None):
    """Run the whole trace.  `hook(it, batch, layer_tensors)` (tests only) is called after an
    iteration's steps were issued and synchronised, with batch = [(req_id, q_len, ctx_off,
    pages)] and layer_tensors(l) -> (q, k_new, v_new, pool_l, out_l).  Returns a report dict
    plus the per-iteration measured microseconds (what the scheduler was told).

    The report carries, per iteration class, the algorithmic bytes and FLOPs of the attention steps (SURVEY.md 8(d)
    formulas x layers) over the measured busy time: what fraction of the HBM / tensor roofline the serving loop
    reaches, and the per-layer time of the decode-only rounds against the per-step floor (fixed
    per-round overheads -- feature extraction, latency prediction, kernel launch latency)."""
    kw = dict(alpha=100.0, beta=-1.0, B_max=2048, S_max=1024, num_blocks=pages_per_layer, block_size=B,
              page_mb=2 * Hkv * B * D * 2 * layers / 2**20)
    kw.update(sched_kw or {})
    B_max, S_max = kw["B_max"], kw["S_max"]
    sched = binding.Scheduler(**{**kw, "max_batch": S_max})
    for rid, a, p, o in zip(*trace):
        sched.cp_sched_add_request(int(rid), int(a), int(p), int(o))
    n_req = len(trace[0])
    runner = IterationRunner(Hq, Hkv, D, B, layers, pages_per_layer, B_max, S_max, seed, device, layer_gemms,
                             d_model, d_ff, rope_inv_freq)
    digest = hashlib.sha256()
    now, n_it, tokens = 0, 0, 0
    iter_us_log = []
    names = ("decode_only", "mixed", "prefill_only")
    classes = {k: [] for k in names}
    work = {k: [0.0, 0.0] for k in names}                    # algorithmic [bytes, flops] of the attention steps, all layers
    busy_us = 0
    t_wall = time.perf_counter()
    while sched.cp_sched_has_work():
        n = sched.cp_sched_next(now)
        digest.update(pack_batch(sched.descs, n))
        if n == 0:
            nxt = sched.cp_sched_next_arrival()
            if nxt < 0:
                raise RuntimeError("scheduler has work but nothing is runnable and nothing will arrive "
                                   "(a request that can never be admitted under this configuration)")
            now = max(now, nxt)
            continue
        us, r0, info = runner.run(sched.descs, n)
        iter_us = max(1, int(round(us)) + overhead_us)
        cls = "decode_only" if r0.n_prefill == 0 else ("prefill_only" if r0.n_decode == 0 else "mixed")
        classes[cls].append(us)
        work[cls][0] += info.alg_bytes * layers
        work[cls][1] += info.alg_flops * layers
        T = info.n_tokens
        tokens += T
        if hook is not None:
            hook(n_it, sched.batch(), lambda l: runner.layer_tensors(l, T))
        sched.cp_sched_commit(iter_us)
        iter_us_log.append(iter_us)
        now += iter_us
        busy_us += iter_us
        n_it += 1
        if max_iters is not None and n_it >= max_iters:
            break
    wall_s = time.perf_counter() - t_wall
    ttft, e2e = [], []
    for rid, a in zip(trace[0], trace[1]):
        t1, t2 = sched.cp_sched_request_times(int(rid))
        if t1 >= 0:
            ttft.append((t1 - int(a)) * 1e-6)
        if t2 >= 0:
            e2e.append((t2 - int(a)) * 1e-6)
    st = sched.cp_sched_get_stats()
    hist = {k: {"iterations": len(v), "us_mean": float(np.mean(v)) if v else None, "us_p50": percentile(v, 50),
                "us_p95": percentile(v, 95), "us_max": float(np.max(v)) if v else None,
                "us_per_layer_p50": percentile(v, 50) / layers if v else None} for k, v in classes.items()}
    peaks = _peaks()
    roof = {}
    for k in names:
        t = float(np.sum(classes[k])) * 1e-6
        if t <= 0:
            continue
        gbs, tfs = work[k][0] / t / 1e9, work[k][1] / t / 1e12
        roof[k] = {"algorithmic_bytes": work[k][0], "algorithmic_flops": work[k][1], "busy_s": t, "gbs": gbs, "tflops": tfs,
                   "frac_of_hbm_peak": gbs / peaks["hbm_gbs"], "frac_of_tensor_peak": tfs / peaks["bf16_tflops"]}
    tot_t = float(sum(np.sum(v) for v in classes.values())) * 1e-6
    if tot_t > 0:
        tb, tf = sum(w[0] for w in work.values()), sum(w[1] for w in work.values())
        roof["all"] = {"algorithmic_bytes": tb, "algorithmic_flops": tf, "busy_s": tot_t, "gbs": tb / tot_t / 1e9,
                       "tflops": tf / tot_t / 1e12, "frac_of_hbm_peak": tb / tot_t / 1e9 / peaks["hbm_gbs"],
                       "frac_of_tensor_peak": tf / tot_t / 1e12 / peaks["bf16_tflops"]}
    report = {
        "workload": "trace", "requests": n_req, "layers": layers, "iterations": n_it,
        "virtual_time_s": now * 1e-6, "gpu_busy_frac": busy_us / max(now, 1), "wall_s": wall_s,
        "tokens": tokens, "tokens_per_s_virtual": tokens / max(now * 1e-6, 1e-9),
        "tokens_per_s_gpu_busy": tokens / max(busy_us * 1e-6, 1e-9),
        "iteration_us_by_class": hist,
        "attention_roofline_by_class": roof, "peaks": peaks,
        "clock": "whole forward pass (attention + dense GEMM filler)" if layer_gemms else "attention steps of all layers, one submission",
        "e2e_s": {"mean": float(np.mean(e2e)) if e2e else None, "p95": percentile(e2e, 95), "finished": len(e2e)},
        "ttft_s": {"mean": float(np.mean(ttft)) if ttft else None, "p95": percentile(ttft, 95), "started": len(ttft)},
        "blocked_by_activity_cap": int(st.blocked_by_activity_cap), "blocked_by_min_chunk": int(st.blocked_by_min_chunk),
        "schedule_sha256": digest.hexdigest(),
        "sched": {k: v for k, v in kw.items() if not hasattr(v, "__len__")},
    }
    runner.close()
    sched.close()
    return report, iter_us_log


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--requests", type=int, default=1000)
    ap.add_argument("--rate", type=float, default=8.0, help="Poisson arrivals per second")
    ap.add_argument("--layers", type=int, default=32)
    ap.add_argument("--pages-per-layer", type=int, default=20480)
    ap.add_argument("--budget", type=int, default=2048)
    ap.add_argument("--alpha", type=float, default=100.0)
    ap.add_argument("--beta", type=float, default=-1.0)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--max-iters", type=int, default=None)
    ap.add_argument("--iter-us-out", default=None, help="write the measured iteration us (one per line)")
    ap.add_argument("--layer-gemms", action="store_true", help="add the dense projections of each layer (library GEMMs) to the iteration time")
    a = ap.parse_args()
    from . import build
    build.build()
    trace = wl.make_trace(a.requests, rate_per_s=a.rate, seed=a.seed)
    report, log = run_trace(trace, layers=a.layers, pages_per_layer=a.pages_per_layer, seed=a.seed,
                            sched_kw=dict(alpha=a.alpha, beta=a.beta, B_max=a.budget), max_iters=a.max_iters,
                            layer_gemms=a.layer_gemms)
    report["arrival_rate_per_s"] = a.rate
    if a.iter_us_out:
        with open(a.iter_us_out, "w") as f:
            f.write("\n".join(map(str, log)) + "\n")
    print(json.dumps(report))


if __name__ == "__main__":
    main()
