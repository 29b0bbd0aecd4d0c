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

The pool is zero-filled once: page slots that were never written must hold finite values
(include/cp.h, R6).
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


def run_trace(trace, *, Hq=32, Hkv=8, D=128, B=16, layers=32, pages_per_layer=20480,
              sched_kw: Optional[dict] = None, seed=0, device=0, kernel_variant=0,
              hook: Optional[Callable] = None, max_iters: Optional[int] = None,
              overhead_us: int = 0, layer_gemms: bool = False, d_model: int = 4096, d_ff: int = 14336,
              rope_inv_freq=None):
    """Run the whole trace.  `hook(it, batch, layer_tensors)` (tests only) is called after an
    iteration's steps were issued and synchronised, with batch = [(req_id, q_len, ctx_off,
    pages)] and layer_tensors(l) -> (q, k_new, v_new, pool_l, out_l).  Returns a report dict
    plus the per-iteration measured microseconds (what the scheduler was told).

    layer_gemms=True adds, per layer, the dense projections of a Llama-shaped
    block around the attention step -- QKV, O, gate/up, down as plain library GEMMs (torch.matmul =
    cuBLAS) on seeded random bf16 weights shared by all layers -- so that the iteration time the
    scheduler sees is that of a whole forward pass; it is timed with CUDA events around the whole
    iteration.  The GEMMs are filler for the clock, not part of libcp.

    rope_inv_freq (float64 [D/2]): every step goes through cp_attention_step_rope, i.e. the
    Q / new-K banks are taken as unrotated and rotated by absolute position inside the append."""
    import torch
    dev = torch.device(f"cuda:{device}")
    torch.cuda.set_device(dev)
    kw = dict(alpha=100.0, beta=-1.0, B_max=2048, S_max=1024, num_blocks=pages_per_layer, block_size=B,
              page_mb=2 * Hkv * B * D * 2 * layers / 2**20)
    kw.update(sched_kw or {})
    B_max, S_max = kw["B_max"], kw["S_max"]
    sched = binding.Scheduler(**{**kw, "max_batch": S_max})
    for rid, a, p, o in zip(*trace):
        sched.cp_sched_add_request(int(rid), int(a), int(p), int(o))
    n_req = len(trace[0])

    g = torch.Generator(device=dev)
    g.manual_seed(seed + 0x7ACE)
    bank = lambda h: torch.randn((layers, B_max, h, D), generator=g, device=dev, dtype=torch.float32).bfloat16()
    q_bank, k_bank, v_bank = bank(Hq), bank(Hkv), bank(Hkv)
    pool = torch.zeros((layers, pages_per_layer, 2, Hkv, B, D), device=dev, dtype=torch.bfloat16)
    out = torch.empty((layers, B_max, Hq, D), device=dev, dtype=torch.bfloat16)
    ptr = lambda t: [int(t[l].data_ptr()) for l in range(layers)]
    q_p, k_p, v_p, pool_p, out_p = ptr(q_bank), ptr(k_bank), ptr(v_bank), ptr(pool), ptr(out)

    ctx = binding.Context(Hq, Hkv, D, pages_per_layer, B, num_layers=layers, max_tokens=B_max, max_reqs=S_max,
                          max_total_pages=pages_per_layer, device=device, kernel_variant=kernel_variant)
    if rope_inv_freq is not None:
        ctx.cp_enable_rope(rope_inv_freq)
    attention_step = ctx.cp_attention_step if rope_inv_freq is None else ctx.cp_attention_step_rope
    free_b, total_b = torch.cuda.mem_get_info(dev)
    ctx.cp_set_memory_stats((total_b - free_b) / 2**20, free_b / 2**20,
                            torch.cuda.memory_allocated(dev) / 2**20, torch.cuda.memory_reserved(dev) / 2**20)

    if layer_gemms:
        gw = lambda k, n: (torch.randn((k, n), generator=g, device=dev, dtype=torch.float32) * 0.02).bfloat16()
        w_qkv, w_o = gw(d_model, (Hq + 2 * Hkv) * D), gw(Hq * D, d_model)
        w_gu, w_dn = gw(d_model, 2 * d_ff), gw(d_ff, d_model)
        x_buf = torch.randn((B_max, d_model), generator=g, device=dev, dtype=torch.float32).bfloat16()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def dense_part(T):
        x = x_buf[:T]
        qkv = x @ w_qkv                                        # the attention inputs stay the seeded banks
        h = (x @ w_gu)
        y = (torch.nn.functional.silu(h[:, :d_ff]) * h[:, d_ff:]) @ w_dn
        return qkv, y, out[0, :T].reshape(T, Hq * D) @ w_o

    digest = hashlib.sha256()
    now, n_it, tokens = 0, 0, 0
    iter_us_log, classes = [], {"decode_only": [], "mixed": [], "prefill_only": []}
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
        ctx.cp_build_batch(descs=sched.descs, n=n)
        if layer_gemms:
            T_it = sum(sched.descs[i].q_len for i in range(n))
            ev0.record()
        for l in range(layers):
            attention_step(l, q_p[l], k_p[l], v_p[l], pool_p[l], out_p[l])
            if layer_gemms:
                dense_part(T_it)
        if layer_gemms:
            ev1.record()
        rows = ctx.cp_latency_table(cap=layers)            # waits for the iteration (H6)
        us = float(sum(r.us for r in rows))
        if layer_gemms:
            ev1.synchronize()
            us = ev0.elapsed_time(ev1) * 1e3                   # whole forward pass: attention + dense GEMMs
        iter_us = max(1, int(round(us)) + overhead_us)
        r0 = rows[0]
        cls = "decode_only" if r0.n_prefill == 0 else ("prefill_only" if r0.n_decode == 0 else "mixed")
        classes[cls].append(us)
        T = int(r0.feat[0] + r0.feat[1])
        tokens += T
        if hook is not None:
            batch = sched.batch()
            hook(n_it, batch, lambda l: (q_bank[l, :T], k_bank[l, :T], v_bank[l, :T], pool[l], out[l, :T]))
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
                "us_p95": percentile(v, 95), "us_max": float(np.max(v)) if v else None} for k, v in classes.items()}
    report = {
        "workload": "trace", "requests": n_req, "layers": layers, "iterations": n_it,
        "virtual_time_s": now * 1e-6, "gpu_busy_frac": busy_us / max(now, 1), "wall_s": wall_s,
        "tokens": tokens, "tokens_per_s_virtual": tokens / max(now * 1e-6, 1e-9),
        "tokens_per_s_gpu_busy": tokens / max(busy_us * 1e-6, 1e-9),
        "iteration_us_by_class": hist,
        "e2e_s": {"mean": float(np.mean(e2e)) if e2e else None, "p95": percentile(e2e, 95), "finished": len(e2e)},
        "ttft_s": {"mean": float(np.mean(ttft)) if ttft else None, "p95": percentile(ttft, 95), "started": len(ttft)},
        "blocked_by_activity_cap": int(st.blocked_by_activity_cap), "blocked_by_min_chunk": int(st.blocked_by_min_chunk),
        "schedule_sha256": digest.hexdigest(),
        "sched": {k: v for k, v in kw.items() if not hasattr(v, "__len__")},
    }
    ctx.close()
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
