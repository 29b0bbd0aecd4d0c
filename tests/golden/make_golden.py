"""Writes tests/golden/sched_digests.txt: SHA-256 of the REFERENCE scheduler's batch
composition (oracle/ref_scheduler.py, canonical packing `pack_record`) on seeded traces.

  python -m tests.golden.make_golden

Calls only oracle/ and the seeded trace generators (paper_2606_09061_b200/workloads.py,
which holds none of the method's arithmetic); never the C++ scheduler.  The paper prints no
worked example, so these digests are not the paper's values: they
freeze the reference scheduler's readings S1-S14 so that a later change to either
scheduler shows up as a diff of this file and must be justified against the paper.
"""
import hashlib
import os

from oracle import ref_scheduler as rs
from paper_2606_09061_b200 import workloads as wl

HERE = os.path.dirname(os.path.abspath(__file__))
OUT = os.path.join(HERE, "sched_digests.txt")

LIN_W = [0.0] * 16
LIN_W[11], LIN_W[12], LIN_W[14], LIN_W[15], LIN_W[7] = 37.5, 0.31, 0.0021, 1.3e-5, 0.01


def iter_us_model(batch):
    """Deterministic stand-in for the measured iteration time (integer us): an INPUT of the
    scheduler (PAPER.md:155 measures it), not part of the method."""
    tokens = sum(b[1] for b in batch)
    ctx = sum(b[2] + b[1] for b in batch)
    return 40 + (tokens * 3) // 10 + ctx // 700


def small_trace(seed, n=150, rate=400.0):
    return wl.make_trace(n, rate_per_s=rate, seed=seed, short_median=120, long_lo=600, long_hi=2500,
                         out_median=12, out_max=60)


CASES = {
    # name: (trace factory, scheduler config)
    "aging_budget256": (lambda: small_trace(0), dict(alpha=100.0, beta=-1.0, B_max=256, S_max=32, num_blocks=2000)),
    "fcfs_beta0": (lambda: small_trace(5), dict(alpha=1.0, beta=0.0, B_max=128, S_max=16, num_blocks=1500)),
    "lprs_apc_linear": (lambda: small_trace(7), dict(B_max=512, S_max=48, mode=rs.MODE_LPRS, apc=True, Delta=32,
                                                     T_star=120.0, lambda_u=1.0, lambda_o=2.5, C_max=3, L_min=24,
                                                     num_blocks=2500, page_mb=0.0625, pred_weights=LIN_W)),
    "apc_ablation_shape": (lambda: wl.make_apc_trace(400, seed=2),
                           dict(B_max=96, S_max=64, mode=rs.MODE_LPRS, apc=True, Delta=8, T_star=70.0, C_max=2,
                                L_min=16, num_blocks=4000, pred_weights=LIN_W)),
}


def drive(sched_next, sched_commit, has_work, next_arrival):
    """Run a scheduler to completion under iter_us_model; returns (sha256 hex, iterations)."""
    h, t, n_it = hashlib.sha256(), 0, 0
    while has_work():
        batch = sched_next(t)
        h.update(rs.pack_record(batch))
        if not batch:
            t = next_arrival()
            continue
        dt = iter_us_model(batch)
        sched_commit(dt)
        t += dt
        n_it += 1
    return h.hexdigest(), n_it


def reference_digest(name):
    make_trace, kw = CASES[name]
    ref = rs.RefScheduler(rs.SchedConfig(**kw))
    for rid, a, p, o in zip(*make_trace()):
        ref.add_request(int(rid), int(a), int(p), int(o))
    return drive(ref.next, ref.commit, ref.has_work, ref.next_arrival_us)


def read_golden():
    out = {}
    with open(OUT) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                name, digest, n_it = line.split()
                out[name] = (digest, int(n_it))
    return out


def main():
    with open(OUT, "w") as f:
        f.write("# written by `python -m tests.golden.make_golden` (reference scheduler only; see its docstring)\n")
        f.write("# name sha256(batch composition of every iteration) iterations\n")
        for name in CASES:
            d, n = reference_digest(name)
            f.write(f"{name} {d} {n}\n")
            print(name, d, n)


if __name__ == "__main__":
    main()
