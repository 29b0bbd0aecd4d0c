"""LPRS latency predictor, offline half (Tables 1-2, 7-8).

  python -m paper_2606_09061_b200.predictor [--samples 6000] [--out predictor.json]

Pipeline, as the paper describes it: (1) collect, per scheduling round, the 11 raw
features of Table 1 and the measured batch latency -- here the rows of cp_latency_table for swept
synthetic batches of the 8B shape; (2) clean, bucket by scheduled tokens, downsample the
over-represented full-budget bucket, split 8:1:1; (3) add the 5 derived features of Table 2; (4)
fit the predictor: a 16-coefficient linear model (least squares) and the 16 -> 128 -> 64 -> 32 -> 1
ReLU MLP (dropout 0.1, AdamW lr 2e-3, wd 1e-3, 300 epochs, batch 256: Table 7)
under a weighted asymmetric Huber loss (Eq. 5); (5) report MAE / RMSE / MAPE,
absolute-error percentiles and bounded-error ratios (Eq. 15-17, Table 8).

Readings (the paper gives neither value): Huber delta = 1.0 in units of the target's standard
deviation; under-estimates (y_hat < y) weigh 2x; bucket weight w_i = mean bucket size / size of the
sample's bucket.  The paper's 36,868 samples and trained weights are not available: the numbers this
module reports are for OUR latencies (attention step only, one layer) and are not comparable with
Table 8's milliseconds of a whole Qwen3-8B iteration.

The fitted model is data for the scheduler: `export_*` returns (pred_kind, weights, mu, inv_sigma)
in the layout cp_sched_config expects; both schedulers evaluate it in fixed-order fp64.
"""
from __future__ import annotations

import argparse
import json

import numpy as np

from . import binding

N_RAW, N_FEAT = 11, 16
MLP_DIMS = [16, 128, 64, 32, 1]


def features16(raw11: np.ndarray) -> np.ndarray:
    """Tables 1-2: [n, 11] raw -> [n, 16] = raw + (bias, scheduled_tokens, avg_decode_ctx,
    decode_ctx_interaction, prefill_interaction)."""
    r = np.asarray(raw11, dtype=np.float64).reshape(-1, N_RAW)
    pf, dec, sum_ctx, pf_proc = r[:, 0], r[:, 1], r[:, 3], r[:, 5]
    avg = sum_ctx / np.maximum(dec, 1.0)
    return np.concatenate([r, np.ones((len(r), 1)), (dec + pf)[:, None], avg[:, None], (dec * avg)[:, None],
                           (pf * pf_proc)[:, None]], axis=1)


def metrics(y: np.ndarray, y_hat: np.ndarray, bounds=(5.0, 10.0)) -> dict:
    """Eq. 15-17 + the percentile / bounded-error columns of Table 8 (units of y)."""
    e = np.abs(np.asarray(y_hat, np.float64) - np.asarray(y, np.float64))
    out = {"mae": float(e.mean()), "rmse": float(np.sqrt((e ** 2).mean())),
           "mape_pct": float(100.0 * (e / np.abs(y)).mean())}
    for q in (50, 90, 95, 99):
        out[f"p{q}"] = float(np.percentile(e, q))
    for b in bounds:
        out[f"within_{b:g}"] = float((e <= b).mean())
    return out


def bucket_downsample_split(tokens: np.ndarray, rng, bucket=256, full_budget=2048, seed_split=(0.8, 0.1, 0.1)):
    """Bucket by scheduled tokens, cut the full-budget bucket down to the size of the largest other
    bucket, split 8:1:1.  Returns (train, val, test index arrays, bucket ids)."""
    b = np.minimum(tokens // bucket, full_budget // bucket).astype(np.int64)
    keep = np.ones(len(tokens), bool)
    full = np.flatnonzero(b == full_budget // bucket)
    others = np.bincount(b[b < full_budget // bucket]) if (b < full_budget // bucket).any() else np.array([0])
    cap = max(int(others.max()), 1)
    if len(full) > cap:
        keep[rng.choice(full, size=len(full) - cap, replace=False)] = False
    idx = rng.permutation(np.flatnonzero(keep))
    n_tr, n_va = int(seed_split[0] * len(idx)), int(seed_split[1] * len(idx))
    return idx[:n_tr], idx[n_tr:n_tr + n_va], idx[n_tr + n_va:], b


def fit_linear(X16, y, w=None):
    """Weighted least squares on standardised features (the bias column stays 1).  Returns
    (weights[16], mu[16], inv_sigma[16]) so that y_hat = sum_k weights[k] * (x[k] - mu[k]) * inv_sigma[k]."""
    X = np.asarray(X16, np.float64)
    mu, sd = X.mean(0), X.std(0)
    mu[11], sd[11] = 0.0, 1.0
    inv = np.where(sd > 0, 1.0 / np.where(sd > 0, sd, 1.0), 0.0)
    Z = (X - mu) * inv
    sw = np.sqrt(np.ones(len(y)) if w is None else np.asarray(w, np.float64))
    coef, *_ = np.linalg.lstsq(Z * sw[:, None], np.asarray(y, np.float64) * sw, rcond=None)
    return coef, mu, inv


def predict_linear(model, X16):
    coef, mu, inv = model
    return ((np.asarray(X16, np.float64) - mu) * inv) @ coef


def asymmetric_huber(y_hat, y, w, delta=1.0, under=2.0):
    """Eq. 5: L = (1/N) sum_i w_i l_i, l_i = Huber_delta(y_hat - y) x (under if y_hat < y else 1)."""
    import torch
    r = y_hat - y
    a = r.abs()
    h = torch.where(a <= delta, 0.5 * r * r, delta * (a - 0.5 * delta))
    return (w * h * torch.where(r < 0, torch.full_like(r, under), torch.ones_like(r))).mean()


def fit_mlp(X16, y, w, Xv, yv, epochs=300, lr=2e-3, weight_decay=1e-3, dropout=0.1, batch=256, seed=0):
    """Table 7.  Trains in standardised feature / target space; returns (flat weights in the
    cp_sched layout for targets in the ORIGINAL unit, mu, inv_sigma, best validation loss)."""
    import torch
    torch.manual_seed(seed)
    X = np.asarray(X16, np.float64)
    mu, sd = X.mean(0), X.std(0)
    mu[11], sd[11] = 0.0, 1.0
    inv = np.where(sd > 0, 1.0 / np.where(sd > 0, sd, 1.0), 0.0)
    ym, ys = float(np.mean(y)), float(np.std(y)) or 1.0
    t = lambda a: torch.tensor(a, dtype=torch.float32)
    Z, Zv = t((X - mu) * inv), t((np.asarray(Xv, np.float64) - mu) * inv)
    Y, Yv, W = t((np.asarray(y) - ym) / ys), t((np.asarray(yv) - ym) / ys), t(w)
    Wv = t((float(np.median(y)) / np.asarray(yv, np.float64)) ** 2)      # validation in relative error too
    Wv = Wv / Wv.mean()
    layers = []
    for i in range(4):
        layers.append(torch.nn.Linear(MLP_DIMS[i], MLP_DIMS[i + 1]))
        if i < 3:
            layers += [torch.nn.ReLU(), torch.nn.Dropout(dropout)]
    net = torch.nn.Sequential(*layers)
    opt = torch.optim.AdamW(net.parameters(), lr=lr, weight_decay=weight_decay)
    best, best_state = float("inf"), None
    g = torch.Generator().manual_seed(seed)
    for _ in range(epochs):
        net.train()
        perm = torch.randperm(len(Z), generator=g)
        for s in range(0, len(Z), batch):
            i = perm[s:s + batch]
            opt.zero_grad()
            asymmetric_huber(net(Z[i]).squeeze(1), Y[i], W[i]).backward()
            opt.step()
        net.eval()
        with torch.no_grad():
            v = float(asymmetric_huber(net(Zv).squeeze(1), Yv, Wv))
        if v < best:
            best, best_state = v, {k: p.detach().clone() for k, p in net.state_dict().items()}
    net.load_state_dict(best_state)
    lin = [m for m in net if isinstance(m, torch.nn.Linear)]
    flat = []
    for li, m in enumerate(lin):
        Wm, bm = m.weight.detach().double().numpy().copy(), m.bias.detach().double().numpy().copy()
        if li == 3:                      # fold the target de-standardisation into the last layer
            Wm, bm = Wm * ys, bm * ys + ym
        flat += [Wm.reshape(-1), bm.reshape(-1)]      # row-major [out][in], then bias: cp_sched layout
    return np.concatenate(flat), mu, inv, best


def predict_mlp(model, X16):
    """Plain fp64 forward of the exported weights (same arithmetic as cp_sched_predict, vectorised)."""
    flat, mu, inv = model[:3]
    z = (np.asarray(X16, np.float64) - mu) * inv
    pos = 0
    for li in range(4):
        n_in, n_out = MLP_DIMS[li], MLP_DIMS[li + 1]
        Wm = flat[pos:pos + n_out * n_in].reshape(n_out, n_in)
        pos += n_out * n_in
        bm = flat[pos:pos + n_out]
        pos += n_out
        z = z @ Wm.T + bm
        if li < 3:
            z = np.maximum(z, 0.0)
    return z[:, 0]


# ------------------------------------------------------------------------------------------------
# data collection on the GPU (the logging half is cp_latency_table, H6)
# ------------------------------------------------------------------------------------------------
def harvest(n_samples=6000, seed=0, Hq=32, Hkv=8, D=128, B=16, budget=2048, pages_per_layer=131072, layers=1,
            layer_gemms=False, device=0, repeats=2):
    """Sweep synthetic mixed batches shaped like the token-budget scheduler's rounds (decodes first,
    prefill chunks fill the rest: PAPER.md:87) and log (11 raw features, us) per round -- through the SAME
    IterationRunner the serving loop uses (trace_run.py), so the target is exactly the time the scheduler's clock
    is advanced by: all `layers` attention steps including the KV append, plus, with layer_gemms=True, the dense
    projections of every layer (the whole-forward-pass clock of PAPER.md:109, :456).  A batch is run 1 + repeats
    times; the first run warms the metadata / TLB, the others are AVERAGED into one row (one row per batch: no batch
    can sit on both sides of the train / test split)."""
    from . import trace_run
    rng = np.random.default_rng(seed)
    runner = trace_run.IterationRunner(Hq, Hkv, D, B, layers, pages_per_layer, budget, 1024, seed, device, layer_gemms,
                                       random_pool=True)
    raw, us = [], []
    for _ in range(n_samples):
        n_dec = int(rng.choice([0, 1, 4, 16, 64, 128, 256, 512])) if rng.random() < 0.8 else int(rng.integers(0, 513))
        med = float(rng.choice([256, 1024, 4096]))
        dctx = np.clip(np.rint(np.exp(np.log(med) + rng.standard_normal(n_dec))), 1, 32768).astype(np.int64)
        room = budget - n_dec
        q_len, ctx_off = [1] * n_dec, list(dctx - 1)
        if rng.random() < 0.75 and room > 0:                # most rounds carry prefill; many fill the budget
            fill = room if rng.random() < 0.5 else int(rng.integers(1, room + 1))
            while fill > 0 and len(q_len) < 1000:
                c = fill if rng.random() < 0.6 else int(rng.integers(1, fill + 1))
                q_len.append(c)
                ctx_off.append(int(rng.choice([0, 0, 512, 2048, 8192, 30720])) if rng.random() < 0.7 else int(rng.integers(0, 30720)))
                fill -= c
        if not q_len:
            continue
        need = [(int(c) + int(l) + B - 1) // B for l, c in zip(q_len, ctx_off)]
        if sum(need) > pages_per_layer:
            continue
        ids = rng.choice(pages_per_layer, size=sum(need), replace=False).astype(np.int32)
        tabs, pos = [], 0
        for n in need:
            tabs.append(ids[pos:pos + n])
            pos += n
        flags = [0] * n_dec + [binding.CP_REQ_PREFILL] * (len(q_len) - n_dec)      # a 1-token chunk is still prefill
        ts = []
        for r in range(repeats + 1):
            descs, keep = binding.make_descs(q_len, ctx_off, tabs, flags=flags)
            t, row, _ = runner.run(descs, len(q_len))
            if r > 0:
                ts.append(t)
        raw.append(list(row.feat))
        us.append(float(np.mean(ts)))
    runner.close()
    return np.asarray(raw, np.float64), np.asarray(us, np.float64)


def train_and_report(raw, us, seed=0, epochs=300, budget=2048):
    rng = np.random.default_rng(seed)
    ok = np.isfinite(us) & (us > 0)                           # "cleaned"
    raw, us = raw[ok], us[ok]
    X = features16(raw)
    tr, va, te, b = bucket_downsample_split(X[:, 12].astype(np.int64), rng, full_budget=budget)
    counts = np.bincount(b[tr], minlength=b.max() + 1).astype(np.float64)
    w = (counts[counts > 0].mean() / counts[b[tr]])          # bucket-aware sample weight (Eq. 5)
    # Reading of Eq. 5's per-sample weight w_i (the paper gives no formula): bucket weight x (median / y_i)^2, so that
    # the Huber term measures the RELATIVE error -- rounds range over two orders of magnitude in time, and Eq. 10
    # compares T_hat with T* for short and long candidate rounds alike.
    w = w * (float(np.median(us[tr])) / us[tr]) ** 2
    w = w / w.mean()
    lin = fit_linear(X[tr], us[tr], w)
    mlp = fit_mlp(X[tr], us[tr], w, X[va], us[va], epochs=epochs, seed=seed)
    bounds = (0.05 * float(np.median(us)), 0.10 * float(np.median(us)))
    rep = {"samples": int(len(us)), "train": int(len(tr)), "val": int(len(va)), "test": int(len(te)),
           "target_unit": "us (what IterationRunner.run returns: every layer of the round)", "median_us": float(np.median(us)),
           "linear_test": metrics(us[te], predict_linear(lin, X[te]), bounds),
           "mlp_test": metrics(us[te], predict_mlp(mlp, X[te]), bounds),
           "bounded_error_thresholds_us": list(bounds)}
    return rep, lin, mlp


def export_linear(model):
    coef, mu, inv = model
    return binding.CP_PRED_LINEAR, [float(x) for x in coef], [float(x) for x in mu], [float(x) for x in inv]


def export_mlp(model):
    flat, mu, inv = model[:3]
    return binding.CP_PRED_MLP, [float(x) for x in flat], [float(x) for x in mu], [float(x) for x in inv]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--samples", type=int, default=6000)
    ap.add_argument("--epochs", type=int, default=300)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    from . import build
    build.build()
    raw, us = harvest(a.samples, a.seed)
    rep, lin, mlp = train_and_report(raw, us, a.seed, a.epochs)
    if a.out:
        kind, wts, mu, inv = export_mlp(mlp)
        lk, lw, lmu, linv = export_linear(lin)
        with open(a.out, "w") as f:
            json.dump({"report": rep, "mlp": {"weights": wts, "mu": mu, "inv_sigma": inv},
                       "linear": {"weights": lw, "mu": lmu, "inv_sigma": linv}}, f)
    print(json.dumps(rep))


if __name__ == "__main__":
    main()
