"""Offline half of the LPRS latency predictor: Tables 1-2 features, Eq. 5 loss,
Eq. 15-17 metrics, the bucketing / 8:1:1 split, and that an exported model means the same thing to
the numpy forward, the reference scheduler and the C++ scheduler."""
import numpy as np
import pytest

from oracle import ref_scheduler as rs
from paper_2606_09061_b200 import binding, build, predictor as pr


def test_features16_match_tables_1_and_2():
    raw = np.array([[300., 4., 6., 1000., 700., 5000., 4096., 10., 20., 5., 8.],
                    [0., 0., 1., 0., 0., 0., 0., 1., 2., 3., 4.]])
    X = pr.features16(raw)
    assert X.shape == (2, 16) and np.array_equal(X[:, :11], raw)
    # bias, scheduled_tokens, avg_decode_ctx, decode_ctx_interaction, prefill_interaction
    assert X[0, 11:].tolist() == [1.0, 304.0, 250.0, 1000.0, 1.5e6]
    assert X[1, 11:].tolist() == [1.0, 0.0, 0.0, 0.0, 0.0]          # max(decode_tokens, 1) guards the division
    # the reference scheduler builds the same vector from its own state
    ref = rs.RefScheduler(rs.SchedConfig(num_blocks=16, page_mb=0.0))
    x = ref.features(4, 1000, 700, 300, 2, 5000, 4096)
    assert x[:7] == raw[0, :7].tolist() and x[11:] == X[0, 11:].tolist()


def test_metrics_closed_forms():
    y = np.array([10.0, 20.0, 40.0, 50.0])
    m = pr.metrics(y, y + np.array([1.0, -2.0, 4.0, -5.0]), bounds=(2.0, 5.0))
    assert m["mae"] == 3.0 and m["rmse"] == pytest.approx(np.sqrt(46 / 4))          # Eq. 15-16
    assert m["mape_pct"] == pytest.approx(100 * (0.1 + 0.1 + 0.1 + 0.1) / 4)        # Eq. 17
    assert m["within_2"] == 0.5 and m["within_5"] == 1.0 and m["p50"] == 3.0


def test_asymmetric_huber_eq5():
    torch = pytest.importorskip("torch")
    y = torch.zeros(4)
    y_hat = torch.tensor([0.5, -0.5, 3.0, -3.0])
    w = torch.tensor([1.0, 1.0, 2.0, 2.0])
    got = float(pr.asymmetric_huber(y_hat, y, w, delta=1.0, under=2.0))
    # quadratic inside delta, linear outside, under-estimates (y_hat < y) doubled, weights applied, mean
    want = (0.125 + 2 * 0.125 + 2 * 2.5 + 2 * 2 * 2.5) / 4
    assert got == pytest.approx(want)


def test_bucket_downsample_and_split():
    rng = np.random.default_rng(0)
    tokens = np.concatenate([np.full(900, 2048), rng.integers(1, 2048, 300)])
    tr, va, te, b = pr.bucket_downsample_split(tokens, rng)
    kept = np.concatenate([tr, va, te])
    assert len(set(kept)) == len(kept)
    full = (b[kept] == 8).sum()
    assert full == np.bincount(b[b < 8]).max()                   # full-budget bucket cut to the largest other bucket
    assert abs(len(tr) / len(kept) - 0.8) < 0.01 and abs(len(va) / len(kept) - 0.1) < 0.01


def test_linear_fit_recovers_planted_model_and_exports_to_both_schedulers():
    build.build()
    rng = np.random.default_rng(1)
    raw = np.abs(rng.standard_normal((400, 11))) * np.array([500, 100, 100, 1e5, 3e4, 2e4, 2e4, 0, 0, 0, 0]) + np.array([0.0] * 7 + [10, 20, 5, 8])
    X = pr.features16(raw)
    true = 37.5 + 0.31 * X[:, 12] + 0.0021 * X[:, 14] + 1.3e-5 * X[:, 15]
    model = pr.fit_linear(X, true)
    assert np.abs(pr.predict_linear(model, X) - true).max() < 1e-6 * true.max()
    kind, w, mu, inv = pr.export_linear(model)
    kw = dict(mode=rs.MODE_LPRS, num_blocks=64, pred_kind=kind, pred_weights=w, feat_mu=mu, feat_inv_sigma=inv)
    ref, cpp = rs.RefScheduler(rs.SchedConfig(**kw)), binding.Scheduler(**kw)
    for i in range(20):
        x = X[i].tolist()
        assert cpp.cp_sched_predict(x) == ref.predict(x)                               # bit-exact
        assert ref.predict(x) == pytest.approx(true[i], rel=1e-9)


def test_mlp_export_means_the_same_everywhere():
    pytest.importorskip("torch")
    build.build()
    rng = np.random.default_rng(2)
    raw = np.abs(rng.standard_normal((600, 11))) * np.array([500, 100, 100, 1e5, 3e4, 2e4, 2e4, 0, 0, 0, 0]) + np.array([0.0] * 7 + [10, 20, 5, 8])
    X = pr.features16(raw)
    y = 40 + 0.3 * X[:, 12] + 2e-3 * X[:, 14] + 1e-5 * X[:, 15]
    model = pr.fit_mlp(X[:500], y[:500], np.ones(500), X[500:], y[500:], epochs=40)
    assert len(model[0]) == rs.mlp_num_weights()
    y_hat = pr.predict_mlp(model, X[500:])
    assert pr.metrics(y[500:], y_hat)["mape_pct"] < 25.0                               # it learned something
    kind, w, mu, inv = pr.export_mlp(model)
    kw = dict(mode=rs.MODE_LPRS, num_blocks=64, pred_kind=kind, pred_weights=w, feat_mu=mu, feat_inv_sigma=inv)
    ref, cpp = rs.RefScheduler(rs.SchedConfig(**kw)), binding.Scheduler(**kw)
    for i in range(500, 520):
        x = X[i].tolist()
        assert cpp.cp_sched_predict(x) == ref.predict(x)                               # bit-exact, sequential fp64
        assert ref.predict(x) == pytest.approx(y_hat[i - 500], rel=1e-9, abs=1e-9)     # = the vectorised forward
