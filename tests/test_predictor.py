"""Batch latency predictor (§3.2, Eq. 4-5, Table 1) — host-side, CPU only."""
import numpy as np

from paper_2606_05933_b200.features import features, scene
from paper_2606_05933_b200.predictor import BatchLatencyPredictor, LinearLatencyModel, scores


def _batches(rng, n):
    out = []
    for _ in range(n):
        kind = rng.integers(0, 3)
        reqs = []
        if kind != 0:
            reqs += [(int(rng.integers(2, 2048)), int(rng.integers(0, 4096))) for _ in range(rng.integers(1, 4))]
        if kind != 1:
            reqs += [(1, int(rng.integers(1, 8192))) for _ in range(rng.integers(1, 128))]
        out.append(reqs)
    return out


def test_linear_model_recovers_exact_linear_latency():
    rng = np.random.default_rng(0)
    bs = _batches(rng, 200)
    X = np.array([[features(b)[f"x{j}"] for j in range(1, 8)] for b in bs], dtype=np.float64)
    w = np.array([3e-6, -1e-6, 2e-4, 0.05, 4e-4, 1e-3, 2e-3])
    y = 7.0 + X @ w
    m = LinearLatencyModel().fit(X, y)
    assert abs(m.intercept - 7.0) < 1e-6 and np.allclose(m.weights, w, rtol=1e-6, atol=1e-12)
    s = scores(y, m.predict(X))
    assert s["mae"] < 1e-6 and s["r2"] > 1 - 1e-12


def test_scene_experts_and_fallback_to_global():
    rng = np.random.default_rng(1)
    bs = _batches(rng, 300)
    sc = [scene(b) for b in bs]
    X = np.array([[features(b)[f"x{j}"] for j in range(1, 8)] for b in bs], dtype=np.float64)
    # scene-dependent intercepts: only expert models can fit this exactly
    base = {"pure_decode": 5.0, "pure_prefill": 40.0, "mixed": 15.0}
    y = np.array([base[s] for s in sc]) + X[:, 4] * 4e-4 + X[:, 0] * 3e-6
    p = BatchLatencyPredictor(min_expert_samples=12).fit(X, y, sc)
    assert set(p.experts) == {"pure_decode", "pure_prefill", "mixed"}
    assert scores(y, p.predict(X, sc))["mae"] < 1e-6
    assert scores(y, p.global_model.predict(X))["mae"] > 0.1
    # too few samples of one scene -> no expert, the global model answers
    keep = [i for i, s in enumerate(sc) if s != "pure_prefill"][:100] + [i for i, s in enumerate(sc) if s == "pure_prefill"][:3]
    q = BatchLatencyPredictor(min_expert_samples=12).fit(X[keep], y[keep], [sc[i] for i in keep])
    assert "pure_prefill" not in q.experts
    i = [i for i, s in enumerate(sc) if s == "pure_prefill"][0]
    assert q.predict(X[i:i + 1], ["pure_prefill"])[0] == q.global_model.predict(X[i:i + 1])[0]
