"""Batch Latency Predictor of the paper (§3.2) fitted on OUR measured latency surface
(SURVEY.md §8(f) NEXT-1).  Host-side numpy only; it consumes the CSV that `surface.py` writes on the GPU.

Model (Eq. 5, index read as j = 1..7, reading 13):  T_hat = b^(m) + sum_j w_j^(m) x_j  with
the 7 features of Table 1, a global model trained on all samples and a scene expert model
(pure decode / pure prefill / mixed, Eq. 3) for every scene with at least `min_expert_samples`
samples; inference uses the expert if one exists, else the global model.  The paper names the
threshold but gives no value: 12 here (reading 15).  Fit = ordinary least squares (the paper says
"lightweight ... linear"; no regulariser is mentioned), features scaled to unit max for conditioning only.

    python -m paper_2606_05933_b200.predictor profiles/r1_v4_surface.csv profiles/r1_v4_surface_dense.csv

prints MAE / RMSE / R^2 the way Table 5 does, in-sample and leave-one-out.
"""
from __future__ import annotations

import csv
import sys
from typing import Dict, List, Optional, Sequence

import numpy as np

FEATURES = ["x1", "x2", "x3", "x4", "x5", "x6", "x7"]
SCENES = ["pure_decode", "pure_prefill", "mixed"]


class LinearLatencyModel:
    """T_hat = b + w . x  (Eq. 5), least squares."""

    def __init__(self):
        self.scale: Optional[np.ndarray] = None
        self.coef: Optional[np.ndarray] = None

    def fit(self, X: np.ndarray, y: np.ndarray) -> "LinearLatencyModel":
        X = np.asarray(X, dtype=np.float64)
        self.scale = np.maximum(np.abs(X).max(axis=0), 1.0)
        A = np.hstack([np.ones((X.shape[0], 1)), X / self.scale])
        self.coef, *_ = np.linalg.lstsq(A, np.asarray(y, dtype=np.float64), rcond=None)
        return self

    def predict(self, X: np.ndarray) -> np.ndarray:
        X = np.atleast_2d(np.asarray(X, dtype=np.float64))
        return self.coef[0] + (X / self.scale) @ self.coef[1:]

    @property
    def intercept(self) -> float:
        return float(self.coef[0])

    @property
    def weights(self) -> np.ndarray:
        return self.coef[1:] / self.scale


class BatchLatencyPredictor:
    """Global model + scene experts."""

    def __init__(self, min_expert_samples: int = 12):
        self.min_expert_samples = min_expert_samples
        self.global_model = LinearLatencyModel()
        self.experts: Dict[str, LinearLatencyModel] = {}

    def fit(self, X: np.ndarray, y: np.ndarray, scenes: Sequence[str]) -> "BatchLatencyPredictor":
        X, y, scenes = np.asarray(X, dtype=np.float64), np.asarray(y, dtype=np.float64), np.asarray(scenes)
        self.global_model.fit(X, y)
        self.experts = {}
        for sc in SCENES:
            idx = scenes == sc
            if int(idx.sum()) >= self.min_expert_samples:
                self.experts[sc] = LinearLatencyModel().fit(X[idx], y[idx])
        return self

    def predict(self, X: np.ndarray, scenes: Sequence[str]) -> np.ndarray:
        X = np.atleast_2d(np.asarray(X, dtype=np.float64))
        out = np.empty(X.shape[0])
        for i, sc in enumerate(scenes):
            out[i] = self.experts.get(sc, self.global_model).predict(X[i:i + 1])[0]
        return out


def scores(y: np.ndarray, yhat: np.ndarray) -> Dict[str, float]:
    err = yhat - y
    ss_res, ss_tot = float((err ** 2).sum()), float(((y - y.mean()) ** 2).sum())
    return {"mae": float(np.abs(err).mean()), "rmse": float(np.sqrt((err ** 2).mean())),
            "r2": 1.0 - ss_res / ss_tot if ss_tot > 0 else float("nan")}


def load_surface(path):
    """One CSV path, or several (grid + dense points) to be concatenated."""
    paths = [path] if isinstance(path, str) else list(path)
    rows = [r for p in paths for r in csv.DictReader(open(p))]
    X = np.array([[float(r[f]) for f in FEATURES] for r in rows])
    y = np.array([float(r["median_us"]) for r in rows])
    scenes = [r["scene"] for r in rows]
    shapes = [r["shape"] for r in rows]
    return rows, X, y, scenes, shapes


def evaluate(path: str, shape: str = "32/8/128", min_expert_samples: int = 12) -> Dict[str, Dict[str, float]]:
    """In-sample and leave-one-out fidelity on the points of one layer shape (latency depends on the shape)."""
    rows, X, y, scenes, shapes = load_surface(path)
    keep = [i for i, s in enumerate(shapes) if s == shape]
    X, y, scenes = X[keep], y[keep], [scenes[i] for i in keep]
    p = BatchLatencyPredictor(min_expert_samples).fit(X, y, scenes)
    res = {"n": {"points": len(keep), **{sc: scenes.count(sc) for sc in SCENES}},
           "experts": {sc: 1.0 for sc in p.experts},
           "in_sample": scores(y, p.predict(X, scenes)),
           "global_only_in_sample": scores(y, p.global_model.predict(X))}
    loo = np.empty(len(y))
    for i in range(len(y)):
        m = np.ones(len(y), dtype=bool)
        m[i] = False
        q = BatchLatencyPredictor(min_expert_samples).fit(X[m], y[m], [s for s, k in zip(scenes, m) if k])
        loo[i] = q.predict(X[i:i + 1], [scenes[i]])[0]
    res["leave_one_out"] = scores(y, loo)
    res["mean_latency_us"] = {"value": float(y.mean())}
    return res


def main(argv: Optional[List[str]] = None):
    argv = sys.argv[1:] if argv is None else argv
    path = argv if argv else ["profiles/r1_v4_surface.csv", "profiles/r1_v4_surface_dense.csv"]
    res = evaluate(path)
    print(f"surface: {path}  points (8B shape): {res['n']}")
    print(f"experts trained for: {sorted(res['experts'])}")
    for k in ("in_sample", "global_only_in_sample", "leave_one_out"):
        r = res[k]
        print(f"{k:24s} MAE {r['mae']:.2f} us  RMSE {r['rmse']:.2f} us  R^2 {r['r2']:.4f}")
    print(f"mean latency {res['mean_latency_us']['value']:.1f} us")


if __name__ == "__main__":
    main()
