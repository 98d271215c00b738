"""Batch Latency Predictor of the paper (§3.2) fitted on OUR measured latency surface
(SURVEY.md §8(f) NEXT-1).  Host-side numpy only; it consumes the CSV that `surface.py` writes on the GPU.

Model (Eq. 5, index read as j = 1..7, reading 13):  T_hat = b^(m) + sum_j w_j^(m) x_j  with
the 7 features of Table 1, a global model trained on all samples and a scene expert model
(pure decode / pure prefill / mixed, Eq. 3) for every scene with at least `min_expert_samples`
samples; inference uses the expert if one exists, else the global model.  The paper names the
threshold but gives no value: 12 here (reading 15).

Fit.  The paper says only "lightweight ... linear"; no regulariser or constraint is mentioned.  Two fits are offered:
  "ols"   ordinary least squares (round 1): best in-sample error, but on a small surface it takes negative weights on
          x6 / x7, so T_hat is NOT monotone in the token budget;
  "nnls"  (default) least squares with a free intercept and NON-NEGATIVE weights on the basis
          (x1 - x2/2, x2, x3, ..., x7) (Lawson-Hanson via scipy.optimize.nnls), mapped back to weights on x1..x7, so
          the model is still Eq. 5's linear form; the only weight that may be negative is w2 >= -w1/2.  Why this
          basis: a causal chunk visits c*u + c(c+1)/2 = x1 - x2/2 + x6/2 (row, key) pairs, so the physical weight
          of x2 IS negative; every basis element is a count of work that is non-decreasing in the token budget
          (d/dc [c(u+c) - c^2/2] = u + c >= 0), hence Pred(b) is non-decreasing in b, which TimeToBudget's binary
          search needs (reading 16).
Features are scaled to unit max for conditioning only.

    python -m paper_2606_05933_b200.predictor [--shape 32/8/128] [--fit nnls|ols] surface.csv [more.csv ...]

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
    """T_hat = b + w . x  (Eq. 5), least squares; fit = "nnls" (w >= 0, intercept free) or "ols"."""

    def __init__(self, fit: str = "nnls"):
        if fit not in ("nnls", "ols"):
            raise ValueError(fit)
        self.fit_mode = fit
        self.scale: Optional[np.ndarray] = None
        self.coef: Optional[np.ndarray] = None

    def fit(self, X: np.ndarray, y: np.ndarray) -> "LinearLatencyModel":
        X, y = np.asarray(X, dtype=np.float64), np.asarray(y, dtype=np.float64)
        self.scale = np.maximum(np.abs(X).max(axis=0), 1.0)
        Xs = X / self.scale
        if self.fit_mode == "ols":
            A = np.hstack([np.ones((X.shape[0], 1)), Xs])
            self.coef, *_ = np.linalg.lstsq(A, y, rcond=None)
        else:
            from scipy.optimize import nnls
            # basis z = (x1 - x2/2, x2, x3..x7) in scaled units; free intercept = difference of two non-negative
            # columns (+1, -1); a >= 0 on the basis, then w1 = a1, w2 = a2 - a1/2 (in unscaled units)
            Z = X.copy()
            Z[:, 0] = X[:, 0] - 0.5 * X[:, 1]
            zs = np.maximum(np.abs(Z).max(axis=0), 1.0)
            A = np.hstack([np.ones((X.shape[0], 1)), -np.ones((X.shape[0], 1)), Z / zs])
            z, _ = nnls(A, y, maxiter=50 * A.shape[1])
            a = z[2:] / zs                                   # unscaled basis weights
            w = a.copy()
            w[1] = a[1] - 0.5 * a[0]
            self.coef = np.concatenate([[z[0] - z[1]], w * self.scale])
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

    def __init__(self, min_expert_samples: int = 12, fit: str = "nnls"):
        self.min_expert_samples = min_expert_samples
        self.fit_mode = fit
        self.global_model = LinearLatencyModel(fit)
        self.experts: Dict[str, LinearLatencyModel] = {}

    def fit(self, X: np.ndarray, y: np.ndarray, scenes: Sequence[str]) -> "BatchLatencyPredictor":
        X, y, scenes = np.asarray(X, dtype=np.float64), np.asarray(y, dtype=np.float64), np.asarray(scenes)
        self.global_model.fit(X, y)
        self.experts = {}
        for sc in SCENES:
            idx = scenes == sc
            if int(idx.sum()) >= self.min_expert_samples:
                self.experts[sc] = LinearLatencyModel(self.fit_mode).fit(X[idx], y[idx])
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
    # one model set per layer shape AND cache type: points measured over an FP8 KV cache (point id .../fp8) move half
    # the bytes and are left out of the bf16 fit
    rows = [r for r in rows if r.get("kv_dtype", "fp8" if r["point"].endswith("/fp8") else "bf16") == "bf16"]
    X = np.array([[float(r[f]) for f in FEATURES] for r in rows])
    y = np.array([float(r["median_us"]) for r in rows])
    scenes = [r["scene"] for r in rows]
    shapes = [r["shape"] for r in rows]
    return rows, X, y, scenes, shapes


def evaluate(path, shape: str = "32/8/128", min_expert_samples: int = 12, fit: str = "nnls") -> Dict[str, Dict[str, float]]:
    """In-sample and leave-one-out fidelity on the points of one layer shape (latency depends on the shape)."""
    rows, X, y, scenes, shapes = load_surface(path)
    keep = [i for i, s in enumerate(shapes) if s == shape]
    X, y, scenes = X[keep], y[keep], [scenes[i] for i in keep]
    p = BatchLatencyPredictor(min_expert_samples, fit).fit(X, y, scenes)
    res = {"n": {"points": len(keep), **{sc: scenes.count(sc) for sc in SCENES}},
           "experts": {sc: 1.0 for sc in p.experts},
           "in_sample": scores(y, p.predict(X, scenes)),
           "global_only_in_sample": scores(y, p.global_model.predict(X))}
    loo = np.empty(len(y))
    for i in range(len(y)):
        m = np.ones(len(y), dtype=bool)
        m[i] = False
        q = BatchLatencyPredictor(min_expert_samples, fit).fit(X[m], y[m], [s for s, k in zip(scenes, m) if k])
        loo[i] = q.predict(X[i:i + 1], [scenes[i]])[0]
    res["leave_one_out"] = scores(y, loo)
    res["mean_latency_us"] = {"value": float(y.mean())}
    res["weights"] = {sc: {"intercept": m.intercept, **{f: float(w) for f, w in zip(FEATURES, m.weights)}}
                      for sc, m in [("global", p.global_model), *p.experts.items()]}
    return res


def main(argv: Optional[List[str]] = None):
    import argparse
    ap = argparse.ArgumentParser()
    ap.add_argument("--shape", default="32/8/128")
    ap.add_argument("--fit", default="nnls", choices=["nnls", "ols"])
    ap.add_argument("csv", nargs="+")
    args = ap.parse_args(argv)
    res = evaluate(args.csv, shape=args.shape, fit=args.fit)
    print(f"surface: {args.csv}  shape {args.shape}  fit {args.fit}  points: {res['n']}")
    print(f"experts trained for: {sorted(res['experts'])}")
    for k in ("in_sample", "global_only_in_sample", "leave_one_out"):
        r = res[k]
        print(f"{k:24s} MAE {r['mae']:.2f} us  RMSE {r['rmse']:.2f} us  R^2 {r['r2']:.4f}")
    print(f"mean latency {res['mean_latency_us']['value']:.1f} us")
    for sc, w in res["weights"].items():
        print(f"weights[{sc}]: " + "  ".join(f"{k}={v:.4g}" for k, v in w.items()))


if __name__ == "__main__":
    main()
