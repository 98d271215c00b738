"""A Fig. 1-style two-iteration example (Figure 1) with B200 latencies.

The paper's figure: two consecutive iterations with TBT deadlines; "Single-step" takes the largest chunk the CURRENT
deadline allows and is left with a small chunk in the next iteration; SlidingChunker (Algorithm 1)
takes a slightly smaller chunk now so that both iterations run in an efficient range.  Here the iteration time is the
one this library produces - one layer's mixed attention on a B200 - so the deadlines are in microseconds:

  * the latency model T_hat is the paper's linear predictor (Eq. 5) fitted, with non-negative weights, on the measured
    surface (`profiles/r2_surface*.csv`, written by `surface.py` on the GPU);
  * Single-step: b1 = TimeToBudget(T_cur), b2 = TimeToBudget(T_next)                      (Eq. 14-15 give T_cur, T_next)
  * SlidingChunker: B* = argmin_b T_hat(b) + T_hat(B_sigma - b), B_sigma = b1 + b2 (Eq. 16), then B_sigma - B*;
  * both strategies move the same B_sigma tokens; what differs is the time the two iterations take, i.e. how many
    tokens are done when the second deadline expires.

    python -m paper_2606_05933_b200.fig1_example [--measure] [--out table.md]

`--measure` (needs a B200) also RUNS the four batches through ss_mixed_attention, with the state carried from the first
iteration to the second (the prefill request's cached length grows by its chunk, every decode context by one), and
prints the measured microseconds beside the predicted ones.  Host logic only otherwise; imports nothing from oracle/.
"""
from __future__ import annotations

import argparse
import sys
from pathlib import Path
from typing import List, Sequence, Tuple

import numpy as np

from .chunker import BatchForwarder, PrefillState, sliding_chunker, surface_predict_fn
from .predictor import BatchLatencyPredictor, load_surface

ROOT = Path(__file__).resolve().parent.parent
SURFACES = [ROOT / "profiles" / "r2_surface.csv", ROOT / "profiles" / "r2_surface_dense.csv"]
SHAPE = (32, 8, 128)                 # Llama-3-8B-shaped layer (BASELINE.json configs[1], [2])


def scenario(seed: int = 11):
    """64 decodes with contexts U{512..4096} (C2's recipe) + one 8192-token prompt of which 1024 tokens are cached;
    chunk budget B = 4096; the protected decodes leave T_cur = 180 us now and T_next = 135 us for the next iteration."""
    rng = np.random.default_rng(seed)
    decodes = [int(u) for u in rng.integers(512, 4096, size=64, endpoint=True)]
    prefills = [PrefillState(remaining=8192 - 1024, cached=1024)]
    return decodes, prefills, 4096, 180.0, 135.0


def fitted_forwarder(max_budget: int) -> BatchForwarder:
    paths = [str(p) for p in SURFACES if p.exists()]
    if not paths:
        raise SystemExit("no committed latency surface under profiles/ (run surface.py on a B200 first)")
    rows, X, y, scenes, shapes = load_surface(paths)
    keep = [i for i, s in enumerate(shapes) if s == "%d/%d/%d" % SHAPE]          # load_surface keeps bf16-cache points only
    p = BatchLatencyPredictor(fit="nnls").fit(X[keep], y[keep], [scenes[i] for i in keep])
    return BatchForwarder(surface_predict_fn(p), max_budget)


def plan(F: BatchForwarder, decodes, prefills, t_cur: float, t_next: float):
    """((b1, b2) single-step, (b1, b2) sliding, B_sigma)."""
    g1 = F.time_to_budget(decodes, prefills, t_cur)
    g2 = F.time_to_budget(decodes, prefills, t_next)
    b_star, _, _, b_sigma = sliding_chunker(F, decodes, prefills, t_cur, t_next)
    return (g1, g2), (b_star, b_sigma - b_star), b_sigma


def iteration_batches(decodes: Sequence[int], prefills: Sequence[PrefillState], budgets: Tuple[int, int], F: BatchForwarder):
    """The two iterations' request lists [(c, u)] with the state carried over, and their predicted times."""
    dec = list(decodes)
    pre = [PrefillState(p.remaining, p.cached) for p in prefills]
    out = []
    for b in budgets:
        t_hat, alloc = F.forward(dec, pre, b)
        reqs = [(1, u) for u in dec] + [(c, p.cached) for c, p in zip(alloc, pre) if c > 0]
        out.append((reqs, t_hat, sum(alloc)))
        dec = [u + 1 for u in dec]
        pre = [PrefillState(p.remaining - c, p.cached + c) for c, p in zip(alloc, pre)]
    return out


def measure_us(reqs, seed: int, iters: int = 30) -> float:
    """Median us of ss_mixed_attention on this batch (CUDA events, L2 flushed between iterations)."""
    import torch
    from . import surface, workloads as wl
    b = wl.make_batch("fig1", *SHAPE, list(reqs), seed, with_append=False)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda:0")
    return float(np.median(surface.time_batch(b, "cuda:0", iters, 5, flush)))


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--measure", action="store_true", help="also run the four batches on cuda:0")
    ap.add_argument("--out", default=None)
    args = ap.parse_args(argv)
    decodes, prefills, B, t_cur, t_next = scenario()
    F = fitted_forwarder(B)
    single, sliding, b_sigma = plan(F, decodes, prefills, t_cur, t_next)
    lines = ["| strategy | iteration | budget b (tokens) | prefill chunk | T_hat us (predictor) | measured us (B200) |",
             "|---|---|---|---|---|---|"]
    totals = {}
    for name, budgets in (("Single-step", single), ("SlidingChunker", sliding)):
        its = iteration_batches(decodes, prefills, budgets, F)
        tot_hat, tot_meas, chunk_tokens = 0.0, 0.0, 0
        for k, ((reqs, t_hat, chunk), b) in enumerate(zip(its, budgets)):
            meas = measure_us(reqs, 900 + k) if args.measure else float("nan")
            lines.append(f"| {name} | {k + 1} | {b} | {chunk} | {t_hat:.1f} | {meas:.1f} |" if args.measure
                         else f"| {name} | {k + 1} | {b} | {chunk} | {t_hat:.1f} | - |")
            tot_hat += t_hat
            tot_meas += meas
            chunk_tokens += chunk
        totals[name] = (tot_hat, tot_meas, chunk_tokens)
        lines.append(f"| {name} | both | {sum(budgets)} | {chunk_tokens} | {tot_hat:.1f} | "
                     + (f"{tot_meas:.1f} |" if args.measure else "- |"))
    head = [f"Scenario: {len(decodes)} decodes (contexts U{{512..4096}}), one prompt with {prefills[0].remaining} tokens left "
            f"({prefills[0].cached} cached), B = {B}, T_cur = {t_cur:.0f} us, T_next = {t_next:.0f} us, B_sigma = {b_sigma}.", ""]
    s_hat, s_meas, _ = totals["Single-step"]
    c_hat, c_meas, _ = totals["SlidingChunker"]
    tail = ["", f"Two-iteration time for the same {b_sigma} tokens: predictor {s_hat:.1f} -> {c_hat:.1f} us"
            + (f", measured {s_meas:.1f} -> {c_meas:.1f} us" if args.measure else "") + "."]
    text = "\n".join(head + lines + tail) + "\n"
    sys.stdout.write(text)
    if args.out:
        Path(args.out).parent.mkdir(parents=True, exist_ok=True)
        Path(args.out).write_text(text)


if __name__ == "__main__":
    main()
