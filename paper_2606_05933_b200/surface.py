"""Measured latency surface of one mixed_attention iteration over chunk-token budget x decode count x
context length (north_star): what a SlidingChunker-style batch latency predictor
(§3.2, Eq. 4-5, Table 1) would be fitted on.

    python -m paper_2606_05933_b200.surface --out gpurun_out/surface.csv [--with-c4]

One CSV row per point: config id, seed, R, T, x1..x7 (Table 1), algorithmic bytes and flops, t_HBM, t_TC,
roofline, measured us (median, p10, p90 over >= 30 timed iterations after >= 5 warm-ups, CUDA events on the
launching stream, L2 flushed between iterations outside the event window), fraction of the batch
roofline, and for mixed points overlap = t_mixed / (t_prefill_only + t_decode_only).

Needs a B200 and the built library (no CPU fallback).  Imports nothing from oracle/.
"""
from __future__ import annotations

import argparse
import csv
import sys
from pathlib import Path
from typing import List, Optional

import numpy as np

from . import accounting as acc
from . import workloads as wl
from .features import features, scene

FIELDS = ["point", "name", "seed", "shape", "kv_dtype", "scene", "R", "T", "chunk", "n_prefill", "n_decode", "ctx_median",
          "x1", "x2", "x3", "x4", "x5", "x6", "x7", "bytes", "flops", "t_hbm_us", "t_tc_us", "roofline_us", "bound",
          "median_us", "p10_us", "p90_us", "frac_of_roofline", "prefill_only_us", "decode_only_us", "overlap"]


def dense_points() -> List[tuple]:
    """Extra points between the grid lines (for the predictor fit): more chunk budgets and decode counts."""
    pts = []
    for nd in (0, 16, 48, 64, 96, 192):
        for C in (0, 128, 384, 768, 1536, 2048):
            for n in (1, 2):
                if (C == 0 and (nd == 0 or n == 2)):
                    continue
                pts.append((f"DN:{C},{n},{nd}", lambda C=C, n=n, nd=nd: wl.config_dense(C, n, nd)))
    return pts


def model_points(model: str) -> List[tuple]:
    """The same grid on another layer shape (one predictor model set per shape: latency depends on Hq/Hkv/D)."""
    Hq, Hkv, D = wl.MODEL_SHAPES[model]
    pts = []
    for nd in (32, 128):
        for C in (256, 512, 1024, 2048):
            for n in (1, 2, 4):
                pts.append((f"{model}/C3:{C},{n},{nd}", lambda C=C, n=n, nd=nd: wl.config_c3(C, n, nd, model=model)))
    for med in (500, 4000):
        for nd in (32, 128):
            for C in (0, 1024):
                pts.append((f"{model}/CTX:{C},1,{nd},m{med}", lambda C=C, nd=nd, med=med: wl.config_c3(C, 1, nd, ctx_median=med, model=model)))
    for nd in (16, 32, 64, 128, 192):
        pts.append((f"{model}/PD-{nd}", lambda nd=nd: wl.config_c3(0, 1, nd, model=model)))
    for i, (c, u) in enumerate([(256, 0), (512, 2048), (1024, 0), (1024, 4096), (2048, 0), (2048, 4096), (2048, 8192), (4096, 0),
                                (128, 1024), (768, 512), (1536, 3000), (384, 6000)]):
        pts.append((f"{model}/PP:{c},{u}", lambda c=c, u=u, i=i: wl.make_batch(f"PP-{model}-{c}-{u}", Hq, Hkv, D, [(c, u)], 7200 + i)))
    for i, rs in enumerate([[(512, 0), (512, 3000)], [(1024, 0), (1024, 6000)], [(256, 100), (256, 2000), (256, 4000), (256, 8000)]]):
        pts.append((f"{model}/PP2:{i}", lambda rs=rs, i=i: wl.make_batch(f"PP2-{model}-{i}", Hq, Hkv, D, rs, 7300 + i)))
    return pts


def surface_points(with_c4: bool = False, dense: bool = False, model: Optional[str] = None) -> List[tuple]:
    """(point id, Batch factory) for the whole grid, in a fixed order."""
    if model:
        return model_points(model)
    if dense:
        return dense_points()
    pts = []
    for nd in (32, 128):                                   # BASELINE.json configs[2]: the predictor grid
        for C in (256, 512, 1024, 2048):
            for n in (1, 2, 3, 4):
                pts.append((f"C3:{C},{n},{nd}", lambda C=C, n=n, nd=nd: wl.config_c3(C, n, nd)))
    for med in (500, 4000):                                # third axis: decode-context length
        for nd in (32, 128):
            for C in (0, 512, 2048):
                pts.append((f"CTX:{C},1,{nd},m{med}", lambda C=C, nd=nd, med=med: wl.config_c3(C, 1, nd, ctx_median=med)))
    for name in sorted(wl.SCENE_EDGES):                    # pure-prefill scene edges (tensor-bound)
        pts.append((name, lambda name=name: wl.config_scene_edge(name)))
    for name in ("PD-32", "PD-128", "PD-C2", "PD-C5"):     # pure-decode scene edges
        pts.append((name, lambda name=name: wl.config_decode_only(name)))
    for name in ("PD-32", "PD-128", "PD-C2", "PD-C5"):     # the same pure-decode edges over an FP8 E4M3 KV cache (NEXT-3)
        pts.append((name + "/fp8", lambda name=name: fp8_variant(wl.config_decode_only(name))))
    pts.append(("C2", wl.config_c2))
    pts.append(("C2-shuffled", lambda: wl.config_c2(shuffle=True)))
    pts.append(("C5", wl.config_c5))
    for name in ("PP-b", "PP-e", "PP-f"):                  # prefill and mixed batches over the FP8 cache
        pts.append((name + "/fp8", lambda name=name: fp8_variant(wl.config_scene_edge(name))))
    pts.append(("C2/fp8", lambda: fp8_variant(wl.config_c2())))
    pts.append(("C5/fp8", lambda: fp8_variant(wl.config_c5())))
    if with_c4:
        pts.append(("C4", wl.config_c4))
        pts.append(("C4/fp8", lambda: fp8_variant(wl.config_c4())))
    return pts


def fp8_variant(b: wl.Batch) -> wl.Batch:
    return wl.Batch(**{**b.__dict__, "name": b.name + "/fp8", "meta": {**b.meta, "kv_fp8": True}})


def sub_batch(b: wl.Batch, kind: str) -> Optional[wl.Batch]:
    """The prefill-only (c > 1) or decode-only (c == 1) part of a mixed batch, re-paged on its own pool."""
    reqs = [(c, u) for c, u in b.reqs if (c > 1 if kind == "prefill" else c == 1)]
    if not reqs:
        return None
    return wl.make_batch(f"{b.name}/{kind}", b.num_q_heads, b.num_kv_heads, b.head_dim, reqs, b.seed + 1,
                         with_append=False)


def time_batch(b: wl.Batch, device: str, iters: int, warmup: int, flush) -> np.ndarray:
    """us per ss_mixed_attention call (work list + main launch), one sample per timed iteration."""
    import torch
    from . import binding
    if b.meta.get("kv_fp8"):
        t = wl.make_tensors(b, device, caches=False)
        kc, vc, ks, vs = wl.make_fp8_caches(b, device)
        h = binding.handle_for(b, t, fp8_caches=(kc, vc), kv_scales=(ks, vs))
    else:
        t = wl.make_tensors(b, device)
        h = binding.handle_for(b, t)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    out = torch.empty_like(t.q)
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        flush.fill_(1)
        binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=out)
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(iters)]
    for e0, e1 in evs:
        flush.fill_(1)
        e0.record(stream)
        binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=out)
        e1.record(stream)
    torch.cuda.synchronize()
    us = np.array([e0.elapsed_time(e1) * 1e3 for e0, e1 in evs])
    h.close()
    del t, out, h
    torch.cuda.empty_cache()
    return us


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="gpurun_out/surface.csv")
    ap.add_argument("--iters", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--with-c4", action="store_true", help="include the 40 GB-pool decode-heavy config")
    ap.add_argument("--only", default=None, help="comma-separated point-id prefixes")
    ap.add_argument("--dense", action="store_true", help="the extra between-the-lines points instead of the grid")
    ap.add_argument("--model", default=None, help="run the grid on another layer shape (workloads.MODEL_SHAPES key)")
    args = ap.parse_args(argv)
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("surface sweep needs a CUDA device: the product path has no CPU fallback")
    device = "cuda:0"
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=device)
    peaks = acc.load_peaks()
    Path(args.out).parent.mkdir(parents=True, exist_ok=True)
    with open(args.out, "w", newline="") as f:
        wr = csv.DictWriter(f, fieldnames=FIELDS)
        wr.writeheader()
        for pid, make in surface_points(args.with_c4, args.dense, args.model):
            if args.only and not any(pid.startswith(p) for p in args.only.split(",")):
                continue
            b = make()
            us = time_batch(b, device, args.iters, args.warmup, flush)
            w, roof, x = acc.work(b), acc.roofline_us(b, peaks), features(b.reqs)
            row = {"point": pid, "name": b.name, "seed": b.seed, "shape": f"{b.num_q_heads}/{b.num_kv_heads}/{b.head_dim}", "kv_dtype": "fp8" if b.meta.get("kv_fp8") else "bf16",
                   "scene": scene(b.reqs), "R": b.R, "T": b.T, "chunk": b.meta.get("chunk", x["x6"]),
                   "n_prefill": sum(1 for c, _ in b.reqs if c > 1), "n_decode": x["x4"],
                   "ctx_median": b.meta.get("ctx_median", ""), **x, "bytes": w["bytes"], "flops": w["flops"],
                   "t_hbm_us": round(roof["t_hbm_us"], 2), "t_tc_us": round(roof["t_tc_us"], 2),
                   "roofline_us": round(roof["roofline_us"], 2), "bound": roof["bound"],
                   "median_us": round(float(np.median(us)), 2), "p10_us": round(float(np.percentile(us, 10)), 2),
                   "p90_us": round(float(np.percentile(us, 90)), 2),
                   "frac_of_roofline": round(roof["roofline_us"] / float(np.median(us)), 4),
                   "prefill_only_us": "", "decode_only_us": "", "overlap": ""}
            if scene(b.reqs) == "mixed":
                tp = float(np.median(time_batch(sub_batch(b, "prefill"), device, args.iters, args.warmup, flush)))
                td = float(np.median(time_batch(sub_batch(b, "decode"), device, args.iters, args.warmup, flush)))
                row.update(prefill_only_us=round(tp, 2), decode_only_us=round(td, 2),
                           overlap=round(float(np.median(us)) / (tp + td), 4))
            wr.writerow(row)
            f.flush()
            print(pid, row["median_us"], row["roofline_us"], row["frac_of_roofline"], row["overlap"], file=sys.stderr, flush=True)


if __name__ == "__main__":
    main()
