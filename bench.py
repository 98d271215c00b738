#!/usr/bin/env python
"""bench.py — one JSON line for the driver.

A "step" = one pass of the whole hot path over one synthetic batch: kv_append of the batch's new tokens
(a1) + mixed_attention (a2 work list, a3 prefill tiles, a4 decode splits, a5 merge), through the C ABI.
Workload at N=1: BASELINE.json configs[1] ("C2": Llama-3-8B-shaped layer, 512-token chunk at ctx 1024 +
64 decodes ctx U{512..4096}); other configs via --workload.  Metric: BASELINE.json's "mixed prefill+decode
attention us/iter and % of HBM/tensor roofline" -> value = microseconds per iteration (lower is better),
roofline fraction in the `roofline` object.  N>1: independent replicas, one per GPU (DESIGN.md "Multi-GPU":
replicas only, no collective on the data path); value = max-over-ranks time / (N*K) iterations.

--impl reference times the fp64 CPU oracle (oracle/) as it stands on the host cores, on a bounded row
sample per step, extrapolated to the whole batch by visible-pair count.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "mixed prefill+decode attention us/iter and % of HBM/tensor roofline"
UNIT = "us/iter"


def get_batch(name: str):
    from paper_2606_05933_b200 import workloads as wl
    if name == "C1":
        return wl.config_tiny()
    if name == "C2":
        return wl.config_c2()
    if name == "C4":
        return wl.config_c4()
    if name == "C5":
        return wl.config_c5()
    if name.startswith("PP-"):
        return wl.config_scene_edge(name)
    if name.startswith("PD-"):
        return wl.config_decode_only(name)
    if name.startswith("C3:"):
        C, n, nd = (int(x) for x in name[3:].split(","))
        return wl.config_c3(C, n, nd)
    raise SystemExit(f"unknown workload {name}")


class ClockSampler(threading.Thread):
    """Samples SM clock and clock-event reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._halt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.dev = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                 "hw_power_brake": 0x80}
        while not self._halt.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM)))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.dev))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.dev))
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._halt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def visible_device_index() -> int:
    import torch
    idx = torch.cuda.current_device()
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[idx])
        except Exception:
            return idx
    return idx


# ------------------------------------------------------------------------------------------------
# Multi-GPU bookkeeping (replicas only, no collective on the data path).  Kept free of CUDA so
# the world-size-2 gloo test can run it on CPU.
def max_over_ranks(x: float, world: int, device="cpu") -> float:
    """Device time of the slowest rank (all_reduce MAX over the default process group)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_metric(total_ms_max: float, steps: int, world: int):
    """N independent replicas each finish one batch per step: (ms per step, whole-job us per iteration)."""
    ms_per_step = total_ms_max / steps
    return ms_per_step, ms_per_step * 1e3 / world


def reference_rank_runs(rank: int) -> bool:
    """--impl reference: rank 0 alone runs and prints; the other ranks exit 0 without work."""
    return rank == 0


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """Oracle arm: rank 0 only; each step = the oracle on a bounded row sample of the workload."""
    if not reference_rank_runs(int(os.environ.get("RANK", "0"))):
        return
    import oracle
    from paper_2606_05933_b200 import workloads as wl, accounting as acc
    from paper_2606_05933_b200.features import causal_pairs
    b = get_batch(args.workload)
    t = wl.make_tensors(b, "cpu")
    k, v = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    qh, kn, vn = wl.to_u16(t.q), wl.to_u16(t.k_new), wl.to_u16(t.v_new)
    oracle.kv_append(k, v, kn, vn, b.block_table, b.query_start_loc, b.ctx_lens)
    total_pairs = causal_pairs(b.reqs)
    cores = oracle.num_threads()
    # size the per-step sample: total budget ~150 s over (steps + warmup) steps
    rng = np.random.default_rng(0)
    probe_rows = np.sort(rng.choice(b.T, size=min(b.T, 4 * cores), replace=False)).astype(np.int32)
    t0 = time.perf_counter()
    _, _, probe_pairs = oracle.mixed_attention(qh, k, v, b.block_table, b.query_start_loc, b.ctx_lens, b.scale, rows=probe_rows)
    rate = probe_pairs / max(time.perf_counter() - t0, 1e-6)          # pairs per second
    budget_s = min(150.0 / max(args.steps + args.warmup, 1), 30.0)
    want_pairs = min(total_pairs, max(int(rate * budget_s), 1))
    order = rng.permutation(b.T)
    row_pairs = np.empty(b.T, dtype=np.int64)
    for r, (c, u) in enumerate(b.reqs):
        s = int(b.query_start_loc[r])
        row_pairs[s:s + c] = u + 1 + np.arange(c)
    csum = np.cumsum(row_pairs[order])
    n_rows = int(min(b.T, np.searchsorted(csum, want_pairs) + 1))
    rows = np.sort(order[:n_rows]).astype(np.int32)
    sample_pairs = int(row_pairs[rows].sum())
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.mixed_attention(qh, k, v, b.block_table, b.query_start_loc, b.ctx_lens, b.scale, rows=rows)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
    us = float(np.mean(times)) * 1e6 * (total_pairs / sample_pairs)
    sample = f"{n_rows} of {b.T} query rows ({sample_pairs} of {total_pairs} visible pairs/head) per step, extrapolated by pair count"
    line = {
        "impl": "reference", "metric": METRIC, "value": us, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": us / 1e3, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload} {b.name}", "R": b.R, "T": b.T, "shape": [b.num_q_heads, b.num_kv_heads, b.head_dim]},
        "cpu_baseline": {"value": us, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": us, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2606_05933_b200 import binding, workloads as wl, accounting as acc
    from paper_2606_05933_b200.features import features, scene

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    devname = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(devname))

    b = get_batch(args.workload)
    t = wl.make_tensors(b, devname)
    h = binding.handle_for(b, t)
    to_dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(devname)
    bt, qsl, ctx = to_dev(b.block_table), to_dev(b.query_start_loc), to_dev(b.ctx_lens)
    out = torch.empty_like(t.q)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=devname)       # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step():
        binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx)
        n = h.last_launch_count()
        binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=out)
        return n + h.last_launch_count()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    launches_per_step = 0
    for _ in range(max(args.warmup, 3)):
        flush.fill_(1)
        launches_per_step = step()
    barrier()

    # ---- timed region: exactly K steps, CUDA events per step on the launching stream; L2 flushed
    # (512 MB write) between steps, outside the event windows ----
    sampler = ClockSampler(visible_device_index())
    sampler.start()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    wall0 = time.perf_counter()
    for e0, e1 in evs:
        flush.fill_(1)
        e0.record(stream)
        step()
        e1.record(stream)
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    per_step_ms = np.array([e0.elapsed_time(e1) for e0, e1 in evs], dtype=np.float64)
    total_ms = max_over_ranks(float(per_step_ms.sum()), world, devname)
    ms_per_step, value_us = replica_metric(total_ms, args.steps, world)

    # ---- dominant kernel: main attention launch, timed by events inside the library on the same stream ----
    h.set_kernel_timing(True)
    kt = []
    for _ in range(args.steps):
        flush.fill_(1)
        step()
        kt.append(h.last_kernel_time_us())
    h.set_kernel_timing(False)
    kern_us = float(np.mean(kt))
    peaks = acc.load_peaks()
    w = acc.work(b)
    roof = acc.roofline_us(b, peaks)
    if roof["bound"] == "hbm":
        achieved = w["bytes"] / (kern_us * 1e-6) / 1e9
        peak, unit = peaks["hbm_gbs"], "GB/s"
    else:
        achieved = w["flops"] / (kern_us * 1e-6) / 1e12
        peak, unit = peaks["bf16_tflops"], "TFLOP/s"
    traffic = None
    tp = ROOT / "profiles" / "traffic.json"
    if tp.exists():
        traffic = json.loads(tp.read_text()).get(args.workload)
    roofline = {"bound": roof["bound"], "achieved": achieved, "peak": peak, "unit": unit, "frac": achieved / peak,
                "traffic": traffic, "kernel": "main attention launch (a3+a4)", "kernel_us": kern_us,
                "peak_source": peaks["source"], "algorithmic_bytes": w["bytes"], "algorithmic_flops": w["flops"],
                "batch_roofline_us": roof["roofline_us"], "batch_frac_of_roofline": roof["roofline_us"] / (ms_per_step * 1e3)}

    # ---- e2e: the same step through the C ABI's host-buffer entry point (pinned host tensors) ----
    hq, hk, hv = (x.cpu().pin_memory() for x in (t.q, t.k_new, t.v_new))
    hbt, hqsl, hctx = (torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in (b.block_table, b.query_start_loc, b.ctx_lens))
    hout = torch.empty_like(hq).pin_memory()
    for _ in range(3):
        h.iteration_host(hq, hk, hv, hbt, hqsl, hctx, b.scale, hout)
    barrier()
    e2e_steps = max(min(args.steps, 50), 1)
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        flush.fill_(1)
        torch.cuda.synchronize()
        h.iteration_host(hq, hk, hv, hbt, hqsl, hctx, b.scale, hout)
    torch.cuda.synchronize()
    # subtract nothing: flush time is inside this wall clock, so time it separately and remove it
    t1 = time.perf_counter()
    for _ in range(e2e_steps):
        flush.fill_(1)
        torch.cuda.synchronize()
    t2 = time.perf_counter()
    e2e_s = ((t1 - t0) - (t2 - t1)) / e2e_steps
    e2e_s = max_over_ranks(e2e_s, world, devname)
    h2d = sum(x.numel() * x.element_size() for x in (hq, hk, hv, hbt, hqsl, hctx))
    d2h = hout.numel() * hout.element_size()
    assert torch.equal(hout, out.cpu()), "e2e output differs from the device-resident path"
    e2e = {"value": e2e_s * 1e6 / world, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)}

    # ---- cpu_baseline: the oracle on the host cores, rank 0 at N=1 only, bounded sample ----
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        from paper_2606_05933_b200.features import causal_pairs
        if b.num_pages > 200000:            # e.g. C4's 40 GB pool: gather only the used pages
            btab, (k, v) = wl.compact_pool(b, t.k_cache, t.v_cache)
        else:
            btab, k, v = b.block_table, wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
        total_pairs = causal_pairs(b.reqs)
        rng = np.random.default_rng(0)
        cores = oracle.num_threads()
        # ~15 s of CPU work: pick rows until the pair budget (rate probed on a few rows) is met
        probe = np.sort(rng.choice(b.T, size=min(b.T, 2 * cores), replace=False)).astype(np.int32)
        t0 = time.perf_counter()
        _, _, pp = oracle.mixed_attention(wl.to_u16(t.q), k, v, btab, b.query_start_loc, b.ctx_lens, b.scale, rows=probe)
        rate = pp / max(time.perf_counter() - t0, 1e-6)
        row_pairs = np.empty(b.T, dtype=np.int64)
        for r, (c, u) in enumerate(b.reqs):
            s = int(b.query_start_loc[r])
            row_pairs[s:s + c] = u + 1 + np.arange(c)
        order = rng.permutation(b.T)
        want = min(total_pairs, int(rate * 15.0))
        n_rows = int(min(b.T, np.searchsorted(np.cumsum(row_pairs[order]), want) + 1))
        rows = np.sort(order[:n_rows]).astype(np.int32)
        sp = int(row_pairs[rows].sum())
        t0 = time.perf_counter()
        ref, _, _ = oracle.mixed_attention(wl.to_u16(t.q), k, v, btab, b.query_start_loc, b.ctx_lens, b.scale, rows=rows)
        dt = time.perf_counter() - t0
        err = np.abs(out[torch.from_numpy(rows).long().to(devname)].to(torch.float64).cpu().numpy() - ref)
        cpu_baseline = {"value": dt * 1e6 * total_pairs / sp, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"{n_rows} of {b.T} query rows ({sp} of {total_pairs} visible pairs/head), one pass, extrapolated by pair count",
                        "parity_on_sample": {"max_abs": float(err.max()), "mean_abs": float(err.mean())}}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value_us, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16", "data": "synthetic",
            "config": {"workload": f"{args.workload} {b.name}", "R": b.R, "T": b.T,
                       "shape": {"Hq": b.num_q_heads, "Hkv": b.num_kv_heads, "D": b.head_dim, "page": b.page_size},
                       "scene": scene(b.reqs), "features": features(b.reqs), "step": "kv_append + mixed_attention",
                       "l2": "flushed between steps (512 MB write outside the event window)",
                       "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                       "median_us": float(np.median(per_step_ms) * 1e3), "p10_us": float(np.percentile(per_step_ms, 10) * 1e3),
                       "p90_us": float(np.percentile(per_step_ms, 90) * 1e3), "wall_s": wall},
            "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e,
            "gpu_launches": int(launches_per_step * args.steps), "launches_per_step": int(launches_per_step),
            "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="C2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
