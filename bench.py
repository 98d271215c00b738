#!/usr/bin/env python
"""bench.py — one JSON line for the driver.

A "step" = one pass of the whole hot path over one synthetic batch: kv_append of the batch's new tokens
(a1) + mixed_attention (a2 work list, a3 prefill tiles, a4 decode splits, a5 merge), through the C ABI.

Headline workload at N=1: BASELINE.json configs[4] "C5" — the largest MIXED single-GPU configuration
(Llama-3-70B-shaped layer, 2 x 1024 chunk tokens + 192 decodes, with append), which runs every row of
SURVEY.md §8(a).  The same line carries `per_config`: C2 (configs[1]), C4 (configs[3], decode-heavy, the
>= 70 % HBM target), C4/fp8 (the same batch over an FP8 E4M3 KV cache: half the algorithmic KV bytes), PP-b / PP-f
(chunk-heavy scene edges, the >= 50 % tensor target) and PD-32 (small pure-decode call), each timed with the same
protocol and with its own roofline object, and ends with `targets`: one compact record per workload (step us, batch
roofline fraction, the dominant kernel's fraction of its peak, and for HBM-bound ones the same against the stricter
read-only streaming peak measured live) - last on purpose, so a log tail keeps it.  Other workloads:
--workload NAME; --per-config a,b,c or "none".

Metric: BASELINE.json's "mixed prefill+decode attention us/iter and % of HBM/tensor roofline" -> value =
microseconds per iteration (lower is better), roofline fraction in the `roofline` object.  N>1:
independent replicas, one per GPU (replicas only, no collective on the data path);
value = max-over-ranks time / (N*K) iterations.  Without torchrun, `--gpus N` re-executes itself under
torch.distributed.run with N ranks.

--impl reference times the fp64 CPU oracle (oracle/) as it stands on the host cores, on a bounded row
sample per step, extrapolated to the whole batch by visible-pair count.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "mixed prefill+decode attention us/iter and % of HBM/tensor roofline"
UNIT = "us/iter"
HEADLINE = "C5"
PER_CONFIG = "C2,C4,C4/fp8,PP-b,PP-f,PD-32"


def get_batch(name: str):
    from paper_2606_05933_b200 import workloads as wl
    if name.endswith("/fp8"):                       # the same batch over an FP8 E4M3 KV cache (SS_FLAG_KV_FP8)
        b = get_batch(name[:-4])
        return wl.Batch(**{**b.__dict__, "name": b.name + "/fp8", "meta": {**b.meta, "kv_fp8": True}})
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
    if name.startswith("MX-"):
        return wl.config_model_mixed(name[3:])
    if name.startswith("C3:"):
        C, n, nd = (int(x) for x in name[3:].split(","))
        return wl.config_c3(C, n, nd)
    raise SystemExit(f"unknown workload {name}")


def config_object(name: str, b, world: int = 1) -> dict:
    """The `config` both arms print (identical objects for the same workload)."""
    from paper_2606_05933_b200.features import features, scene
    return {"workload": f"{name} {b.name}", "R": b.R, "T": b.T,
            "shape": {"Hq": b.num_q_heads, "Hkv": b.num_kv_heads, "D": b.head_dim, "page": b.page_size},
            "scene": scene(b.reqs), "features": features(b.reqs), "step": "kv_append + mixed_attention",
            "l2": "flushed between steps (512 MB write outside the event window)",
            "parallelism": f"replicas x{world}" if world > 1 else "single GPU"}


class ClockSampler(threading.Thread):
    """Samples SM clock and clock-event reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.002):
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


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn_ranks(args, argv) -> int:
    """`python bench.py --gpus N` without torchrun: re-execute under torch.distributed.run, one rank per GPU."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(Path(__file__).resolve()), *argv]
    return subprocess.call(cmd)


def run_dry(args):
    """Replica plumbing without kernels (CPU test of the N > 1 entry): process group, max-over-ranks, rank-0 line."""
    import torch
    import torch.distributed as dist
    world, rank = int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl" if torch.cuda.is_available() else "gloo")
    total = max_over_ranks(10.0 * (rank + 1) * args.steps, world)           # rank r "measures" 10(r+1) ms per step
    ms_per_step, value_us = replica_metric(total, args.steps, world)
    if world > 1:
        dist.barrier()
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": value_us, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": False,
                          "scaling": "weak", "dry_run": True}), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------
def oracle_sample(b, budget_s: float, cores: int, qh, k, v, btab, seed: int = 0):
    """Rows for a bounded oracle run: the whole batch if it fits the budget at the probed rate, else a random row
    sample sized by visible-pair count.  Returns (rows or None, sample_pairs, total_pairs, per-row pair counts)."""
    import oracle
    from paper_2606_05933_b200.features import causal_pairs
    total_pairs = causal_pairs(b.reqs)
    rng = np.random.default_rng(seed)
    probe = np.sort(rng.choice(b.T, size=min(b.T, 2 * cores), replace=False)).astype(np.int32)
    t0 = time.perf_counter()
    _, _, pp = oracle.mixed_attention(qh, k, v, btab, b.query_start_loc, b.ctx_lens, b.scale, rows=probe)
    rate = pp / max(time.perf_counter() - t0, 1e-6)
    row_pairs = np.empty(b.T, dtype=np.int64)
    for r, (c, u) in enumerate(b.reqs):
        s = int(b.query_start_loc[r])
        row_pairs[s:s + c] = u + 1 + np.arange(c)
    if total_pairs <= rate * budget_s:
        return None, total_pairs, total_pairs
    order = rng.permutation(b.T)
    n_rows = int(min(b.T, np.searchsorted(np.cumsum(row_pairs[order]), int(rate * budget_s)) + 1))
    rows = np.sort(order[:n_rows]).astype(np.int32)
    return rows, int(row_pairs[rows].sum()), total_pairs


def run_reference(args):
    """Oracle arm: rank 0 only; each step = the oracle on a bounded row sample of the workload."""
    if not reference_rank_runs(int(os.environ.get("RANK", "0"))):
        return
    import oracle
    from paper_2606_05933_b200 import workloads as wl
    b = get_batch(args.workload)
    t = wl.make_tensors(b, "cpu")
    k, v = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    qh, kn, vn = wl.to_u16(t.q), wl.to_u16(t.k_new), wl.to_u16(t.v_new)
    oracle.kv_append(k, v, kn, vn, b.block_table, b.query_start_loc, b.ctx_lens)
    cores = oracle.num_threads()
    budget_s = min(150.0 / max(args.steps + args.warmup, 1), 30.0)       # whole run ~150 s of CPU work
    rows, sample_pairs, total_pairs = oracle_sample(b, budget_s, cores, qh, k, v, b.block_table)
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.mixed_attention(qh, k, v, b.block_table, b.query_start_loc, b.ctx_lens, b.scale, rows=rows)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
    us = float(np.mean(times)) * 1e6 * (total_pairs / sample_pairs)
    n_rows = b.T if rows is None else len(rows)
    sample = (f"{n_rows} of {b.T} query rows ({sample_pairs} of {total_pairs} visible pairs/head) per step"
              + ("" if rows is None else ", extrapolated by pair count"))
    line = {
        "impl": "reference", "metric": METRIC, "value": us, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": us / 1e3, "higher_is_better": False, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_object(args.workload, b, args.gpus),
        "cpu_baseline": {"value": us, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": us, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
def load_traffic(name: str):
    """DRAM bytes (read + write) of the main launch from the committed `ncu --set full` capture of this workload
    (profiles/traffic.json: bytes + the commit and command it was captured with), or None."""
    tp = ROOT / "profiles" / "traffic.json"
    if not tp.exists():
        return None, None
    ent = json.loads(tp.read_text()).get(name)
    if ent is None:
        return None, None
    if isinstance(ent, dict):
        return ent.get("bytes"), {k: ent[k] for k in ("commit", "command", "file") if k in ent}
    return ent, None


class Bench:
    """One workload resident on the device, ready to be stepped."""

    def __init__(self, name: str, devname: str):
        import torch
        from paper_2606_05933_b200 import binding, workloads as wl
        self.name, self.devname = name, devname
        self.b = get_batch(name)
        if self.b.meta.get("kv_fp8"):
            self.t = wl.make_tensors(self.b, devname, caches=False)
            kc, vc, ks, vs = wl.make_fp8_caches(self.b, devname)
            self.h = binding.handle_for(self.b, self.t, fp8_caches=(kc, vc), kv_scales=(ks, vs))
        else:
            self.t = wl.make_tensors(self.b, devname)
            self.h = binding.handle_for(self.b, self.t)
        to_dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(devname)
        self.bt, self.qsl, self.ctx = to_dev(self.b.block_table), to_dev(self.b.query_start_loc), to_dev(self.b.ctx_lens)
        self.out = torch.empty_like(self.t.q)

    def step(self) -> int:
        from paper_2606_05933_b200 import binding
        b, t, h = self.b, self.t, self.h
        binding.kv_append(h, t.k_new, t.v_new, self.bt, self.qsl, self.ctx)
        n = h.last_launch_count()
        binding.mixed_attention(h, t.q, self.bt, self.qsl, self.ctx, b.scale, out=self.out)
        return n + h.last_launch_count()

    def close(self):
        import torch
        self.h.close()
        del self.t, self.out, self.h
        torch.cuda.empty_cache()

    def time_steps(self, steps: int, warmup: int, flush, barrier=None):
        """(per-step ms array, launches per step, wall seconds): CUDA events per step on the launching stream, L2
        flushed between steps outside the event window."""
        import torch
        barrier = barrier or torch.cuda.synchronize
        stream = torch.cuda.current_stream()
        launches = 0
        for _ in range(max(warmup, 3)):
            flush.fill_(1)
            launches = self.step()
        barrier()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        barrier()
        wall0 = time.perf_counter()
        for e0, e1 in evs:
            flush.fill_(1)
            e0.record(stream)
            self.step()
            e1.record(stream)
        barrier()
        wall = time.perf_counter() - wall0
        return np.array([e0.elapsed_time(e1) for e0, e1 in evs], dtype=np.float64), launches, wall

    def time_graph(self, steps: int, flush) -> float:
        """Median us per step when the step (append + attention) is replayed from a CUDA graph: same protocol."""
        import torch
        from paper_2606_05933_b200 import binding
        b, t, h = self.b, self.t, self.h
        g, s = torch.cuda.CUDAGraph(), torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            binding.kv_append(h, t.k_new, t.v_new, self.bt, self.qsl, self.ctx, stream=s)
            binding.mixed_attention(h, t.q, self.bt, self.qsl, self.ctx, b.scale, out=self.out, stream=s)
            s.synchronize()
            with torch.cuda.graph(g, stream=s):
                binding.kv_append(h, t.k_new, t.v_new, self.bt, self.qsl, self.ctx, stream=s)
                binding.mixed_attention(h, t.q, self.bt, self.qsl, self.ctx, b.scale, out=self.out, stream=s)
        torch.cuda.current_stream().wait_stream(s)
        stream = torch.cuda.current_stream()
        us = []
        for i in range(steps + 3):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            g.replay()
            e1.record(stream)
            torch.cuda.synchronize()
            if i >= 3:
                us.append(e0.elapsed_time(e1) * 1e3)
        del g
        return float(np.median(us))

    def roofline(self, steps: int, flush, step_ms: float, read_peak_gbs: float = None) -> dict:
        """Dominant kernel = the main attention launch (a3+a4+a5); algorithmic bytes / flops of the batch (DESIGN.md
        section 8) over its duration vs the measured peak.  Its duration: the step of the timed region is append +
        main launch with the append hidden under the main launch's prologue (PDL), so the step time bounds the
        kernel time from above.  A second pass brackets the main launch alone with CUDA events inside the library;
        those event records sit between the two launches and undo the overlap, so that figure can come out ABOVE the
        step.  kernel_us is the smaller of the two - never more than the step it is part of -
        and both are printed."""
        from paper_2606_05933_b200 import accounting as acc
        h, b = self.h, self.b
        h.set_kernel_timing(True)
        kt = []
        for _ in range(steps):
            flush.fill_(1)
            self.step()
            kt.append(h.last_kernel_time_us())
        h.set_kernel_timing(False)
        events_us, step_us = float(np.mean(kt)), step_ms * 1e3
        kern_us = min(events_us, step_us)
        peaks, w = acc.load_peaks(), acc.work(b)
        roof = acc.roofline_us(b, peaks)
        if roof["bound"] == "hbm":
            achieved, peak, unit = w["bytes"] / (kern_us * 1e-6) / 1e9, peaks["hbm_gbs"], "GB/s"
        else:
            achieved, peak, unit = w["flops"] / (kern_us * 1e-6) / 1e12, peaks["bf16_tflops"], "TFLOP/s"
        traffic, src = load_traffic(self.name)
        out = {"bound": roof["bound"], "achieved": achieved, "peak": peak, "unit": unit, "frac": achieved / peak,
               "traffic": traffic, "kernel": "main attention launch (a3+a4+a5)", "kernel_us": kern_us,
               "kernel_us_source": "library events around the main launch" if events_us <= step_us else
                                   "step time of the timed region (upper bound: the append overlaps the main launch by PDL)",
               "kernel_us_events_pass": events_us, "step_us": step_us, "peak_source": peaks["source"],
               "algorithmic_bytes": w["bytes"], "algorithmic_flops": w["flops"],
               "batch_roofline_us": roof["roofline_us"], "batch_frac_of_roofline": roof["roofline_us"] / (step_ms * 1e3)}
        if roof["bound"] == "tensor":
            out["frac_of_sustained_peak"] = achieved / peaks["bf16_tflops_sustained"]
        elif read_peak_gbs:
            # the decode path only reads: against the stricter of the copy peak and the read-only streaming peak
            # measured live in this run (ss_debug_stream_read), no HBM fraction can exceed 1
            out["hbm_read_peak_gbs"] = read_peak_gbs
            out["frac_vs_read_peak"] = achieved / max(peak, read_peak_gbs)
        if src and "commit" in src:
            out["traffic_commit"] = src["commit"]          # command and file: profiles/traffic.json
        return out

    def read_peak(self, flush, passes: int = 12) -> float:
        """GB/s of a read-only streaming pass over 16 GiB (ss_debug_stream_read), L2 flushed, median of `passes`."""
        import torch
        buf = torch.empty(16 << 30, dtype=torch.uint8, device=self.devname)
        buf.fill_(3)
        stream = torch.cuda.current_stream()
        us = []
        for i in range(passes + 3):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            self.h.stream_read(buf)
            e1.record(stream)
            torch.cuda.synchronize()
            if i >= 3:
                us.append(e0.elapsed_time(e1) * 1e3)
        del buf
        return float((16 << 30) / (np.median(us) * 1e-6) / 1e9)

    def time_paced(self, steps: int, flush, pause_s: float = 0.010) -> float:
        """Mean us per step with a 10 ms host pause between steps (a serving loop's other layers would sit there): the
        SM clock recovers between steps, unlike in the back-to-back timed region."""
        import torch
        stream = torch.cuda.current_stream()
        us = []
        for _ in range(steps):
            flush.fill_(1)
            torch.cuda.synchronize()
            time.sleep(pause_s)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            self.step()
            e1.record(stream)
            torch.cuda.synchronize()
            us.append(e0.elapsed_time(e1) * 1e3)
        return float(np.mean(us))

    def time_rope_append(self, flush, iters: int = 10) -> dict:
        """ss_qkv_rope_append (NEXT-4, the step before the path) on this batch against its own HBM roofline: reads the
        fused projection [T][(Hq + 2 Hkv) D] bf16 once, writes q_out and the K / V slots once."""
        import torch
        from paper_2606_05933_b200 import accounting as acc
        b, h = self.b, self.h
        width = (b.num_q_heads + 2 * b.num_kv_heads) * b.head_dim
        gen = torch.Generator(device=self.devname)
        gen.manual_seed(12345)
        qkv = torch.randn(b.T, width, generator=gen, device=self.devname, dtype=torch.float32).to(torch.bfloat16)
        q_out = torch.empty(b.T, b.num_q_heads, b.head_dim, dtype=torch.bfloat16, device=self.devname)
        stream = torch.cuda.current_stream()
        us = []
        for i in range(iters + 3):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            h.qkv_rope_append(qkv, self.bt, self.qsl, self.ctx, 500000.0, q_out=q_out)
            e1.record(stream)
            torch.cuda.synchronize()
            if i >= 3:
                us.append(e0.elapsed_time(e1) * 1e3)
        esz = 1 if b.meta.get("kv_fp8") else 2
        nbytes = b.T * width * 2 + b.T * b.num_q_heads * b.head_dim * 2 + 2 * b.T * b.num_kv_heads * b.head_dim * esz
        med = float(np.median(us))
        return {"us": med, "algorithmic_bytes": int(nbytes), "achieved_gbs": nbytes / (med * 1e-6) / 1e9,
                "frac_of_hbm_peak": nbytes / (med * 1e-6) / 1e9 / acc.load_peaks()["hbm_gbs"],
                "timing": "CUDA events around the one launch, L2 flushed; includes ~10 us of launch-to-exit overhead"}


def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2606_05933_b200 import workloads as wl

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    devname = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(devname))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    flush = torch.empty(512 << 20, dtype=torch.uint8, device=devname)       # > 126 MB L2
    bench = Bench(args.workload, devname)
    b, t, h = bench.b, bench.t, bench.h

    # ---- timed region: exactly K steps ----
    sampler = ClockSampler(visible_device_index())
    sampler.start()
    per_step_ms, launches_per_step, wall = bench.time_steps(args.steps, args.warmup, flush, barrier)
    clocks = sampler.stop()
    total_ms = max_over_ranks(float(per_step_ms.sum()), world, devname)
    ms_per_step, value_us = replica_metric(total_ms, args.steps, world)
    read_peak = bench.read_peak(flush)
    roofline = bench.roofline(min(args.steps, 100), flush, float(per_step_ms.mean()), read_peak)
    paced_us = bench.time_paced(min(args.steps, 20), flush)

    # ---- a1 alone: kv_append against its own roofline, 4*T*Hkv*D*2 bytes ----
    from paper_2606_05933_b200 import accounting as acc, binding
    stream = torch.cuda.current_stream()
    ka = []
    for i in range(13):
        flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        binding.kv_append(h, t.k_new, t.v_new, bench.bt, bench.qsl, bench.ctx)
        e1.record(stream)
        torch.cuda.synchronize()
        if i >= 3:
            ka.append(e0.elapsed_time(e1) * 1e3)
    append_bytes = 4 * b.T * b.num_kv_heads * b.head_dim * 2
    kv_append_obj = {"us": float(np.median(ka)), "algorithmic_bytes": append_bytes,
                     "achieved_gbs": append_bytes / (float(np.median(ka)) * 1e-6) / 1e9,
                     "frac_of_hbm_peak": append_bytes / (float(np.median(ka)) * 1e-6) / 1e9 / acc.load_peaks()["hbm_gbs"]}

    rope_append_obj = bench.time_rope_append(flush)
    # kv_append_obj was timed before the fused append overwrote the same slots; the caches now hold the rotated tokens,
    # so restore them for the parity sample below
    binding.kv_append(h, t.k_new, t.v_new, bench.bt, bench.qsl, bench.ctx)

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
    # the L2 flush sits inside this wall clock: time it separately and remove it
    t1 = time.perf_counter()
    for _ in range(e2e_steps):
        flush.fill_(1)
        torch.cuda.synchronize()
    t2 = time.perf_counter()
    e2e_s = ((t1 - t0) - (t2 - t1)) / e2e_steps
    e2e_s = max_over_ranks(e2e_s, world, devname)
    h2d = sum(x.numel() * x.element_size() for x in (hq, hk, hv, hbt, hqsl, hctx))
    d2h = hout.numel() * hout.element_size()
    assert torch.equal(hout, bench.out.cpu()), "e2e output differs from the device-resident path"
    e2e = {"value": e2e_s * 1e6 / world, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)}

    # ---- cpu_baseline: the oracle on the host cores, rank 0 at N=1 only, bounded sample (~15 s) ----
    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        if b.num_pages > 200000:            # e.g. C4's 40 GB pool: gather only the used pages
            btab, (k, v) = wl.compact_pool(b, t.k_cache, t.v_cache)
        else:
            btab, k, v = b.block_table, wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
        cores = oracle.num_threads()
        qh = wl.to_u16(t.q)
        rows, sp, total_pairs = oracle_sample(b, 15.0, cores, qh, k, v, btab)
        t0 = time.perf_counter()
        ref, _, _ = oracle.mixed_attention(qh, k, v, btab, b.query_start_loc, b.ctx_lens, b.scale, rows=rows)
        dt = time.perf_counter() - t0
        got = bench.out if rows is None else bench.out[torch.from_numpy(rows).long().to(devname)]
        err = np.abs(got.to(torch.float64).cpu().numpy() - ref)
        n_rows = b.T if rows is None else len(rows)
        cpu_baseline = {"value": dt * 1e6 * total_pairs / sp, "unit": UNIT, "cores": cores, "kind": "oracle",
                        "sample": f"{n_rows} of {b.T} query rows ({sp} of {total_pairs} visible pairs/head), one pass"
                                  + ("" if rows is None else ", extrapolated by pair count"),
                        "parity_on_sample": {"max_abs": float(err.max()), "mean_abs": float(err.mean())}}
        del k, v, ref
    headline_cfg = config_object(args.workload, b, world)
    bench.close()

    # ---- per_config: the configs the north_star targets are quoted on, same protocol, rank 0 at N=1 ----
    per_config = []
    names = [] if args.per_config.lower() == "none" else [n for n in args.per_config.split(",") if n and n != args.workload]
    if world == 1:
        pc_steps = max(min(args.steps, 50), 5)
        for name in names:
            pb = Bench(name, devname)
            ms, nl, _ = pb.time_steps(pc_steps, args.warmup, flush)
            ent = {"workload": f"{name} {pb.b.name}", "R": pb.b.R, "T": pb.b.T,
                   "shape": {"Hq": pb.b.num_q_heads, "Hkv": pb.b.num_kv_heads, "D": pb.b.head_dim},
                   "steps": pc_steps, "us_per_iter": float(ms.mean() * 1e3), "median_us": float(np.median(ms) * 1e3),
                   "p10_us": float(np.percentile(ms, 10) * 1e3), "p90_us": float(np.percentile(ms, 90) * 1e3),
                   "launches_per_step": int(nl), "roofline": pb.roofline(pc_steps, flush, float(ms.mean()), read_peak)}
            if name in ("PD-32", "C2"):
                ent["graph_replay_median_us"] = pb.time_graph(min(pc_steps, 20), flush)   # the same step replayed from a CUDA graph
            per_config.append(ent)
            pb.close()

    if rank == 0:
        timing = {"median_us": float(np.median(per_step_ms) * 1e3), "p10_us": float(np.percentile(per_step_ms, 10) * 1e3),
                  "p90_us": float(np.percentile(per_step_ms, 90) * 1e3), "wall_s": wall,
                  "headline": "value = mean of the back-to-back timed region (L2 flushed between steps)",
                  "paced_10ms_us": paced_us}

        def target(name, us, r):
            o = {"w": name, "us": round(us, 1), "bound": r["bound"], "frac": round(r["batch_frac_of_roofline"], 3),
                 "kfrac": round(r["frac"], 3)}
            if "frac_vs_read_peak" in r:
                o["kfrac_rd"] = round(r["frac_vs_read_peak"], 3)
            return o
        # compact and LAST, so that a log tail keeps the decode-heavy target (C4) and the prefill edges: per workload the
        # step time, the batch roofline fraction (roofline us / step us), the dominant kernel's fraction of its peak
        # and, for HBM-bound ones, the same against max(copy peak, read-only streaming peak)
        targets = [target(args.workload, value_us, roofline)] + \
                  [target(e["workload"].split()[0], e["us_per_iter"], e["roofline"]) for e in per_config]
        line = {
            "metric": METRIC, "value": value_us, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16", "data": "synthetic", "config": headline_cfg, "timing": timing,
            "roofline": roofline, "cpu_baseline": cpu_baseline, "e2e": e2e, "kv_append": kv_append_obj,
            "qkv_rope_append": rope_append_obj,
            "gpu_launches": int(launches_per_step * args.steps), "launches_per_step": int(launches_per_step),
            "clocks": clocks, "per_config": per_config, "hbm_read_peak_gbs": read_peak, "targets": targets,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default=HEADLINE)
    ap.add_argument("--per-config", default=PER_CONFIG, help='comma-separated extra workloads timed into "per_config", or "none"')
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--dry-run", action="store_true", help="replica plumbing only (no kernels): CPU test of the N > 1 entry")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(spawn_ranks(args, sys.argv[1:]))
    if args.dry_run:
        run_dry(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
