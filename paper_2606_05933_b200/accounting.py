"""Algorithmic work of one mixed_attention iteration.

bytes = every visible K and V row once (2 bytes per element, 1 for an FP8 cache: batch.meta["kv_fp8"]) + Q in +
O out;  flops = 4*D*Hq*pairs.  Block tables, the
work list and split partials are excluded (they are the implementation's, not the method's)."""
from __future__ import annotations

import json
import os
from pathlib import Path
from typing import Dict

from .features import causal_pairs, split_sets

FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks() -> Dict[str, float]:
    """MEASURED_PEAKS.json at the repo root (driver-written), else B200_PROFILING.md's fallback."""
    p = Path(os.environ.get("SS_MEASURED_PEAKS", Path(__file__).resolve().parent.parent / "MEASURED_PEAKS.json"))
    if p.exists():
        d = json.loads(p.read_text())
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                "source": "measured"}
    return dict(FALLBACK_PEAKS, source="fallback")


def work(batch) -> Dict[str, float]:
    Hq, Hkv, D = batch.num_q_heads, batch.num_kv_heads, batch.head_dim
    reqs = [(c, u) for c, u in batch.reqs if c > 0]
    kv_tokens = sum(c + u for c, u in reqs)
    T = sum(c for c, _ in reqs)
    esz = 1 if batch.meta.get("kv_fp8") else 2       # bytes per cached element (FP8 E4M3 cache: 1)
    kv_bytes = kv_tokens * 2 * Hkv * D * esz
    qo_bytes = 2 * T * Hq * D * 2
    pairs = causal_pairs(reqs)
    Dset, Pset = split_sets(reqs)
    pairs_P = causal_pairs([reqs[i] for i in Pset])
    kv_bytes_D = sum(reqs[i][0] + reqs[i][1] for i in Dset) * 2 * Hkv * D * esz
    return {
        "kv_bytes": kv_bytes, "qo_bytes": qo_bytes, "bytes": kv_bytes + qo_bytes,
        "flops": 4 * D * Hq * pairs, "pairs": pairs,
        "prefill_flops": 4 * D * Hq * pairs_P, "decode_kv_bytes": kv_bytes_D,
        "append_bytes": 2 * T * Hkv * D * (2 + esz) if batch.with_append else 0,
    }


def roofline_us(batch, peaks=None, sustained: bool = False) -> Dict[str, float]:
    peaks = peaks or load_peaks()
    w = work(batch)
    tf = peaks["bf16_tflops_sustained" if sustained else "bf16_tflops"]
    t_hbm = w["bytes"] / (peaks["hbm_gbs"] * 1e9) * 1e6
    t_tc = w["flops"] / (tf * 1e12) * 1e6
    return {"t_hbm_us": t_hbm, "t_tc_us": t_tc, "roofline_us": max(t_hbm, t_tc),
            "bound": "hbm" if t_hbm >= t_tc else "tensor"}
