"""Batch descriptors the paper defines on B = {(c_i, u_i)}: the decode / prefill sets (PAPER.md:111
Eq. 2), the scene label (Eq. 3) and the 7 predictor features (Table 1).
Host-side integer bookkeeping only; emitted beside every timing so the measured latency surface is
directly what a SlidingChunker-style predictor (Eq. 5) would be fitted on."""
from __future__ import annotations

from typing import Dict, Iterable, Tuple


def split_sets(reqs: Iterable[Tuple[int, int]]):
    """D = {i : c_i <= 1}, P = {i : c_i > 1}  (Eq. 2)."""
    reqs = list(reqs)
    D = [i for i, (c, _) in enumerate(reqs) if c <= 1]
    P = [i for i, (c, _) in enumerate(reqs) if c > 1]
    return D, P


def scene(reqs: Iterable[Tuple[int, int]]) -> str:
    """pure decode if |P| = 0, pure prefill if |D| = 0, else mixed  (Eq. 3)."""
    D, P = split_sets(reqs)
    if not P:
        return "pure_decode"
    if not D:
        return "pure_prefill"
    return "mixed"


def features(reqs: Iterable[Tuple[int, int]]) -> Dict[str, int]:
    """x1..x7 of Table 1.  x7 = 0 when P is empty (reading 13)."""
    reqs = [(int(c), int(u)) for c, u in reqs]
    D, P = split_sets(reqs)
    return {
        "x1": sum(reqs[i][0] * (reqs[i][1] + reqs[i][0]) for i in P),
        "x2": sum(reqs[i][0] ** 2 for i in P),
        "x3": sum(u for _, u in reqs),
        "x4": len(D),
        "x5": sum(reqs[i][1] for i in D),
        "x6": sum(reqs[i][0] for i in P),
        "x7": max((reqs[i][0] for i in P), default=0),
    }


def causal_pairs(reqs: Iterable[Tuple[int, int]]) -> int:
    """Number of (query row, visible key) pairs per query head: sum_i c_i*u_i + c_i(c_i+1)/2."""
    return sum(c * u + c * (c + 1) // 2 for c, u in reqs)
