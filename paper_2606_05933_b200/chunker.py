"""SlidingChunker (§3.4, Algorithm 1 :226-268) driven by the batch latency predictor fitted on OUR
measured latency surface.  Host-side scheduling logic, tens of items: plain Python.

Pieces, in the paper's names:
  BatchForwarder F  forms the batch a budget b would run and predicts its time:
      Forward(D, P, b) -> (T_hat, A): every decode request gets its 1 token (b >= |D|), the remaining b - |D| tokens go
          to the prefill requests in the order of the SORTED set P (Eq. 13 orders it; here the caller
          passes it sorted), each taking min(remaining prompt, what is left);  A = the per-request allocation.
      Pred(b, D, P)     = the T_hat of Forward.
      TimeToBudget(D, P, T) = the largest b in [|D|, B] with Pred(b) <= T, by binary search ("approximated
          using binary search"); |D| if even the decode-only batch is too slow.
  T_cur  = min over protected decodes of their TBT slack s_i(t)                     (Eq. 14, "D_cafe" read
  T_next = min over protected decodes of s_i(t) - T_cur + L_i^tbt                     as D_safe: DESIGN.md reading 14)
  B*     = argmin_b T_hat(b) + T_hat(B_sigma - b),  B_sigma = B_cur + B_next         (Eq. 16)
           by the discrete ternary search of Algorithm 1 (stop at r - l <= 30, then compare {l0, r0, mid}).

Readings of the garbled listing: line 9-15 = "if T1 <= T2 then r <- m2 - 1 else l <- m1 + 1"; ties go to the larger
budget (line 23).  The search range is the b for which BOTH windows get a budget an iteration can run,
max(|D|, B_sigma - B) <= b <= min(B, B_sigma - |D|): "B_sigma - b [is] the approximate budget for the next window"
(PAPER.md:210), so the two windows always carry B_sigma tokens between them.  (Round 2 searched [|D|, B] and clamped
B_sigma - b instead; with plenty of slack, B_sigma = 2B, the clamped objective is smallest at b = |D| - it rewards
dropping the prefill tokens rather than balancing them, and a calm system starved its prefill.  DESIGN.md reading 17.)
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Callable, List, Sequence, Tuple

from .features import features, scene

Request = Tuple[int, int]          # (tokens this round c_i, cached tokens u_i)  -- PAPER.md:107


@dataclass
class PrefillState:
    remaining: int                 # prompt tokens still to prefill, r_i(t)
    cached: int                    # tokens already in the KV cache, u_i


class BatchForwarder:
    """F of Algorithm 1.  `predict(reqs) -> seconds-like latency` is any model of one iteration, e.g.
    `lambda reqs: predictor.predict([features...], [scene...])` on the measured surface."""

    def __init__(self, predict: Callable[[Sequence[Request]], float], max_budget: int):
        self.predict = predict
        self.B = int(max_budget)

    def forward(self, decodes: Sequence[int], prefills: Sequence[PrefillState], b: int):
        """(T_hat, A): A[i] = tokens given to prefill request i (in the order of the sorted set)."""
        b = max(len(decodes), min(int(b), self.B))
        left = b - len(decodes)
        alloc: List[int] = []
        for p in prefills:
            c = min(p.remaining, left)
            alloc.append(c)
            left -= c
        reqs: List[Request] = [(1, int(u)) for u in decodes]
        reqs += [(c, p.cached) for c, p in zip(alloc, prefills) if c > 0]
        return (self.predict(reqs) if reqs else 0.0), alloc

    def pred(self, b: int, decodes: Sequence[int], prefills: Sequence[PrefillState]) -> float:
        return self.forward(decodes, prefills, b)[0]

    def time_to_budget(self, decodes: Sequence[int], prefills: Sequence[PrefillState], T: float) -> int:
        lo, hi = len(decodes), self.B
        if self.pred(lo, decodes, prefills) > T:
            return lo
        while lo < hi:                                   # invariant: Pred(lo) <= T
            mid = (lo + hi + 1) // 2
            if self.pred(mid, decodes, prefills) <= T:
                lo = mid
            else:
                hi = mid - 1
        return lo


def window_bounds(slacks: Sequence[float], tbt_slo: Sequence[float]) -> Tuple[float, float]:
    """(T_cur, T_next) of Eq. 14-15 over the protected decode requests."""
    t_cur = min(slacks)
    t_next = min(s - t_cur + L for s, L in zip(slacks, tbt_slo))
    return t_cur, t_next


def sliding_chunker(F: BatchForwarder, decodes: Sequence[int], prefills: Sequence[PrefillState], t_cur: float,
                    t_next: float, stop_width: int = 30):
    """Algorithm 1.  Returns (B*, A*, T*, B_sigma)."""
    b_cur = F.time_to_budget(decodes, prefills, t_cur)
    b_next = F.time_to_budget(decodes, prefills, t_next)
    b_sigma = b_cur + b_next
    l, r = max(len(decodes), b_sigma - F.B), min(F.B, b_sigma - len(decodes))
    l0, r0 = l, r
    two = lambda b: F.pred(b, decodes, prefills) + F.pred(b_sigma - b, decodes, prefills)
    while r - l > stop_width:
        m1 = l + (r - l) // 3
        m2 = r - (r - l) // 3
        if two(m1) <= two(m2):
            r = m2 - 1
        else:
            l = m1 + 1
    m = (l + r) // 2
    best_b, best_t, best_a = l0, float("inf"), []
    for b in (l0, r0, m):
        t_b, a_b = F.forward(decodes, prefills, b)
        t_b += F.pred(b_sigma - b, decodes, prefills)
        if t_b < best_t or (t_b == best_t and b > best_b):
            best_t, best_b, best_a = t_b, b, a_b
    return best_b, best_a, best_t, b_sigma


def surface_predict_fn(predictor) -> Callable[[Sequence[Request]], float]:
    """Adapter: a fitted predictor.BatchLatencyPredictor as the iteration-time model (microseconds)."""
    def fn(reqs: Sequence[Request]) -> float:
        x = features(reqs)
        return float(predictor.predict([[x[f"x{j}"] for j in range(1, 8)]], [scene(reqs)])[0])
    return fn
