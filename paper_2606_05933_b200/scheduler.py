"""The rest of SlidingServe's scheduling round, host side, driven by the batch latency
predictor fitted on OUR measured B200 surface: Multi-Level Priority Sorter (§3.3, Eq. 6-13),
Violation Checker (§3.1 steps 3-6), BatchConstructor (§3.5, Eq. 17-22, Algorithm 2
:319-367) and one scheduling round that ties them to the SlidingChunker (chunker.py, Algorithm 1).  Tens of items
per round: plain Python.  The GPU runs what the round returns: a batch {(c_i, u_i)}.

Readings of silent / garbled passages (#17-#21):
  * epsilon (Eq. 10), alpha (Eq. 11), rho_t's window: named, no values.  Defaults here: epsilon = 1e-3 time units,
    alpha = 1.0 ("needs longer than its slack"), rho_t = tokens / time over the last `rho_window` executed rounds.
  * Eq. 18 is garbled; read as v_j = 1 / ( s_j / sum_{k in S_a} s_k  +  r_j / sum_{k in S_a} r_k ), which matches the
    sentence after it ("prioritizes requests with smaller slack values and fewer remaining tokens").
  * Algorithm 2 line 10 sorts "C": read as the candidate set = P; line 16 T_a = s_a; a request with
    r_j = 0 cannot occur in P.  Slacks <= 0 are clamped to epsilon inside Eq. 18 only.
  * COMPARER: lexicographic on (|Y|, sum v, sum r), larger wins; the initial (B_dec, empty) decision
    loses to any feasible anchor solution.
  * Violation Checker: "whether directly executing this largest candidate batch would increase the TTFT or generation
    latency risk" (PAPER.md:99 step 4) - read as: T_hat(max candidate batch) exceeds the TTFT slack of a prefill
    request in it (the R_risk test of Algorithm 2 line 6) -> BatchConstructor branch; else SlidingChunker branch.
"""
from __future__ import annotations

from collections import deque
from dataclasses import dataclass, field
from typing import Callable, Deque, Dict, List, Optional, Sequence, Tuple

from .chunker import BatchForwarder, PrefillState, sliding_chunker, window_bounds

Request = Tuple[int, int]          # (tokens this round c_i, cached tokens u_i)  -- PAPER.md:107


@dataclass
class PrefillRequest:
    """A waiting or prefilling request (Eq. 6-8)."""
    rid: int
    arrival: float                 # a_i
    ttft_slo: float                # L_i^ttft
    prompt_len: int                # p_i
    computed: int = 0              # c_i(t): prompt tokens already prefilled (= cached tokens u_i)
    safeguard: int = 0             # g_i

    def remaining(self) -> int:    # r_i(t) = p_i - c_i(t)                         (Eq. 7)
        return self.prompt_len - self.computed

    def slack(self, t: float) -> float:   # s_i(t) = a_i + L_i^ttft - t            (Eq. 8)
        return self.arrival + self.ttft_slo - t


@dataclass
class DecodeRequest:
    rid: int
    ctx: int                       # u_i
    tbt_slo: float                 # L_i^tbt
    last_token_time: float         # its TBT slack at time t is last_token_time + L^tbt - t

    def slack(self, t: float) -> float:
        return self.last_token_time + self.tbt_slo - t


# ------------------------------------------------------------------------------------------------------------------
# 3.3 Multi-Level Priority Sorter
# ------------------------------------------------------------------------------------------------------------------
class ThroughputWindow:
    """rho_t: recently observed system throughput (tokens per time unit) over the last `window` executed rounds."""

    def __init__(self, window: int = 16, initial: float = 1.0):
        self.samples: Deque[Tuple[int, float]] = deque(maxlen=window)
        self.initial = float(initial)

    def observe(self, tokens: int, elapsed: float) -> None:
        if elapsed > 0:
            self.samples.append((int(tokens), float(elapsed)))

    @property
    def rho(self) -> float:
        tok = sum(s[0] for s in self.samples)
        tim = sum(s[1] for s in self.samples)
        return tok / tim if tim > 0 and tok > 0 else self.initial


def urgency(req: PrefillRequest, t: float, rho: float, eps: float = 1e-3) -> float:
    """u_i(t) = r_i(t) / (rho_t * max(s_i(t), eps))                                 (Eq. 9-10)."""
    return req.remaining() / (rho * max(req.slack(t), eps))


def priority_key(req: PrefillRequest, t: float, rho: float, alpha: float = 1.0, eps: float = 1e-3):
    """K_i(t) = (1 - g_i, 1 - e_i(t), r_i(t)),  e_i = 1[u_i(t) > alpha]              (Eq. 11-12)."""
    e = 1 if urgency(req, t, rho, eps) > alpha else 0
    return (1 - req.safeguard, 1 - e, req.remaining())


def priority_sort(cands: Sequence[PrefillRequest], t: float, rho: float, alpha: float = 1.0,
                  eps: float = 1e-3) -> List[PrefillRequest]:
    """Q_t = LexSort over P_t = P_prefill U P_wait, ascending K_i(t) (Eq. 6, 13); stable, ties keep arrival order."""
    return sorted(cands, key=lambda r: priority_key(r, t, rho, alpha, eps))


# ------------------------------------------------------------------------------------------------------------------
# 3.5 BatchConstructor
# ------------------------------------------------------------------------------------------------------------------
def knapsack_01(weights: Sequence[int], values: Sequence[float], capacity: int) -> List[int]:
    """0/1 knapsack by dynamic programming over capacity (Eq. 19): indices of the chosen items.  Maximises the total
    value; among equal values prefers more items, then more weight (COMPARER's order), so the result is unique up
    to exact float ties."""
    n = len(weights)
    capacity = max(int(capacity), 0)
    # best[c] = (value, count, weight) achievable with capacity c using the items seen so far
    best = [(0.0, 0, 0)] * (capacity + 1)
    take = [[False] * (capacity + 1) for _ in range(n)]
    for i in range(n):
        w, v = int(weights[i]), float(values[i])
        if w > capacity:
            continue
        for c in range(capacity, w - 1, -1):
            cand = (best[c - w][0] + v, best[c - w][1] + 1, best[c - w][2] + w)
            if cand > best[c]:
                best[c] = cand
                take[i][c] = True
    chosen, c = [], capacity
    for i in range(n - 1, -1, -1):
        if take[i][c]:
            chosen.append(i)
            c -= int(weights[i])
    return sorted(chosen)


def knapsack_values(slacks: Sequence[float], remaining: Sequence[int], eps: float = 1e-3) -> List[float]:
    """v_j = 1 / ( s_j / sum_k s_k + r_j / sum_k r_k ) over the candidate set S_a          (Eq. 18, as read)."""
    s = [max(float(x), eps) for x in slacks]
    ssum, rsum = sum(s), float(sum(remaining))
    return [1.0 / (sj / ssum + rj / rsum) for sj, rj in zip(s, remaining)]


@dataclass
class BatchDecision:
    budget: int                                    # B*
    decode_tokens: int                             # |D| (each decode gets 1 token)
    prefill_alloc: Dict[int, int]                  # rid -> tokens this round
    branch: str                                    # "sliding_chunker" | "batch_constructor" | "decode_only"
    predicted: float = 0.0                         # T_hat of the decided batch
    info: dict = field(default_factory=dict)


def _states(cands: Sequence[PrefillRequest]) -> List[PrefillState]:
    return [PrefillState(r.remaining(), r.computed) for r in cands]


def batch_constructor(F: BatchForwarder, decodes: Sequence[int], cands: Sequence[PrefillRequest], t: float,
                      eps: float = 1e-3) -> Optional[BatchDecision]:
    """Algorithm 2.  `cands` is the sorted set P.  Returns None when no request is at risk (line 8)."""
    states = _states(cands)
    t_full, _ = F.forward(decodes, states, F.B)                                      # line 1
    r = [c.remaining() for c in cands]                                               # lines 2-5
    s = [c.slack(t) for c in cands]
    risk = [j for j in range(len(cands)) if s[j] < t_full]                           # line 6
    if not risk:
        return None                                                                  # line 8
    order = sorted(range(len(cands)), key=lambda j: (s[j], r[j]))                    # line 10
    b_dec = len(decodes)                                                             # lines 11-12
    best_key, best = None, BatchDecision(b_dec, b_dec, {}, "batch_constructor")      # line 13
    for a in risk:                                                                   # line 14
        b_a = F.time_to_budget(decodes, states, s[a])                                # line 16 (T_a = s_a)
        c_a = min(F.B, b_a) - b_dec                                                  # line 17 (Eq. 17)
        if c_a <= 0 or r[a] > c_a:
            continue                                                                 # lines 18-20
        S_a = [j for j in order if s[j] >= s[a]]                                     # line 21
        vals = dict(zip(S_a, knapsack_values([s[j] for j in S_a], [r[j] for j in S_a], eps)))   # line 22
        others = [j for j in S_a if j != a]
        pick = knapsack_01([r[j] for j in others], [vals[j] for j in others], c_a - r[a])       # line 23
        Y = sorted([others[i] for i in pick] + [a])                                  # line 24 (Eq. 20)
        key = (len(Y), sum(vals[j] for j in Y), sum(r[j] for j in Y))                # COMPARER
        if best_key is None or key > best_key:                                       # lines 27-29
            best_key = key
            best = BatchDecision(b_dec + sum(r[j] for j in Y), b_dec, {cands[j].rid: r[j] for j in Y},
                                 "batch_constructor", info={"anchor": cands[a].rid, "t_full": t_full})
    best.info.setdefault("t_full", t_full)
    best.info["risk"] = [cands[j].rid for j in risk]
    reqs = [(1, int(u)) for u in decodes] + [(best.prefill_alloc[c.rid], c.computed) for c in cands if c.rid in best.prefill_alloc]
    best.predicted = F.predict(reqs) if reqs else 0.0
    return best                                                                      # line 31 (Eq. 22)


# ------------------------------------------------------------------------------------------------------------------
# 3.1 one scheduling round: sorter -> max candidate batch -> violation checker -> SlidingChunker | BatchConstructor
# ------------------------------------------------------------------------------------------------------------------
def violation_check(F: BatchForwarder, decodes: Sequence[int], cands: Sequence[PrefillRequest], t: float):
    """Steps (3)-(4): build the maximum candidate batch (budget B, sorted order) and compare its predicted time with
    the TTFT slack of the prefill requests in it.  Returns (at_risk rids, T_hat_full, allocation)."""
    t_full, alloc = F.forward(decodes, _states(cands), F.B)
    risky = [c.rid for c, a in zip(cands, alloc) if a > 0 and c.slack(t) < t_full]
    return risky, t_full, alloc


def schedule_round(predict: Callable[[Sequence[Request]], float], max_budget: int, decodes: Sequence[DecodeRequest],
                   prefilling: Sequence[PrefillRequest], waiting: Sequence[PrefillRequest], t: float, rho: float,
                   alpha: float = 1.0, eps: float = 1e-3) -> BatchDecision:
    """Steps (2)-(8) of PAPER.md:99.  `predict` is the batch latency model (time units = the SLOs' units)."""
    F = BatchForwarder(predict, max_budget)
    dctx = [d.ctx for d in decodes]
    cands = priority_sort(list(prefilling) + list(waiting), t, rho, alpha, eps)      # step (2)
    if not cands:
        return BatchDecision(len(dctx), len(dctx), {}, "decode_only",
                             predicted=predict([(1, u) for u in dctx]) if dctx else 0.0)
    risky, t_full, _ = violation_check(F, dctx, cands, t)                             # steps (3)-(4)
    unsavable = []
    if risky:                                                                         # step (6)
        dec = batch_constructor(F, dctx, cands, t, eps)
        # Algorithm 2 ends with its line-13 placeholder (B_dec, {}) when no at-risk anchor can still be saved this round
        # (e.g. a request whose slack is already <= 0).  Running that as the round would repeat forever - the doomed
        # request only gets riskier - and starve every healthy prefill behind it.  An empty Y* is therefore read as
        # Algorithm 2's "no decision" and the round falls through to the SlidingChunker (reading 24).
        if dec is not None and dec.prefill_alloc:
            return dec
        unsavable = risky
    # step (5): SlidingChunker.  Protected decodes = all decodes (g_i = 1 for decoding requests)
    states = _states(cands)
    if decodes:
        t_cur, t_next = window_bounds([d.slack(t) for d in decodes], [d.tbt_slo for d in decodes])
    else:
        t_cur = t_next = float("inf")
    if t_cur == float("inf"):
        b_star, t_star = F.B, None
        _, a_star = F.forward(dctx, states, b_star)
        b_sigma = 2 * F.B
    else:
        b_star, a_star, t_star, b_sigma = sliding_chunker(F, dctx, states, t_cur, t_next)
    alloc = {c.rid: a for c, a in zip(cands, a_star) if a > 0}
    reqs = [(1, u) for u in dctx] + [(a, c.computed) for c, a in zip(cands, a_star) if a > 0]
    return BatchDecision(b_star, len(dctx), alloc, "sliding_chunker", predicted=predict(reqs) if reqs else 0.0,
                         info={"t_cur": t_cur, "t_next": t_next, "b_sigma": b_sigma, "t_two_window": t_star,
                               "t_full": t_full, "unsavable": unsavable})
