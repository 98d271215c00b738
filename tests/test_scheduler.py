"""Multi-Level Priority Sorter, Violation Checker, BatchConstructor and one scheduling round (§3.1, §3.3, §3.5,
Algorithm 2) — host-side, CPU only.  Checked against brute force on small instances and against the paper's statements."""
import itertools

import numpy as np

from paper_2606_05933_b200.chunker import BatchForwarder, PrefillState
from paper_2606_05933_b200.features import features
from paper_2606_05933_b200.scheduler import (DecodeRequest, PrefillRequest, ThroughputWindow, batch_constructor,
                                             knapsack_01, knapsack_values, priority_key, priority_sort,
                                             schedule_round, urgency, violation_check)


def _toy_model(reqs):
    """Eq. 5's form with non-negative weights (milliseconds)."""
    x = features(reqs)
    return 2.0 + 2.5e-6 * x["x1"] + 0.02 * x["x4"] + 5e-5 * x["x5"] + 0.004 * x["x6"]


def test_priority_key_eq_7_to_13():
    t, rho = 100.0, 10.0                                   # 10 tokens per ms
    a = PrefillRequest(1, arrival=0.0, ttft_slo=150.0, prompt_len=1000, computed=400)       # r = 600, s = 50
    assert a.remaining() == 600 and a.slack(t) == 50.0
    assert urgency(a, t, rho) == 600 / (10.0 * 50.0)       # Eq. 10: 1.2 > alpha = 1 -> urgent
    assert priority_key(a, t, rho) == (1, 0, 600)
    b = PrefillRequest(2, arrival=90.0, ttft_slo=200.0, prompt_len=500)                     # r = 500, s = 190 -> 0.26
    assert priority_key(b, t, rho) == (1, 1, 500)
    g = PrefillRequest(3, arrival=95.0, ttft_slo=500.0, prompt_len=4000, safeguard=1)       # protected: first level
    late = PrefillRequest(4, arrival=0.0, ttft_slo=90.0, prompt_len=10)                     # slack < 0 -> eps -> urgent
    assert urgency(late, t, rho) == 10 / (10.0 * 1e-3) and priority_key(late, t, rho) == (1, 0, 10)
    order = [r.rid for r in priority_sort([b, a, late, g], t, rho)]
    assert order == [3, 4, 1, 2]       # safeguard first; then urgent ones by fewer remaining tokens; then the rest


def test_throughput_window_rho():
    w = ThroughputWindow(window=2, initial=5.0)
    assert w.rho == 5.0
    w.observe(1000, 10.0)
    w.observe(3000, 10.0)
    assert w.rho == 200.0
    w.observe(1000, 10.0)              # the oldest sample leaves the window
    assert w.rho == 200.0


def test_knapsack_matches_brute_force():
    rng = np.random.default_rng(0)
    for _ in range(200):
        n = int(rng.integers(0, 9))
        w = [int(x) for x in rng.integers(1, 40, size=n)]
        v = [float(x) for x in rng.uniform(0.1, 5.0, size=n)]
        cap = int(rng.integers(0, 90))
        got = knapsack_01(w, v, cap)
        assert sum(w[i] for i in got) <= cap and len(set(got)) == len(got)
        best = max((sum(v[i] for i in sub) for k in range(n + 1) for sub in itertools.combinations(range(n), k)
                    if sum(w[i] for i in sub) <= cap), default=0.0)
        assert abs(sum(v[i] for i in got) - best) < 1e-9


def test_value_function_prefers_small_slack_and_few_tokens():
    """'prioritizes requests with smaller slack values and fewer remaining tokens'."""
    v = knapsack_values([10.0, 40.0, 10.0], [100, 100, 400])
    assert v[0] > v[1] and v[0] > v[2]
    assert abs(v[0] - 1.0 / (10 / 60 + 100 / 600)) < 1e-12


def _brute_force_constructor(F, decodes, cands, t):
    """Algorithm 2 by exhaustive subset search per anchor: same feasibility, value and COMPARER definitions."""
    states = [PrefillState(c.remaining(), c.computed) for c in cands]
    t_full, _ = F.forward(decodes, states, F.B)
    r = [c.remaining() for c in cands]
    s = [c.slack(t) for c in cands]
    risk = [j for j in range(len(cands)) if s[j] < t_full]
    if not risk:
        return "no-risk"
    best = None
    for a in risk:
        c_a = min(F.B, F.time_to_budget(decodes, states, s[a])) - len(decodes)
        if c_a <= 0 or r[a] > c_a:
            continue
        S_a = [j for j in range(len(cands)) if s[j] >= s[a]]
        vals = dict(zip(S_a, knapsack_values([s[j] for j in S_a], [r[j] for j in S_a])))
        others = [j for j in S_a if j != a]
        top = None
        for k in range(len(others) + 1):
            for sub in itertools.combinations(others, k):
                if sum(r[j] for j in sub) <= c_a - r[a]:
                    key = (sum(vals[j] for j in sub), len(sub), sum(r[j] for j in sub))
                    if top is None or key > top[0]:
                        top = (key, sub)
        Y = sorted(list(top[1]) + [a])
        key = (len(Y), sum(vals[j] for j in Y), sum(r[j] for j in Y))
        if best is None or key > best[0]:
            best = (key, Y)
    return best


def test_batch_constructor_matches_exhaustive_search():
    rng = np.random.default_rng(3)
    triggered = 0
    for trial in range(60):
        F = BatchForwarder(_toy_model, max_budget=int(rng.integers(512, 4096)))
        decodes = [int(u) for u in rng.integers(10, 4000, size=int(rng.integers(0, 40)))]
        t = 1000.0
        cands = [PrefillRequest(i, arrival=t - float(rng.uniform(0, 50)), ttft_slo=float(rng.uniform(52, 75)),
                                prompt_len=int(rng.integers(50, 1500)), computed=int(rng.integers(0, 40)))
                 for i in range(int(rng.integers(1, 7)))]
        cands = priority_sort(cands, t, rho=100.0)
        dec = batch_constructor(F, decodes, cands, t)
        ref = _brute_force_constructor(F, decodes, cands, t)
        if ref == "no-risk":
            assert dec is None
            continue
        if ref is None:                                              # at risk, but no anchor can be saved: decode-only
            assert dec is not None and dec.prefill_alloc == {} and dec.budget == len(decodes)
            continue
        triggered += 1
        assert dec is not None and dec.branch == "batch_constructor" and dec.decode_tokens == len(decodes)
        chosen = sorted(j for j, c in enumerate(cands) if c.rid in dec.prefill_alloc)
        assert chosen == ref[1]                                      # the same set the exhaustive search picks
        # every chosen request gets its FULL remaining prefill (Eq. 22); the batch fits the anchor's token capacity
        # C_a = min(B, TimeToBudget(s_a)) - |D| (Eq. 17) - the paper's proxy for "fits the anchor's deadline"
        for j in chosen:
            assert dec.prefill_alloc[cands[j].rid] == cands[j].remaining()
        anchor = next(c for c in cands if c.rid == dec.info["anchor"])
        states = [PrefillState(c.remaining(), c.computed) for c in cands]
        assert dec.budget <= min(F.B, F.time_to_budget(decodes, states, anchor.slack(t)))
        assert dec.budget == len(decodes) + sum(dec.prefill_alloc.values()) <= F.B
    assert triggered >= 10


def test_batch_constructor_returns_none_without_risk_and_skips_infeasible_anchors():
    F = BatchForwarder(_toy_model, max_budget=1024)
    t = 0.0
    relaxed = [PrefillRequest(1, 0.0, 1e6, 300), PrefillRequest(2, 0.0, 1e6, 900)]
    assert batch_constructor(F, [100] * 8, relaxed, t) is None                     # Algorithm 2 line 8
    # an anchor whose remaining prefill cannot fit its own slack is skipped (line 18): decision stays decode-only
    doomed = [PrefillRequest(1, 0.0, 2.05, 900)]
    dec = batch_constructor(F, [100] * 8, doomed, t)
    assert dec is not None and dec.prefill_alloc == {} and dec.budget == 8


def test_figure_2_scenario_skips_requests_to_save_the_tight_ones():
    """four prefill requests; the full batch would violate r1..r3; the constructor keeps the ones it can
    still save this round and leaves the rest for a later iteration.  Latency model linear in the token count, so the
    token capacity of Eq. 17 is exact."""
    model = lambda reqs: 2.0 + 0.01 * sum(c for c, _ in reqs)
    F = BatchForwarder(model, max_budget=4096)
    t = 0.0
    full = model([(800, 0), (1500, 0), (700, 0), (900, 0)])                  # 41 ms
    tight = model([(800, 0), (700, 0)]) + 0.05                               # 17.05 ms: room for r1 + r3 only
    cands = [PrefillRequest(1, 0.0, tight, 800), PrefillRequest(2, 0.0, tight * 0.5, 1500),
             PrefillRequest(3, 0.0, tight, 700), PrefillRequest(4, 0.0, full * 3, 900)]
    risky, t_full, _ = violation_check(F, [], priority_sort(cands, t, 100.0), t)
    assert set(risky) == {1, 2, 3} and abs(t_full - full) < 1e-9
    dec = batch_constructor(F, [], priority_sort(cands, t, 100.0), t)
    assert set(dec.prefill_alloc) == {1, 3} and dec.predicted <= tight     # r2 cannot be saved, r4 can wait
    assert dec.prefill_alloc == {1: 800, 3: 700}                           # full remaining prefill each (Eq. 22)


def test_schedule_round_takes_the_right_branch():
    t = 0.0
    decodes = [DecodeRequest(i, ctx=500 + 10 * i, tbt_slo=40.0, last_token_time=-5.0) for i in range(16)]
    calm = [PrefillRequest(100, -10.0, 5000.0, 3000), PrefillRequest(101, -5.0, 5000.0, 600, computed=128)]
    d = schedule_round(_toy_model, 2048, decodes, calm[:1], calm[1:], t, rho=100.0)
    assert d.branch == "sliding_chunker" and d.decode_tokens == 16 and 16 <= d.budget <= 2048
    assert sum(d.prefill_alloc.values()) == d.budget - 16
    assert d.predicted <= d.info["t_cur"] + 1e-9                     # the round respects the tightest TBT slack (35 ms)
    tight = [PrefillRequest(200, -50.0, 58.0, 700), PrefillRequest(201, -1.0, 5000.0, 1800)]
    d2 = schedule_round(_toy_model, 2048, decodes, [], tight, t, rho=100.0)
    assert d2.branch == "batch_constructor" and 200 in d2.prefill_alloc and d2.prefill_alloc[200] == 700
    assert d2.predicted <= 8.0 + 1e-9                                # request 200's slack: -50 + 58 - 0
    d3 = schedule_round(_toy_model, 2048, decodes, [], [], t, rho=100.0)
    assert d3.branch == "decode_only" and d3.budget == 16


def test_a_doomed_request_does_not_starve_healthy_prefill():
    """a request that can no longer meet its TTFT (slack <= 0, so no anchor is feasible) makes Algorithm 2 end
    on its empty placeholder every round.  The round must then fall through to the SlidingChunker so the healthy
    requests behind it keep prefilling; simulated over several rounds."""
    decodes = [DecodeRequest(i, ctx=400 + i, tbt_slo=40.0, last_token_time=0.0) for i in range(8)]
    doomed = PrefillRequest(1, arrival=-100.0, ttft_slo=50.0, prompt_len=900)            # slack -50 at t = 0
    healthy = [PrefillRequest(2, 0.0, 5000.0, 1500), PrefillRequest(3, 0.0, 5000.0, 700)]
    reqs = {r.rid: r for r in [doomed] + healthy}
    t, first = 0.0, None
    for rnd in range(12):
        waiting = [r for r in reqs.values() if r.remaining() > 0]
        if not waiting:
            break
        for d in decodes:
            d.last_token_time = t
        dec = schedule_round(_toy_model, 1024, decodes, [], waiting, t, rho=100.0)
        first = first or dec
        assert dec.prefill_alloc, f"round {rnd}: prefill starved ({dec.branch})"
        assert sum(dec.prefill_alloc.values()) + dec.decode_tokens <= dec.budget <= 1024
        for rid, a in dec.prefill_alloc.items():
            assert 0 < a <= reqs[rid].remaining()
            reqs[rid].computed += a
        t += dec.predicted
    assert first.branch == "sliding_chunker" and first.info["unsavable"] == [1]
    assert all(r.remaining() == 0 for r in reqs.values()), "every request, the doomed one included, finishes its prefill"
