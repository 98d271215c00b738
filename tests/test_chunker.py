"""SlidingChunker (§3.4, Algorithm 1) — host-side, CPU only."""
import numpy as np

from paper_2606_05933_b200.chunker import BatchForwarder, PrefillState, sliding_chunker, surface_predict_fn, window_bounds
from paper_2606_05933_b200.features import features
from paper_2606_05933_b200.predictor import BatchLatencyPredictor, load_surface


def _toy_model(reqs):
    """A latency model of the paper's form (Eq. 5): intercept + weights on Table 1's features."""
    x = features(reqs)
    return 8.0 + 2.5e-5 * x["x1"] + 0.12 * x["x4"] + 5e-4 * x["x5"] + 0.01 * x["x6"]


def test_forward_allocates_in_sorted_order_and_respects_the_budget():
    F = BatchForwarder(_toy_model, max_budget=512)
    dec = [100, 2000, 30]
    pre = [PrefillState(200, 0), PrefillState(1000, 64), PrefillState(50, 10)]
    T, A = F.forward(dec, pre, 403)
    assert A == [200, 200, 0] and sum(A) + len(dec) == 403
    T2, A2 = F.forward(dec, pre, 10_000)                     # clamped to B = 512
    assert sum(A2) + len(dec) == 512 and A2 == [200, 309, 0]
    T0, A0 = F.forward(dec, pre, 0)                          # never below the decode tokens
    assert A0 == [0, 0, 0] and T0 == _toy_model([(1, u) for u in dec])
    assert T0 < T < T2


def test_time_to_budget_is_the_largest_feasible_budget():
    F = BatchForwarder(_toy_model, max_budget=2048)
    dec = list(np.random.default_rng(0).integers(10, 4000, size=20))
    pre = [PrefillState(1500, 0), PrefillState(3000, 500)]
    for T in (1.0, 30.0, 45.0, 80.0, 1e9):
        b = F.time_to_budget(dec, pre, T)
        brute = [x for x in range(len(dec), F.B + 1) if F.pred(x, dec, pre) <= T]
        assert b == (max(brute) if brute else len(dec))


def test_window_bounds_eq_14_15():
    t_cur, t_next = window_bounds([30.0, 12.0, 50.0], [40.0, 40.0, 25.0])
    assert t_cur == 12.0 and t_next == min(30 - 12 + 40, 12 - 12 + 40, 50 - 12 + 25)


def test_ternary_search_matches_brute_force_on_the_two_window_objective():
    rng = np.random.default_rng(1)
    for trial in range(20):
        dec = list(rng.integers(10, 6000, size=int(rng.integers(1, 64))))
        pre = [PrefillState(int(rng.integers(50, 4000)), int(rng.integers(0, 2000))) for _ in range(int(rng.integers(1, 5)))]
        F = BatchForwarder(_toy_model, max_budget=int(rng.integers(256, 4096)))
        t_cur, t_next = float(rng.uniform(15, 80)), float(rng.uniform(15, 120))
        b_star, a_star, t_star, b_sigma = sliding_chunker(F, dec, pre, t_cur, t_next)
        assert len(dec) <= b_star <= F.B and sum(a_star) <= b_star - len(dec)
        two = lambda b: F.pred(b, dec, pre) + F.pred(b_sigma - b, dec, pre)
        assert abs(t_star - two(b_star)) < 1e-9
        # Algorithm 1 evaluates {l0, r0, mid of the final bracket}: never worse than both ends of the range, and within
        # the final bracket's resolution of the exhaustive optimum of the (here unimodal-or-flat) objective
        lo, hi = max(len(dec), b_sigma - F.B), min(F.B, b_sigma - len(dec))      # both windows get a runnable budget
        assert lo <= b_star <= hi
        best = min(two(b) for b in range(lo, hi + 1))
        assert t_star <= min(two(lo), two(hi)) + 1e-9
        assert t_star - best <= 0.02 * best + 0.5


def _fitted_forwarder(max_budget):
    from pathlib import Path
    prof = Path(__file__).resolve().parent.parent / "profiles"
    rows, X, y, scenes, shapes = load_surface([str(prof / "r2_surface.csv"), str(prof / "r2_surface_dense.csv")])
    keep = [i for i, s in enumerate(shapes) if s == "32/8/128"]
    p = BatchLatencyPredictor(fit="nnls").fit(X[keep], y[keep], [scenes[i] for i in keep])
    return BatchForwarder(surface_predict_fn(p), max_budget=max_budget), p


def test_fitted_predictor_is_monotone_in_the_budget_inside_a_scene():
    """The non-negative fit (reading 16): Pred(b) never decreases as the budget grows while the batch stays
    in one scene (the expert models of two scenes may disagree at the scene switch b = |D| -> |D| + 1, as the paper's do)."""
    F, p = _fitted_forwarder(4096)
    for w in p.experts.values():
        a = w.weights
        assert a[0] >= 0 and a[1] >= -0.5 * a[0] - 1e-18 and (a[2:] >= 0).all()
    rng = np.random.default_rng(5)
    for trial in range(5):
        dec = list(rng.integers(200, 6000, size=int(rng.integers(8, 128))))
        pre = [PrefillState(int(rng.integers(500, 6000)), int(rng.integers(0, 3000))) for _ in range(int(rng.integers(1, 4)))]
        # a request that is handed exactly 1 token counts as a decode (D = {c_i <= 1}): those budgets
        # switch features / scene and are left out
        bs = [b for b in range(len(dec) + 2, 4097, 37) if 1 not in F.forward(dec, pre, b)[1]]
        t = [F.pred(b, dec, pre) for b in bs]
        assert all(y2 >= y1 - 1e-9 for y1, y2 in zip(t, t[1:]))


def test_chunker_on_the_measured_surface():
    """End to end with the predictor fitted (non-negative weights) on the committed B200 latency surface: TimeToBudget is
    the largest feasible budget (brute force over the mixed-scene range), Algorithm 1's result is the two-window
    objective at B*, never worse than both ends of the range and within the final bracket's resolution of the
    exhaustive optimum."""
    F, _ = _fitted_forwarder(4096)
    dec = list(np.random.default_rng(2).integers(200, 6000, size=64))
    pre = [PrefillState(3800, 0), PrefillState(1900, 1024)]
    lo = len(dec) + 2                                         # first budget of the mixed scene (1 token = a decode)
    for T in (150.0, 180.0, 250.0, 400.0, 1e9):
        b = F.time_to_budget(dec, pre, T)
        feas = [x for x in range(lo, F.B + 1) if F.pred(x, dec, pre) <= T]
        if feas and F.pred(len(dec), dec, pre) <= T:
            assert b == max(feas)
    for slack in (160.0, 180.0, 250.0, 400.0):
        b_star, a_star, t_star, b_sigma = sliding_chunker(F, dec, pre, slack, slack - 30.0)
        assert len(dec) <= b_star <= F.B
        assert sum(a_star) == min(b_star - len(dec), 5700) and a_star[0] == min(3800, b_star - len(dec))
        two = lambda b: F.pred(b, dec, pre) + F.pred(b_sigma - b, dec, pre)
        assert abs(t_star - two(b_star)) < 1e-9
        lo_b, hi_b = max(len(dec), b_sigma - F.B), min(F.B, b_sigma - len(dec))
        assert lo_b <= b_star <= hi_b
        assert t_star <= min(two(lo_b), two(hi_b)) + 1e-9
        best = min(two(b) for b in range(lo_b, hi_b + 1, 7))
        assert t_star - best <= 0.02 * best + 0.5


def test_fig1_example_runs_on_the_committed_surface():
    from paper_2606_05933_b200 import fig1_example as ex
    dec, pre, B, t_cur, t_next = ex.scenario()
    F = ex.fitted_forwarder(B)
    single, sliding, b_sigma = ex.plan(F, dec, pre, t_cur, t_next)
    assert sum(single) == b_sigma == sum(sliding)
    two = lambda b: F.pred(b, dec, pre) + F.pred(b_sigma - b, dec, pre)
    assert two(sliding[0]) <= two(single[0]) + 1e-9            # Eq. 16 on the unchanged (D, P)
    assert F.pred(single[0], dec, pre) <= t_cur and F.pred(single[1], dec, pre) <= t_next


def test_plenty_of_slack_does_not_drop_the_prefill():
    """With slack for two full iterations (B_sigma = 2B) the only split that keeps B_sigma tokens in two runnable
    windows is b = B; the round-2 clamped objective chose b = |D| (decode only) here and starved the prefill."""
    F = BatchForwarder(_toy_model, max_budget=1024)
    dec, pre = [400 + i for i in range(8)], [PrefillState(900, 0), PrefillState(1500, 0)]
    b_star, a_star, _, b_sigma = sliding_chunker(F, dec, pre, 1e6, 1e6)
    assert b_sigma == 2048 and b_star == 1024 and a_star == [900, 116]
