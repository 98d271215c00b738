"""Pins for the fp64 oracle (CPU only).  Each test fixes the oracle to something other than itself:
a closed form, an invariant, a library routine on de-paged tensors, brute force in another precision
and loop order, or hand-computed numbers from the paper's Table 1 definitions (tests/golden/).
A dropped term, wrong sign/index, transposed operand or off-by-one mask in oracle/attn_oracle.c
fails at least one of them."""
import math
from pathlib import Path

import numpy as np
import pytest
import torch

import oracle
from paper_2606_05933_b200 import features as ft
from paper_2606_05933_b200 import workloads as wl
from helpers import depage, f64_to_u16, host_arrays, oracle_run, u16_to_f64

GOLDEN = Path(__file__).parent / "golden"


def small_batch(seed=11, Hq=4, Hkv=2, D=8, reqs=((5, 3), (1, 7), (1, 0), (3, 0), (0, 4), (1, 20), (18, 15))):
    b = wl.make_batch("small", Hq, Hkv, D, list(reqs), seed, with_append=False)
    t = wl.make_tensors(b, "cpu")
    return b, host_arrays(b, t)


# ---------------------------------------------------------------------------------------------
# 1. brute force: long double, dense un-paged K/V, explicit 0/1 mask matrix, NO max-subtraction,
#    loop order (head, request) instead of (row, head)
# ---------------------------------------------------------------------------------------------
def test_bruteforce_longdouble_no_max_subtraction():
    b, a = small_batch()
    out, lse, pairs, _, _ = oracle_run(b, a)
    G = b.num_q_heads // b.num_kv_heads
    qf = u16_to_f64(a["q"]).astype(np.longdouble)
    scale = np.longdouble(np.float32(b.scale))
    checked = 0
    for h in range(b.num_q_heads):
        for r, (c, u) in enumerate(b.reqs):
            if c == 0:
                continue
            n = c + u
            K = depage(b, a["k_cache"], r, n)[:, h // G, :].astype(np.longdouble)
            V = depage(b, a["v_cache"], r, n)[:, h // G, :].astype(np.longdouble)
            Q = qf[b.query_start_loc[r]:b.query_start_loc[r + 1], h, :]
            mask = np.zeros((c, n), dtype=np.longdouble)
            for j in range(c):
                mask[j, :u + j + 1] = 1
            E = np.exp(scale * (Q @ K.T)) * mask                  # no max subtraction
            P = E / E.sum(axis=1, keepdims=True)
            ref = (P @ V).astype(np.float64)
            got = out[b.query_start_loc[r]:b.query_start_loc[r + 1], h, :]
            np.testing.assert_allclose(got, ref, rtol=0, atol=1e-12)
            ref_lse = np.log(E.sum(axis=1)).astype(np.float64)
            np.testing.assert_allclose(lse[b.query_start_loc[r]:b.query_start_loc[r + 1], h], ref_lse,
                                       rtol=0, atol=1e-12)
            checked += c
    assert checked == b.T * b.num_q_heads
    assert pairs == ft.causal_pairs(b.reqs)


# ---------------------------------------------------------------------------------------------
# 2. closed forms
# ---------------------------------------------------------------------------------------------
def prefix_mean(b, a, r, j, g):
    u = b.reqs[r][1]
    V = depage(b, a["v_cache"], r, u + j + 1)[:, g, :]
    return V.mean(axis=0)


def check_prefix_mean(b, a, out):
    G = b.num_q_heads // b.num_kv_heads
    for r, (c, u) in enumerate(b.reqs):
        for j in range(c):
            for h in range(b.num_q_heads):
                np.testing.assert_allclose(out[b.query_start_loc[r] + j, h], prefix_mean(b, a, r, j, h // G),
                                           rtol=0, atol=1e-13)


def test_scale_zero_is_prefix_mean():
    b, a = small_batch(seed=12)
    out, lse, _, _, _ = oracle_run(b, a, scale=0.0)
    check_prefix_mean(b, a, out)
    # lse = log(number of visible keys)
    for r, (c, u) in enumerate(b.reqs):
        for j in range(c):
            np.testing.assert_allclose(lse[b.query_start_loc[r] + j], math.log(u + j + 1), atol=1e-13)


def test_zero_query_is_prefix_mean():
    b, a = small_batch(seed=13)
    a["q"][:] = 0
    out, _, _, _, _ = oracle_run(b, a)
    check_prefix_mean(b, a, out)


def test_equal_keys_is_prefix_mean():
    b, a = small_batch(seed=14)
    row = a["k_cache"][0, 0, 0, :].copy()
    a["k_cache"][:, :, :, :] = row
    out, _, _, _, _ = oracle_run(b, a)
    check_prefix_mean(b, a, out)


def test_single_cached_key_returns_v_exactly():
    # u = 0, c = 1: the row sees only its own key -> out == V[0] bit for bit (north_star invariant)
    b = wl.make_batch("one", 4, 2, 16, [(1, 0), (1, 0)], 21)
    a = host_arrays(b, wl.make_tensors(b, "cpu"))
    out, lse, pairs, _, _ = oracle_run(b, a)
    assert pairs == 2
    for r in range(2):
        V0 = depage(b, a["v_cache"], r, 1)[0]            # [Hkv, D]
        for h in range(4):
            assert np.array_equal(out[r, h], V0[h // 2])
    # and through kv_append: the key written this iteration is the one seen
    b2 = wl.make_batch("one-append", 4, 2, 16, [(1, 0)], 22, with_append=True)
    a2 = host_arrays(b2, wl.make_tensors(b2, "cpu"))
    out2, _, _, _, _ = oracle_run(b2, a2)
    vn = u16_to_f64(a2["v_new"])
    for h in range(4):
        assert np.array_equal(out2[0, h], vn[0, h // 2])


def test_convexity_and_lse_bounds():
    b, a = small_batch(seed=15)
    out, lse, _, _, _ = oracle_run(b, a)
    G = b.num_q_heads // b.num_kv_heads
    qf = u16_to_f64(a["q"])
    for r, (c, u) in enumerate(b.reqs):
        for j in range(c):
            n = u + j + 1
            K = depage(b, a["k_cache"], r, n)
            V = depage(b, a["v_cache"], r, n)
            row = b.query_start_loc[r] + j
            for h in range(b.num_q_heads):
                g = h // G
                assert np.all(out[row, h] <= V[:, g, :].max(axis=0) + 1e-12)
                assert np.all(out[row, h] >= V[:, g, :].min(axis=0) - 1e-12)
                s = float(np.float32(b.scale)) * (K[:, g, :] @ qf[row, h])
                assert lse[row, h] >= s.max() - 1e-12
                assert lse[row, h] <= s.max() + math.log(n) + 1e-12


# ---------------------------------------------------------------------------------------------
# 3. needle keys: pin the mask off-by-one, the page walk and the slot index
# ---------------------------------------------------------------------------------------------
def set_row(b, cache, r, t, g, vec_f64):
    page = int(b.block_table[r, t // b.page_size])
    cache[page, g, t % b.page_size, :] = f64_to_u16(np.asarray(vec_f64, dtype=np.float64))


@pytest.mark.parametrize("c,u", [(1, 40), (6, 30), (20, 0), (3, 15), (2, 16), (40, 17)])
def test_needle_positions(c, u):
    D, Hq, Hkv = 16, 2, 1
    b = wl.make_batch("needle", Hq, Hkv, D, [(2, 5), (c, u), (1, 9)], 31)
    base = host_arrays(b, wl.make_tensors(b, "cpu"))
    r = 1
    n_total = c + u
    qdir = np.zeros(D)
    qdir[3] = 1.0
    beta = 64.0                                  # exactly representable in bf16
    scale = 1.0
    positions = sorted({0, max(u - 1, 0), u, n_total - 1, 15, 16, 31, 32} & set(range(n_total)))
    for j in (0, c - 1):
        row = int(b.query_start_loc[r]) + j
        visible = u + j + 1
        for pos in positions + ([visible] if visible < n_total else []):
            a = {k: v.copy() for k, v in base.items()}
            # all of request r's keys orthogonal to the query direction, small
            for t in range(n_total):
                kv = u16_to_f64(a["k_cache"][int(b.block_table[r, t // 16]), 0, t % 16, :])
                kv[3] = 0.0
                set_row(b, a["k_cache"], r, t, 0, 0.01 * kv)
            set_row(b, a["k_cache"], r, pos, 0, beta * qdir)
            a["q"][row, :, :] = f64_to_u16(np.tile(qdir, (Hq, 1)))
            out, _, _, _, _ = oracle_run(b, a, scale=scale)
            V = depage(b, a["v_cache"], r, n_total)[:, 0, :]
            if pos < visible:
                # softmax weight of the needle >= 1 - n*e^{-63}
                np.testing.assert_allclose(out[row, 0], V[pos], rtol=0, atol=1e-20 + 1e-24 * n_total)
            else:
                # the needle sits at u+j+1: must be invisible -> all visible scores are 0 -> prefix mean
                np.testing.assert_allclose(out[row, 0], V[:visible].mean(axis=0), rtol=0, atol=1e-13)


# ---------------------------------------------------------------------------------------------
# 4. library routine: torch fp64 softmax(QK^T*scale + mask) V on de-paged dense tensors
# ---------------------------------------------------------------------------------------------
def test_matches_torch_fp64_dense_softmax():
    b = wl.random_batch(41, Hq=8, Hkv=2, D=64, n_prefill=2, n_decode=4, max_c=70, max_u=150, with_append=False)
    a = host_arrays(b, wl.make_tensors(b, "cpu"))
    out, lse, pairs, _, _ = oracle_run(b, a)
    assert pairs == ft.causal_pairs(b.reqs)
    G = b.num_q_heads // b.num_kv_heads
    qf = torch.from_numpy(u16_to_f64(a["q"]))
    for r, (c, u) in enumerate(b.reqs):
        if c == 0:
            continue
        n = c + u
        K = torch.from_numpy(depage(b, a["k_cache"], r, n)).repeat_interleave(G, dim=1)   # [n,Hq,D]
        V = torch.from_numpy(depage(b, a["v_cache"], r, n)).repeat_interleave(G, dim=1)
        Q = qf[b.query_start_loc[r]:b.query_start_loc[r + 1]]                             # [c,Hq,D]
        s = torch.einsum("chd,nhd->hcn", Q, K) * float(np.float32(b.scale))
        mask = torch.arange(n)[None, :] > (u + torch.arange(c))[:, None]
        s = s.masked_fill(mask[None], float("-inf"))
        ref = torch.einsum("hcn,nhd->chd", torch.softmax(s, dim=-1), V).numpy()
        got = out[b.query_start_loc[r]:b.query_start_loc[r + 1]]
        np.testing.assert_allclose(got, ref, rtol=0, atol=1e-10)
        ref_lse = torch.logsumexp(s, dim=-1).T.numpy()
        np.testing.assert_allclose(lse[b.query_start_loc[r]:b.query_start_loc[r + 1]], ref_lse, atol=1e-10)


# ---------------------------------------------------------------------------------------------
# 5. invariants that hold bitwise in the oracle
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("chunks", [(40,), (1,) * 6, (15, 16, 17), (16, 1, 31), (127, 3), (5, 128, 7)])
def test_chunking_invariance_bitwise(chunks):
    """Prefill of L tokens as any chunk sequence == unchunked prefill (premise of PAPER.md:44)."""
    L = sum(chunks)
    Hq, Hkv, D = 4, 2, 16
    full = wl.make_batch("full", Hq, Hkv, D, [(L, 0)], 51, num_pages=2 * (L // 16 + 2), with_append=True)
    t = wl.make_tensors(full, "cpu")
    a = host_arrays(full, t)
    ref, ref_lse, _, kc_ref, vc_ref = oracle_run(full, a)
    k, v = a["k_cache"].copy(), a["v_cache"].copy()
    rows = []
    done = 0
    for c in chunks:
        step = wl.Batch("step", Hq, Hkv, D, [(c, done)], full.num_pages, full.block_table,
                        np.array([0, c], dtype=np.int32), np.array([done], dtype=np.int32), 51, True)
        oracle.kv_append(k, v, a["k_new"][done:done + c], a["v_new"][done:done + c], step.block_table,
                         step.query_start_loc, step.ctx_lens)
        o, l, _ = oracle.mixed_attention(a["q"][done:done + c], k, v, step.block_table, step.query_start_loc,
                                         step.ctx_lens, full.scale)
        rows.append((o, l))
        done += c
    got = np.concatenate([o for o, _ in rows])
    got_lse = np.concatenate([l for _, l in rows])
    assert np.array_equal(got, ref) and np.array_equal(got_lse, ref_lse)
    assert np.array_equal(k, kc_ref) and np.array_equal(v, vc_ref)


def test_decode_equals_last_prefill_row():
    Hq, Hkv, D, u = 4, 4, 8, 37
    pre = wl.make_batch("pre", Hq, Hkv, D, [(u + 1, 0)], 61, num_pages=16)
    a = host_arrays(pre, wl.make_tensors(pre, "cpu"))
    ref, _, _, _, _ = oracle_run(pre, a)
    dec = wl.Batch("dec", Hq, Hkv, D, [(1, u)], pre.num_pages, pre.block_table, np.array([0, 1], dtype=np.int32),
                   np.array([u], dtype=np.int32), 61)
    a2 = dict(a, q=a["q"][u:u + 1].copy())
    got, _, _, _, _ = oracle_run(dec, a2)
    assert np.array_equal(got[0], ref[u])


def test_page_permutation_invariance_bitwise():
    b, a = small_batch(seed=71)
    ref, _, _, _, _ = oracle_run(b, a)
    rng = np.random.default_rng(5)
    perm = rng.permutation(b.num_pages)                      # new physical id of old page p is perm[p]
    k2, v2 = np.empty_like(a["k_cache"]), np.empty_like(a["v_cache"])
    k2[perm], v2[perm] = a["k_cache"], a["v_cache"]
    bt2 = np.where(b.block_table >= 0, perm[np.clip(b.block_table, 0, None)], -1).astype(np.int32)
    b2 = wl.Batch(b.name, b.num_q_heads, b.num_kv_heads, b.head_dim, b.reqs, b.num_pages, bt2,
                  b.query_start_loc, b.ctx_lens, b.seed)
    got, _, _, _, _ = oracle_run(b2, dict(a, k_cache=k2, v_cache=v2))
    assert np.array_equal(got, ref)
    # compact_pool (used by the GPU parity tests at large sizes) is such a permutation
    bt3, (k3, v3) = wl.compact_pool(b, torch.from_numpy(a["k_cache"].view(np.int16)).view(torch.bfloat16),
                                    torch.from_numpy(a["v_cache"].view(np.int16)).view(torch.bfloat16))
    b3 = wl.Batch(b.name, b.num_q_heads, b.num_kv_heads, b.head_dim, b.reqs, k3.shape[0], bt3,
                  b.query_start_loc, b.ctx_lens, b.seed)
    got3, _, _, _, _ = oracle_run(b3, dict(a, k_cache=k3, v_cache=v3))
    assert np.array_equal(got3, ref)


def test_batch_composition_and_order_invariance_bitwise():
    """Requests share a batch but are independent inside it."""
    b, a = small_batch(seed=81)
    ref, _, _, _, _ = oracle_run(b, a)
    order = [6, 2, 0, 5]                                     # drop some requests, reorder the rest
    reqs = [b.reqs[i] for i in order]
    qsl = np.zeros(len(order) + 1, dtype=np.int32)
    qsl[1:] = np.cumsum([c for c, _ in reqs])
    sel = np.concatenate([np.arange(b.query_start_loc[i], b.query_start_loc[i + 1]) for i in order])
    b2 = wl.Batch("sub", b.num_q_heads, b.num_kv_heads, b.head_dim, reqs, b.num_pages,
                  b.block_table[order], qsl, b.ctx_lens[order], b.seed)
    got, _, _, _, _ = oracle_run(b2, dict(a, q=a["q"][sel].copy()))
    assert np.array_equal(got, ref[sel])


def test_gqa_equals_replicated_mha():
    b, a = small_batch(seed=91, Hq=6, Hkv=2, D=8)
    ref, _, _, _, _ = oracle_run(b, a)
    G = 3
    k2 = np.repeat(a["k_cache"], G, axis=1)
    v2 = np.repeat(a["v_cache"], G, axis=1)
    b2 = wl.Batch(b.name, 6, 6, 8, b.reqs, b.num_pages, b.block_table, b.query_start_loc, b.ctx_lens, b.seed)
    got, _, _, _, _ = oracle_run(b2, dict(a, k_cache=k2, v_cache=v2))
    assert np.array_equal(got, ref)
    # equal q heads inside a group give equal outputs
    a3 = {k: v.copy() for k, v in a.items()}
    a3["q"][:, 1, :] = a3["q"][:, 0, :]
    a3["q"][:, 2, :] = a3["q"][:, 0, :]
    o3, _, _, _, _ = oracle_run(b, a3)
    assert np.array_equal(o3[:, 0], o3[:, 1]) and np.array_equal(o3[:, 0], o3[:, 2])
    assert not np.array_equal(o3[:, 0], o3[:, 3])


def test_unused_slots_never_read():
    b, _ = small_batch(seed=101)
    t = wl.make_tensors(b, "cpu")
    ref, _, _, _, _ = oracle_run(b, host_arrays(b, t))
    wl.poison_unused_slots(b, t.k_cache, t.v_cache)
    a = host_arrays(b, t)
    assert np.isnan(u16_to_f64(a["k_cache"])).any()
    got, _, _, _, _ = oracle_run(b, a)
    assert np.array_equal(got, ref)


# ---------------------------------------------------------------------------------------------
# 6. mask geometry vs the paper's Table 1 features (hand-computed golden values)
# ---------------------------------------------------------------------------------------------
def read_golden(name):
    vals = {}
    for line in (GOLDEN / name).read_text().splitlines():
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split("=")
            vals[k.strip()] = int(v)
    return vals


def test_tiny_features_and_visit_count_match_table1_by_hand():
    g = read_golden("tiny_table1_features.txt")
    b = wl.config_tiny()
    f = ft.features(b.reqs)
    for k in ("x1", "x2", "x3", "x4", "x5", "x6", "x7"):
        assert f[k] == g[k], k
    a = host_arrays(b, wl.make_tensors(b, "cpu"))
    _, _, pairs, _, _ = oracle_run(b, a)
    assert pairs == g["pairs"]
    # identity: pairs_P = x1 - x2/2 + x6/2 ; pairs_D = x5 + x4
    assert pairs == f["x1"] - f["x2"] // 2 + f["x6"] // 2 + f["x5"] + f["x4"]
    assert ft.scene(b.reqs) == "mixed"
    assert ft.scene([(1, 5), (0, 3)]) == "pure_decode" and ft.scene([(2, 0)]) == "pure_prefill"
    assert ft.split_sets([(0, 3), (1, 3), (2, 3)]) == ([0, 1], [2])
    assert ft.features([(1, 5)])["x7"] == 0


@pytest.mark.parametrize("seed", range(5))
def test_visit_count_identity_random(seed):
    b = wl.random_batch(200 + seed, Hq=2, Hkv=1, D=8, max_c=40, max_u=60, with_append=False)
    a = host_arrays(b, wl.make_tensors(b, "cpu"))
    _, _, pairs, _, _ = oracle_run(b, a)
    f = ft.features(b.reqs)
    n_c1 = sum(1 for c, _ in b.reqs if c == 1)
    u_c0 = sum(u for c, u in b.reqs if c == 0)
    # D in the paper includes c = 0 requests (Eq. 2: c_i <= 1); they contribute no visits
    assert pairs == f["x1"] - (f["x2"] - f["x6"]) // 2 + (f["x5"] - u_c0) + n_c1


# ---------------------------------------------------------------------------------------------
# 7. kv_append: exact
# ---------------------------------------------------------------------------------------------
def test_kv_append_touches_exactly_the_target_slots():
    b = wl.random_batch(301, Hq=4, Hkv=2, D=16, max_c=50, max_u=70)
    t = wl.make_tensors(b, "cpu")
    a = host_arrays(b, t)
    sent_k, sent_v = 0xABCD, 0x1234
    k = np.full_like(a["k_cache"], sent_k)
    v = np.full_like(a["v_cache"], sent_v)
    # special source bit patterns must survive: NaN payload, -0, denormal, inf
    a["k_new"].reshape(-1)[:4] = [0x7FC1, 0x8000, 0x0001, 0x7F80]
    a["v_new"].reshape(-1)[:4] = [0xFFC3, 0x8000, 0x8001, 0xFF80]
    oracle.kv_append(k, v, a["k_new"], a["v_new"], b.block_table, b.query_start_loc, b.ctx_lens)
    touched = 0
    for r, (c, u) in enumerate(b.reqs):
        for j in range(c):
            pos = u + j
            page, slot = int(b.block_table[r, pos // 16]), pos % 16
            tok = int(b.query_start_loc[r]) + j
            assert np.array_equal(k[page, :, slot, :], a["k_new"][tok])
            assert np.array_equal(v[page, :, slot, :], a["v_new"][tok])
            k[page, :, slot, :] = sent_k
            v[page, :, slot, :] = sent_v
            touched += 1
    assert touched == b.T
    assert np.all(k == sent_k) and np.all(v == sent_v)       # nothing else was written


def test_bf16_widening_matches_torch():
    bits = np.arange(0, 1 << 16, dtype=np.uint32).astype(np.uint16)
    finite = ~np.isnan(u16_to_f64(bits)) & ~np.isinf(u16_to_f64(bits))
    bits = bits[finite]
    # out = V[0] for a single key: feeds every finite bf16 pattern through the oracle's conversion
    n = bits.shape[0]
    D = 64
    pad = (-n) % D
    vals = np.concatenate([bits, np.zeros(pad, dtype=np.uint16)]).reshape(-1, 1, 1, D)
    R = vals.shape[0]
    k = np.zeros((R, 1, 16, D), dtype=np.uint16)
    v = np.zeros((R, 1, 16, D), dtype=np.uint16)
    v[:, :, 0:1, :] = vals
    bt = np.arange(R, dtype=np.int32).reshape(R, 1)
    qsl = np.arange(R + 1, dtype=np.int32)
    out, _, _ = oracle.mixed_attention(np.zeros((R, 1, D), dtype=np.uint16), k, v, bt, qsl,
                                       np.zeros(R, dtype=np.int32), 1.0)
    assert np.array_equal(out.reshape(-1)[:n], u16_to_f64(bits))
