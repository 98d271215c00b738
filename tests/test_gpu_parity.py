"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element on the same
seeded inputs.  Tolerances are north_star's: max-abs <= 2e-2, mean-abs <= 2e-3 (bf16 in, fp32 accumulate);
additionally a scale-aware per-request bound ||gpu - oracle||_2 / ||oracle||_2 <= 1e-2 (SURVEY.md §8(c):
the absolute tolerance alone is very loose at long context).  kv_append is compared bit for bit over the
whole pool."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_05933_b200 import binding, workloads as wl
from helpers import f64_to_u16, u16_to_f64

pytestmark = pytest.mark.gpu

MAX_ABS, MEAN_ABS, REL_L2 = 2e-2, 2e-3, 1e-2
DEV = "cuda:0"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def gpu_run(b, t, simple=False, lse=True, handle=None):
    h = handle or binding.handle_for(b, t)
    h.force_simple_path(simple)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    if b.with_append:
        binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx)
    lse_t = torch.full((max(b.T, 1), b.num_q_heads), float("nan"), dtype=torch.float32, device=DEV) if lse else None
    out = torch.full_like(t.q, float("nan"))
    binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=out, lse=lse_t)
    torch.cuda.synchronize()
    return out, lse_t, h


def oracle_run_from_device(b, t, k_before=None, v_before=None, rows=None):
    """Oracle on the same bits.  Uses compact_pool when the pool is large."""
    if k_before is None:
        k, v = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
        bt = b.block_table
    else:
        k, v, bt = k_before, v_before, b.block_table
    out, lse, pairs = oracle.mixed_attention(wl.to_u16(t.q), k, v, bt, b.query_start_loc, b.ctx_lens, b.scale, rows=rows)
    return out, lse


def check(b, out_gpu, ref, lse_gpu=None, lse_ref=None, rows=None):
    got = out_gpu.to(torch.float64).cpu().numpy()
    if rows is not None:
        got = got[rows]
    assert not np.isnan(got).any(), "NaN / unwritten rows in GPU output"
    err = np.abs(got - ref)
    assert err.max() <= MAX_ABS, f"max-abs {err.max():.3e}"
    assert err.mean() <= MEAN_ABS, f"mean-abs {err.mean():.3e}"
    if rows is None:
        for r, (c, u) in enumerate(b.reqs):
            if c == 0:
                continue
            s, e = int(b.query_start_loc[r]), int(b.query_start_loc[r + 1])
            rel = np.linalg.norm(got[s:e] - ref[s:e]) / max(np.linalg.norm(ref[s:e]), 1e-30)
            assert rel <= REL_L2, f"request {r} (c={c},u={u}) rel-L2 {rel:.3e}"
    else:
        rel = np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-30)
        assert rel <= REL_L2, f"sampled rows rel-L2 {rel:.3e}"
    if lse_gpu is not None and lse_ref is not None:
        lg = lse_gpu.to(torch.float64).cpu().numpy()
        if rows is not None:
            lg = lg[rows]
        assert np.abs(lg - lse_ref).max() <= 2e-2, f"lse max-abs {np.abs(lg - lse_ref).max():.3e}"
    return err.max(), err.mean()


def full_parity(b, poison=True, simple=False):
    t = wl.make_tensors(b, DEV, poison_unused=poison)
    k0, v0 = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    out, lse, h = gpu_run(b, t, simple=simple)
    if b.with_append:
        oracle.kv_append(k0, v0, wl.to_u16(t.k_new), wl.to_u16(t.v_new), b.block_table, b.query_start_loc, b.ctx_lens)
        assert np.array_equal(wl.to_u16(t.k_cache), k0), "k_cache differs from oracle after kv_append"
        assert np.array_equal(wl.to_u16(t.v_cache), v0), "v_cache differs from oracle after kv_append"
    ref, lse_ref, _ = oracle.mixed_attention(wl.to_u16(t.q), k0, v0, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    if b.T == 0:
        return 0.0, 0.0
    return check(b, out, ref, lse, lse_ref)


# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("simple", [False, True])
def test_c1_tiny(simple):
    full_parity(wl.config_tiny(), simple=simple)


@pytest.mark.parametrize("seed", range(6))
@pytest.mark.parametrize("shape", [(8, 2, 128), (4, 4, 64), (32, 8, 128), (16, 2, 128), (8, 8, 64),
                                   # head_dim 64 with a GQA group (staged Q copy, 16-row MMA padding, a5 merge at D = 64)
                                   (8, 4, 64), (16, 4, 64), (16, 2, 64), (32, 2, 64),
                                   # G = 7 (Qwen2.5-7B 28/4 and its TP2 slice 14/2), G = 4 TP2 slice of Llama-3-8B, odd G = 3, 5
                                   (28, 4, 128), (14, 2, 128), (16, 4, 128), (6, 2, 128), (10, 2, 64)])
def test_random_ragged_batches(seed, shape):
    Hq, Hkv, D = shape
    b = wl.random_batch(1000 + 17 * seed + Hq, Hq=Hq, Hkv=Hkv, D=D, n_prefill=3, n_decode=6, max_c=300, max_u=700)
    full_parity(b)


def test_simple_path_random():
    b = wl.random_batch(77, Hq=8, Hkv=2, D=128, n_prefill=2, n_decode=4, max_c=150, max_u=300)
    full_parity(b, simple=True)


def test_long_context_small_batch_exercises_split_kv():
    reqs = [(1, 9000), (1, 5), (1, 12345), (300, 4000), (1, 0), (1, 4095), (1, 4096), (1, 511), (1, 512)]
    b = wl.make_batch("long", 32, 8, 128, reqs, 91, with_append=True)
    full_parity(b)


def test_in_kernel_plan_and_two_launch_route_agree_bitwise():
    """Batches of <= 256 requests are planned inside the main kernel (one launch); larger ones, or debug knob 4, take
    the stand-alone work-list kernel first.  Same plan functions => bitwise identical outputs; repeated calls on one
    handle exercise the self-cleaning queue / arrival counters."""
    b = wl.random_batch(4242, Hq=32, Hkv=8, D=128, n_prefill=3, n_decode=40, max_c=400, max_u=5000)
    t = wl.make_tensors(b, DEV, poison_unused=True)
    k0, v0 = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    out1, lse1, h = gpu_run(b, t)
    assert h.last_launch_count() == 1
    out1b, _, _ = gpu_run(wl.Batch(**{**b.__dict__, "with_append": False}), t, handle=h)
    assert torch.equal(out1, out1b), "second call on the same handle differs (queue state not re-armed?)"
    h.debug_set_param(4, 1)
    out2, lse2, _ = gpu_run(wl.Batch(**{**b.__dict__, "with_append": False}), t, handle=h)
    assert h.last_launch_count() == 2
    h.debug_set_param(4, 0)
    assert torch.equal(out1, out2) and torch.equal(lse1, lse2)
    oracle.kv_append(k0, v0, wl.to_u16(t.k_new), wl.to_u16(t.v_new), b.block_table, b.query_start_loc, b.ctx_lens)
    ref, lse_ref, _ = oracle.mixed_attention(wl.to_u16(t.q), k0, v0, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    check(b, out2, ref, lse2, lse_ref)


def test_more_requests_than_the_in_kernel_plan_holds():
    rng = np.random.default_rng(5)
    reqs = [(1, int(u)) for u in rng.integers(0, 300, size=290)] + [(37, 100), (2, 0)]
    b = wl.make_batch("r292", 8, 2, 128, reqs, 93, with_append=True, shuffle_requests=True)
    t = wl.make_tensors(b, DEV, poison_unused=True)
    k0, v0 = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    out, lse, h = gpu_run(b, t)
    assert h.last_launch_count() == 2
    oracle.kv_append(k0, v0, wl.to_u16(t.k_new), wl.to_u16(t.v_new), b.block_table, b.query_start_loc, b.ctx_lens)
    ref, lse_ref, _ = oracle.mixed_attention(wl.to_u16(t.q), k0, v0, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    check(b, out, ref, lse, lse_ref)


def test_group16_shape():
    reqs = [(140, 50), (1, 2000), (1, 31), (1, 700)]
    b = wl.make_batch("g16", 32, 2, 128, reqs, 94, with_append=True)
    full_parity(b)


def test_70b_shape_group8():
    reqs = [(130, 77), (1, 3000), (1, 17), (2, 0), (1, 800)]
    b = wl.make_batch("g8", 64, 8, 128, reqs, 92, with_append=True)
    full_parity(b)


def test_empty_and_degenerate_batches():
    # R = 0 / T = 0: OK and nothing launched
    b = wl.make_batch("empty-req", 8, 2, 128, [(0, 5), (0, 0)], 93, with_append=True)
    t = wl.make_tensors(b, DEV)
    h = binding.handle_for(b, t)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    before = t.k_cache.clone()
    binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx)
    out = binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale)
    torch.cuda.synchronize()
    assert h.last_launch_count() == 0 and out.shape[0] == 0 and torch.equal(before, t.k_cache)
    # c = 0 requests interleaved with real ones
    full_parity(wl.make_batch("with-empty", 8, 2, 128, [(0, 9), (1, 0), (0, 0), (5, 0), (1, 33), (0, 700)], 94, with_append=True))


def test_single_cached_key_returns_v_exactly():
    b = wl.make_batch("one", 8, 2, 128, [(1, 0), (1, 0), (1, 0)], 95, with_append=True)
    t = wl.make_tensors(b, DEV, poison_unused=True)
    out, _, _ = gpu_run(b, t)
    G = 4
    for r in range(3):
        for hq in range(8):
            assert torch.equal(out[r, hq], t.v_new[r, hq // G]), (r, hq)


def test_needle_on_gpu():
    """One key aligned with q, all others orthogonal: out -> V[needle] when visible; a needle one past the
    causal limit must be invisible.  Pins mask off-by-one, page walk and split boundaries on the GPU."""
    D, Hq, Hkv = 128, 8, 2
    reqs = [(1, 700), (140, 300), (1, 5000)]
    b = wl.make_batch("needle", Hq, Hkv, D, reqs, 96)
    t = wl.make_tensors(b, "cpu")
    qdir = torch.zeros(D, dtype=torch.bfloat16)
    qdir[5] = 1.0
    kc, vc = t.k_cache.clone(), t.v_cache.clone()
    kc[..., 5] = 0
    kc *= 0.01
    cases = []      # (req, row j, needle pos)
    for r, (c, u) in enumerate(reqs):
        for j in sorted({0, c - 1}):
            vis = u + j + 1
            for pos in sorted({0, 15, 16, 127, 128, u - 1, u, vis - 1, vis} & set(range(c + u))):
                cases.append((r, j, pos))
    for r, j, pos in cases:
        c, u = reqs[r]
        k2 = kc.clone()
        page, slot = int(b.block_table[r, pos // 16]), pos % 16
        k2[page, :, slot, :] = 0
        k2[page, :, slot, 5] = 64.0
        q2 = t.q.clone()
        row = int(b.query_start_loc[r]) + j
        q2[row] = qdir
        t2 = wl.Tensors(q2.to(DEV), t.k_new.to(DEV), t.v_new.to(DEV), k2.to(DEV), vc.to(DEV))
        b2 = wl.Batch(b.name, Hq, Hkv, D, b.reqs, b.num_pages, b.block_table, b.query_start_loc, b.ctx_lens, b.seed)
        b2_scale = 1.0
        h = binding.handle_for(b2, t2)
        out = binding.mixed_attention(h, t2.q, dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens), b2_scale)
        torch.cuda.synchronize()
        got = out[row].to(torch.float64).cpu()
        if pos < u + j + 1:
            want = vc[page, :, slot, :].to(torch.float64).repeat_interleave(Hq // Hkv, dim=0)
            assert (got - want).abs().max() <= 1e-6, (r, j, pos)
        else:
            # invisible: scores all 0 -> prefix mean
            want = torch.stack([vc[int(b.block_table[r, p // 16]), :, p % 16, :] for p in range(u + j + 1)]
                               ).to(torch.float64).mean(0).repeat_interleave(Hq // Hkv, dim=0)
            assert (got - want).abs().max() <= 2e-2, (r, j, pos)
            assert (got - want).abs().mean() <= 2e-3, (r, j, pos)


@pytest.mark.parametrize("chunks", [(300,), (128, 128, 44), (1, 15, 16, 17, 251), (127, 129, 44), (299, 1)])
def test_chunking_invariance_on_gpu(chunks):
    """Prefill in any chunk sequence (append + attention per step) matches the oracle's unchunked rows."""
    L, Hq, Hkv, D = sum(chunks), 8, 2, 128
    full = wl.make_batch("full", Hq, Hkv, D, [(L, 0)], 97, num_pages=64, with_append=True)
    t = wl.make_tensors(full, DEV, poison_unused=False)
    k0, v0 = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    oracle.kv_append(k0, v0, wl.to_u16(t.k_new), wl.to_u16(t.v_new), full.block_table, full.query_start_loc, full.ctx_lens)
    ref, _, _ = oracle.mixed_attention(wl.to_u16(t.q), k0, v0, full.block_table, full.query_start_loc, full.ctx_lens, full.scale)
    h = binding.handle_for(full, t)
    bt = dev(full.block_table)
    outs, done = [], 0
    for c in chunks:
        qsl, ctx = dev(np.array([0, c], dtype=np.int32)), dev(np.array([done], dtype=np.int32))
        binding.kv_append(h, t.k_new[done:done + c], t.v_new[done:done + c], bt, qsl, ctx)
        outs.append(binding.mixed_attention(h, t.q[done:done + c], bt, qsl, ctx, full.scale))
        done += c
    torch.cuda.synchronize()
    assert np.array_equal(wl.to_u16(t.k_cache), k0) and np.array_equal(wl.to_u16(t.v_cache), v0)
    check(full, torch.cat(outs), ref)


def test_bitwise_reproducible_run_to_run():
    b = wl.random_batch(4242, Hq=32, Hkv=8, D=128, n_prefill=2, n_decode=8, max_c=260, max_u=3000, with_append=False)
    t = wl.make_tensors(b, DEV)
    o1, _, h = gpu_run(b, t)
    o2, _, _ = gpu_run(b, t, handle=h)
    assert torch.equal(o1, o2)


def test_kv_append_bit_exact_special_values():
    b = wl.random_batch(555, Hq=8, Hkv=4, D=128, n_prefill=3, n_decode=5, max_c=90, max_u=200)
    t = wl.make_tensors(b, DEV)
    bits = t.k_new.view(torch.int16)
    bits.view(-1)[:6] = torch.tensor([0x7FC1, -32768, 0x0001, 0x7F80, -64, -127], dtype=torch.int16, device=DEV)
    t.k_cache.view(torch.int16).fill_(0x2BCD)
    t.v_cache.view(torch.int16).fill_(0x1234)
    k0, v0 = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    h = binding.handle_for(b, t)
    binding.kv_append(h, t.k_new, t.v_new, dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens))
    torch.cuda.synchronize()
    oracle.kv_append(k0, v0, wl.to_u16(t.k_new), wl.to_u16(t.v_new), b.block_table, b.query_start_loc, b.ctx_lens)
    assert np.array_equal(wl.to_u16(t.k_cache), k0) and np.array_equal(wl.to_u16(t.v_cache), v0)
    assert int((k0 != 0x2BCD).sum()) <= b.T * 4 * 128


def test_worklist_partitions_the_batch():
    """a2: every (request, head) unit is covered exactly once, ranges tile [0, n) without gaps."""
    b = wl.config_c5(shuffle=True)
    t = wl.make_tensors(wl.make_batch("tinypool", 64, 8, 128, [(1, 0)], 1), DEV)
    h = binding.SlidingAttn(64, 8, 128, t.k_cache, t.v_cache, b.R, b.T, b.max_pages_per_req)
    items, (n_p, n_d, n_part) = h.build_worklist(dev(b.query_start_loc), dev(b.ctx_lens))
    assert len(items) == n_p + n_d
    pre, dec = items[:n_p], items[n_p:]
    assert (pre["kind"] == 1).all() and (dec["kind"] == 2).all()
    covered = np.zeros((b.T, 64), dtype=np.int32)
    for it in pre:
        c, u = b.reqs[it["req"]]
        assert c > 1 and it["kv_end"] == u + it["q_pos0"] + it["nrows"] and it["kv_begin"] == 0
        assert it["row0"] == b.query_start_loc[it["req"]] + it["q_pos0"] and 1 <= it["nrows"] <= 128
        assert it["nheads"] in (1, 2) and it["head"] // 8 == (it["head"] + it["nheads"] - 1) // 8    # one KV group
        covered[it["row0"]:it["row0"] + it["nrows"], it["head"]:it["head"] + it["nheads"]] += 1
    spans = {}
    for it in dec:
        c, u = b.reqs[it["req"]]
        assert c == 1 and it["row0"] == b.query_start_loc[it["req"]]
        assert it["kv_begin"] % 128 == 0 and it["kv_begin"] < it["kv_end"] <= u + 1
        spans.setdefault((int(it["req"]), int(it["head"])), []).append((int(it["kv_begin"]), int(it["kv_end"]), int(it["split"]), int(it["nsplit"]), int(it["partial"])))
    slots = set()
    for (r, g), sp in spans.items():
        sp.sort()
        u = b.reqs[r][1]
        assert sp[0][0] == 0 and sp[-1][1] == u + 1 and all(a[1] == bb[0] for a, bb in zip(sp, sp[1:]))
        assert [s[2] for s in sp] == list(range(len(sp))) and all(s[3] == len(sp) for s in sp)
        if len(sp) > 1:
            for s in sp:
                slot = s[4] + s[2]
                assert slot not in slots and 0 <= slot < n_part
                slots.add(slot)
        covered[b.query_start_loc[r], g * 8:(g + 1) * 8] += 1
    assert len(spans) == sum(1 for c, _ in b.reqs if c == 1) * 8
    assert len(slots) <= n_part          # partial slots share the decode items' index space
    assert (covered == 1).all()
    # heavy-first inside each kind: prefill requests by KV length (u + c), and inside a request the last (heaviest)
    # row tile first; the 32 head pairs of one (request, row tile) are consecutive
    first_head = pre[::32]
    assert (pre["head"].reshape(-1, 32) == 2 * np.arange(32)).all() and (pre["nheads"] == 2).all()
    req_order = list(dict.fromkeys(int(r) for r in first_head["req"]))
    kv_len = [b.reqs[r][0] + b.reqs[r][1] for r in req_order]
    assert kv_len == sorted(kv_len, reverse=True)
    for r in req_order:
        ends = first_head["kv_end"][first_head["req"] == r].astype(np.int64)
        assert (np.diff(ends) < 0).all()
    lens = (dec["kv_end"] - dec["kv_begin"]).astype(np.int64)
    first_of_req = lens[::8]
    assert first_of_req[0] == lens.max()


# ------------------------------------------------------------------------------------------------
# BASELINE.json configs at full size, in the launch configuration bench.py times
# ------------------------------------------------------------------------------------------------
def test_c2_full():
    full_parity(wl.config_c2(), poison=True)


def test_c2_shuffled_request_order():
    full_parity(wl.config_c2(shuffle=True), poison=False)


def sampled_parity(b, n_rows, seed, poison=False):
    t = wl.make_tensors(b, DEV, poison_unused=poison)
    out, lse, h = gpu_run(b, t)
    rng = np.random.default_rng(seed)
    # always include the longest-context rows and the last row of every prefill chunk
    order = np.argsort([-(c + u) for c, u in b.reqs])
    rows = set()
    for r in order[:4]:
        c = b.reqs[r][0]
        if c:
            rows.add(int(b.query_start_loc[r]) + c - 1)
    for r, (c, u) in enumerate(b.reqs):
        if c > 1:
            rows.update(int(b.query_start_loc[r]) + j for j in (0, c // 2, c - 1))
    rows.update(int(x) for x in rng.choice(b.T, size=min(n_rows, b.T), replace=False))
    rows = np.array(sorted(rows), dtype=np.int32)
    bt2, (k, v) = wl.compact_pool(b, t.k_cache, t.v_cache)
    ref, lse_ref, _ = oracle.mixed_attention(wl.to_u16(t.q), k, v, bt2, b.query_start_loc, b.ctx_lens, b.scale, rows=rows)
    assert not torch.isnan(out.float()).any()
    check(b, out, ref, lse, lse_ref, rows=rows)


def all_rows_parity_compacted(b):
    """Every output row against the oracle, for batches whose pool does not fit the host: the oracle runs on the
    pages the block table names (compact_pool; legal by the pinned page-permutation invariance)."""
    t = wl.make_tensors(b, DEV)
    out, lse, h = gpu_run(b, t)
    bt2, (k, v) = wl.compact_pool(b, t.k_cache, t.v_cache)
    ref, lse_ref, _ = oracle.mixed_attention(wl.to_u16(t.q), k, v, bt2, b.query_start_loc, b.ctx_lens, b.scale)
    check(b, out, ref, lse, lse_ref)


def test_c4_decode_heavy_full_pool_all_rows():
    """BASELINE.json configs[3]: 256 decodes over the 2 x 20 GB pool, every row checked (38 GFLOP of fp64)."""
    all_rows_parity_compacted(wl.config_c4())


def test_c5_70b_mixed_with_append_all_rows():
    """BASELINE.json configs[4] in bench.py's launch configuration: kv_append bit-exact over the whole pool, then all
    2240 rows (incl. the 30 136-key decode that takes 8 KV splits) against the oracle."""
    full_parity(wl.config_c5(), poison=False)


def test_c5_shuffled_request_order_poisoned():
    full_parity(wl.config_c5(shuffle=True), poison=True)


@pytest.mark.parametrize("C,n,N_d", [(256, 3, 32), (2048, 1, 32), (1024, 4, 128), (0, 1, 128)])
def test_c3_grid_points(C, n, N_d):
    full_parity(wl.config_c3(C, n, N_d), poison=False)


def test_scene_edge_pure_prefill_sampled():
    sampled_parity(wl.config_scene_edge("PP-d"), n_rows=64, seed=9)


@pytest.mark.parametrize("name", ["PP-b", "PP-f", "PP-q"])
def test_scene_edges_the_tensor_roofline_is_quoted_on_all_rows(name):
    """PP-b (2048 on 4096, 8B shape), PP-f (70B shape, G = 8 prefill), PP-q (Qwen shape, G = 7): every row."""
    full_parity(wl.config_scene_edge(name), poison=False)


def tile_edge_rows(b):
    """Rows 0, 127, 128, last, and the first/last row of every 128-row tile of every prefill chunk."""
    rows = set()
    for r, (c, u) in enumerate(b.reqs):
        s0 = int(b.query_start_loc[r])
        if c > 1:
            rows.update(s0 + j for j in range(0, c, 128))
            rows.update(s0 + min(j + 127, c - 1) for j in range(0, c, 128))
        elif c == 1:
            rows.add(s0)
    return rows


@pytest.mark.parametrize("name", ["PP-e", "PP-g"])
def test_scene_edges_many_row_tiles_sampled(name):
    """PP-e: 8192 rows = 64 row tiles; PP-g: 70B shape (4096, 4096).  Tile-edge rows forced + a random sample."""
    b = wl.config_scene_edge(name)
    t = wl.make_tensors(b, DEV)
    out, lse, h = gpu_run(b, t)
    rng = np.random.default_rng(11)
    rows = tile_edge_rows(b) | set(int(x) for x in rng.choice(b.T, size=96, replace=False))
    rows = np.array(sorted(rows), dtype=np.int32)
    ref, lse_ref, _ = oracle.mixed_attention(wl.to_u16(t.q), wl.to_u16(t.k_cache), wl.to_u16(t.v_cache), b.block_table,
                                             b.query_start_loc, b.ctx_lens, b.scale, rows=rows)
    assert not torch.isnan(out.float()).any()
    check(b, out, ref, lse, lse_ref, rows=rows)


@pytest.mark.parametrize("model", ["qwen2.5-7b", "qwen2.5-7b-tp2", "llama3-8b-tp2"])
def test_next3_model_shapes_mixed(model):
    """the Qwen2.5-7B layer (28/4/128, G = 7) and the TP2 per-GPU slices the paper ran
    (PAPER.md:382), C2's recipe, with append."""
    full_parity(wl.config_model_mixed(model), poison=True)
    full_parity(wl.config_model_mixed(model, shuffle=True), poison=False)


def test_batch_composition_invariance_on_gpu():
    """requests share a batch but are independent.  A prefill chunk and a decode of C2 run (i) inside C2
    and (ii) alone; both times the rows match the oracle's rows for that request (which the oracle pins bitwise
    against composition), and the two GPU results agree to within twice the tolerance."""
    b = wl.config_c2()
    t = wl.make_tensors(b, DEV)
    out_full, _, _ = gpu_run(b, t, lse=False)
    ref_full, _, _ = oracle.mixed_attention(wl.to_u16(t.q), wl.to_u16(t.k_cache), wl.to_u16(t.v_cache), b.block_table,
                                            b.query_start_loc, b.ctx_lens, b.scale)
    longest = int(np.argmax([u if c == 1 else -1 for c, u in b.reqs]))
    for r in (0, 1, longest, b.R - 1):
        c, u = b.reqs[r]
        s0 = int(b.query_start_loc[r])
        solo = wl.Batch(f"solo{r}", b.num_q_heads, b.num_kv_heads, b.head_dim, [(c, u)], b.num_pages,
                        np.ascontiguousarray(b.block_table[r:r + 1]), np.array([0, c], dtype=np.int32),
                        np.array([u], dtype=np.int32), b.seed)
        ts = wl.Tensors(t.q[s0:s0 + c].contiguous(), None, None, t.k_cache, t.v_cache)
        out_solo, _, _ = gpu_run(solo, ts, lse=False)
        ref = ref_full[s0:s0 + c]
        for got in (out_solo, out_full[s0:s0 + c]):
            err = np.abs(got.to(torch.float64).cpu().numpy() - ref)
            assert err.max() <= MAX_ABS and err.mean() <= MEAN_ABS
            assert np.linalg.norm(got.to(torch.float64).cpu().numpy() - ref) / np.linalg.norm(ref) <= REL_L2
        assert (out_solo.float() - out_full[s0:s0 + c].float()).abs().max().item() <= 2 * MAX_ABS


def test_scale_must_be_finite_and_positive():
    """slidingattn.h: scale <= 0 or non-finite is SS_ERR_INVALID_ARG (the kernels take the running max of raw scores).
    A tiny positive scale is the GPU twin of the oracle's scale = 0 closed form: every row -> prefix mean of V."""
    b = wl.random_batch(31, Hq=8, Hkv=2, D=128, n_prefill=2, n_decode=4, max_c=150, max_u=400, with_append=False)
    t = wl.make_tensors(b, DEV, poison_unused=True)
    h = binding.handle_for(b, t)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    for bad in (0.0, -0.125, float("nan"), float("inf"), -float("inf")):
        with pytest.raises(binding.SlidingAttnError) as ei:
            binding.mixed_attention(h, t.q, bt, qsl, ctx, bad)
        assert ei.value.status == binding.SS_ERR_INVALID_ARG
    out = binding.mixed_attention(h, t.q, bt, qsl, ctx, 1e-30)
    torch.cuda.synchronize()
    ref, _, _ = oracle.mixed_attention(wl.to_u16(t.q), wl.to_u16(t.k_cache), wl.to_u16(t.v_cache), b.block_table,
                                       b.query_start_loc, b.ctx_lens, 0.0)
    check(b, out, ref)


# ------------------------------------------------------------------------------------------------
# boundary: debug checks and handle reset
# ------------------------------------------------------------------------------------------------
def _poisoned_metadata_cases(b):
    bt, qsl, ctx = b.block_table.copy(), b.query_start_loc.copy(), b.ctx_lens.copy()
    r = next(i for i, (c, u) in enumerate(b.reqs) if c == 1 and u > 40)
    bad_page = bt.copy(); bad_page[r, 1] = b.num_pages + 7
    neg_page = bt.copy(); neg_page[r, 0] = -3
    bad_qsl = qsl.copy(); bad_qsl[2], bad_qsl[3] = bad_qsl[3] + 1, bad_qsl[2]
    bad_end = qsl.copy(); bad_end[-1] += 1
    too_long = ctx.copy(); too_long[r] = b.max_pages_per_req * 16 + 5
    neg_ctx = ctx.copy(); neg_ctx[r] = -1
    return {"page id >= num_pages": (bad_page, qsl, ctx, 4), "negative page id": (neg_page, qsl, ctx, 4),
            "qsl not monotone": (bt, bad_qsl, ctx, 1), "qsl[R] != T": (bt, bad_end, ctx, 1),
            "too many pages": (bt, qsl, too_long, 3), "negative ctx": (bt, qsl, neg_ctx, 2)}


def test_debug_checks_flag_bad_metadata_and_skip_the_access():
    b = wl.random_batch(77, Hq=8, Hkv=2, D=128, n_prefill=2, n_decode=6, max_c=200, max_u=500)
    t = wl.make_tensors(b, DEV)
    h = binding.handle_for(b, t, debug_checks=True)
    k_before, v_before = t.k_cache.clone(), t.v_cache.clone()
    for what, (bt_h, qsl_h, ctx_h, code) in _poisoned_metadata_cases(b).items():
        out = torch.full_like(t.q, 7.0)
        binding.kv_append(h, t.k_new, t.v_new, dev(bt_h), dev(qsl_h), dev(ctx_h))
        binding.mixed_attention(h, t.q, dev(bt_h), dev(qsl_h), dev(ctx_h), b.scale, out=out)
        with pytest.raises(binding.SlidingAttnError, match=f"device check {code}") as ei:
            h.poll_device_error()
        assert ei.value.status == binding.SS_ERR_DEVICE_CHECK, what
        assert torch.equal(t.k_cache, k_before) and torch.equal(t.v_cache, v_before), f"{what}: cache written"
        assert bool((out == 7.0).all()), f"{what}: out written"
        h.poll_device_error()                         # cleared: a second poll is clean
    # the same handle then serves a good batch, and matches the oracle
    k0, v0 = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    out, lse, _ = gpu_run(b, t, handle=h)
    h.poll_device_error()
    oracle.kv_append(k0, v0, wl.to_u16(t.k_new), wl.to_u16(t.v_new), b.block_table, b.query_start_loc, b.ctx_lens)
    assert np.array_equal(wl.to_u16(t.k_cache), k0) and np.array_equal(wl.to_u16(t.v_cache), v0)
    ref, lse_ref, _ = oracle.mixed_attention(wl.to_u16(t.q), k0, v0, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    check(b, out, ref, lse, lse_ref)
    assert h.last_launch_count() == 2                 # validate + main launch


@pytest.mark.parametrize("route", ["more requests than the in-kernel plan holds", "knob 4", "simple path"])
def test_debug_checks_cover_the_two_launch_route_and_the_simple_path(route):
    """the stand-alone work-list kernel and the warp-per-row kernel must also stand still after a tripped
    check (a negative ctx_len would otherwise divide by zero in the plan / walk a bad page id), the launch count
    includes the validate launch on every route, and the handle serves a good batch afterwards."""
    if route == "more requests than the in-kernel plan holds":
        reqs = [(1, 40 + 3 * i) for i in range(280)] + [(70, 100), (1, 2000)]
    else:
        reqs = [(1, 900), (130, 64), (1, 0), (1, 3000), (40, 0)]
    b = wl.make_batch("dbg-routes", 8, 2, 128, reqs, 93, with_append=False)
    t = wl.make_tensors(b, DEV)
    h = binding.handle_for(b, t, debug_checks=True)
    if route == "knob 4":
        h.debug_set_param(4, 1)
    h.force_simple_path(route == "simple path")
    bt, qsl = dev(b.block_table), dev(b.query_start_loc)
    neg_ctx = b.ctx_lens.copy()
    neg_ctx[1] = -5
    bad_bt = b.block_table.copy()
    bad_bt[3, 0] = b.num_pages + 7
    for ctx_h, bt_h, code in ((neg_ctx, b.block_table, 2), (b.ctx_lens, bad_bt, 4)):
        out = torch.full_like(t.q, 7.0)
        binding.mixed_attention(h, t.q, dev(bt_h), qsl, dev(ctx_h), b.scale, out=out)
        with pytest.raises(binding.SlidingAttnError, match=f"device check {code}"):
            h.poll_device_error()
        assert bool((out == 7.0).all()), "out written after a tripped check"
    out = torch.full_like(t.q, float("nan"))
    binding.mixed_attention(h, t.q, bt, qsl, dev(b.ctx_lens), b.scale, out=out)
    h.poll_device_error()
    assert h.last_launch_count() == (2 if route == "simple path" else 3)    # validate (+ work list) + attention
    ref, _ = oracle_run_from_device(b, t)
    check(b, out, ref)


@pytest.mark.parametrize("two_launch", [False, True])
def test_forced_short_split_never_outgrows_the_workspace(two_launch):
    """the workspace's partial slots are sized for the automatic split length.  Forcing 512-key splits on a
    few very long contexts asks for ~10x more items than there are slots; the plan must raise the length until they
    fit instead of writing past the workspace.  A guard buffer right behind the workspace must stay untouched and the
    result must not depend on the knob."""
    reqs = [(1, 60000), (1, 52345), (1, 7), (1, 33000), (150, 20000)]
    b = wl.make_batch("forced-L", 32, 8, 128, reqs, 94, with_append=False)
    t = wl.make_tensors(b, DEV)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    h = binding.handle_for(b, t)
    ref_out = binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale).clone()
    # the handle's workspace, re-seated at the front of a larger buffer whose tail is the guard
    guard_bytes = 8 << 20
    big = torch.full((h.workspace_bytes + guard_bytes,), 0x5A, dtype=torch.uint8, device=DEV)
    h.workspace = big
    h.debug_set_param(3, 512)
    if two_launch:
        h.debug_set_param(4, 1)
    out = binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=torch.full_like(t.q, float("nan")))
    torch.cuda.synchronize()
    assert bool((big[h.workspace_bytes:] == 0x5A).all()), "wrote past the workspace"
    items, counts = h.build_worklist(qsl, ctx)
    splits = items[items["kind"] == 2]
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    slots = 8 * b.R * (-(-b.max_pages_per_req * 16 // 16384) + 1) + sms + 64          # workspace_layout's max_partials
    assert 8 * 512 * 8 * len(splits) > 145000 * 8, "the forced length was not honoured at all"
    assert len(splits) > 5 * 8 and counts[2] <= slots                                 # still split, and inside the slots
    assert bool((big[h.workspace_bytes:] == 0x5A).all())
    g, r = out.to(torch.float64).cpu().numpy(), ref_out.to(torch.float64).cpu().numpy()
    assert not np.isnan(g).any()
    assert np.abs(g - r).max() <= MAX_ABS and np.abs(g - r).mean() <= MEAN_ABS
    rows = np.asarray([0, 1, 3, 4, 153], dtype=np.int32)
    ref, _ = oracle_run_from_device(b, t, rows=rows)
    check(b, out, ref, rows=rows)


def test_poll_is_clean_without_debug_checks_and_reset_rearms_the_handle():
    b = wl.random_batch(78, Hq=8, Hkv=2, D=128, n_prefill=1, n_decode=5, max_c=100, max_u=3000, with_append=False)
    t = wl.make_tensors(b, DEV)
    out1, _, h = gpu_run(b, t, lse=False)
    h.poll_device_error()
    h.reset()
    out2, _, _ = gpu_run(b, t, lse=False, handle=h)
    assert torch.equal(out1, out2)


def test_iteration_host_matches_device_path():
    b = wl.config_tiny()
    t = wl.make_tensors(b, DEV)
    t_host = wl.Tensors(*[x.cpu().pin_memory() for x in (t.q, t.k_new, t.v_new)], None, None)
    kc, vc = t.k_cache.clone(), t.v_cache.clone()
    out_dev, _, h = gpu_run(b, t, lse=False)
    h2 = binding.SlidingAttn(b.num_q_heads, b.num_kv_heads, b.head_dim, kc, vc, b.R, b.T, b.max_pages_per_req)
    out_host = torch.empty_like(t_host.q).pin_memory()
    h2.iteration_host(t_host.q, t_host.k_new, t_host.v_new, torch.from_numpy(b.block_table), torch.from_numpy(b.query_start_loc),
                      torch.from_numpy(b.ctx_lens), b.scale, out_host)
    assert torch.equal(out_host, out_dev.cpu()) and torch.equal(kc, t.k_cache)


def test_append_plus_attention_is_cuda_graph_capturable():
    """One iteration (a1 + a2..a5, programmatic dependent launch between them) captured into a CUDA graph and replayed:
    nothing on the hot path touches the host besides encoding the Q tensor map from its (fixed) pointer.  The replay
    must reproduce the eager result bit for bit, also after the inputs changed in place."""
    b = wl.config_c3(256, 2, 32)
    b = wl.Batch(**{**b.__dict__, "with_append": True})
    t = wl.make_tensors(b, DEV)
    h = binding.handle_for(b, t)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    out_eager = torch.empty_like(t.q)
    binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx)
    binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=out_eager)
    torch.cuda.synchronize()
    out_graph = torch.zeros_like(t.q)
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx, stream=s)       # warm-up on the capture stream
        binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=out_graph, stream=s)
        s.synchronize()
        with torch.cuda.graph(g, stream=s):
            binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx, stream=s)
            binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=out_graph, stream=s)
    out_graph.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out_graph, out_eager)
    t.q.mul_(-1.0)                                                   # new inputs, same pointers: replay follows them
    binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=out_eager)
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(out_graph, out_eager)
