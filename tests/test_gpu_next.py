"""GPU parity of the "next" rows: RoPE + QKV split fused into the append (NEXT-4) and the FP8 E4M3 KV
cache variant of a1 / a4 (NEXT-3), through the C ABI, against oracle/next_oracle.c on the same seeded inputs.

Tolerances.  V (a bit copy) and the FP8 codes (an integer decision taken in fp32 on both sides) are compared bit for
bit.  Rotated q / k: the kernel rotates in fp32 with cos / sin rounded from double, the oracle in double; both round
once to bf16, so they may differ by one bf16 ulp where the exact value sits within ~1e-7 (relative) of a rounding
tie, and where the two products nearly cancel the fp32 rotation carries an absolute error of a few 2^-24 |x| (|x| <= ~6
for N(0,1) inputs): every element within one bf16 ulp + 3e-6, and fewer than 0.2 % of them different at all.  Attention outputs: north_star's
max-abs <= 2e-2 / mean-abs <= 2e-3 plus the per-request relative L2 <= 1e-2 (FP8: inputs are the SAME codes on both
sides, so the bound is the bf16 path's)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_05933_b200 import binding, workloads as wl
from helpers import u16_to_f64

pytestmark = pytest.mark.gpu

MAX_ABS, MEAN_ABS, REL_L2 = 2e-2, 2e-3, 1e-2
DEV = "cuda:0"
THETA = {"llama3": 500000.0, "qwen2.5": 1000000.0}


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def assert_same_bf16_bits(got_u16, want_u16, what):
    """Round 3: the fused RoPE rotates in double with separately rounded products and one rounding to bf16 - the
    oracle's arithmetic (reading 25) - so the comparison is bit for bit, unused (poisoned) slots included.
    Only cos / sin come from another libm; their last-ulp differences can flip a bf16 rounding with probability
    ~2^-44 per element."""
    bad = got_u16 != want_u16
    assert not bad.any(), (f"{what}: {int(bad.sum())} of {bad.size} elements differ from the oracle, first at "
                           f"{tuple(int(i) for i in np.argwhere(bad)[0])}")


def check_attention(b, out_gpu, ref):
    got = out_gpu.to(torch.float64).cpu().numpy()
    assert not np.isnan(got).any()
    err = np.abs(got - ref)
    assert err.max() <= MAX_ABS and err.mean() <= MEAN_ABS, (err.max(), err.mean())
    for r, (c, u) in enumerate(b.reqs):
        if c:
            s, e = int(b.query_start_loc[r]), int(b.query_start_loc[r + 1])
            rel = np.linalg.norm(got[s:e] - ref[s:e]) / max(np.linalg.norm(ref[s:e]), 1e-30)
            assert rel <= REL_L2, f"request {r} (c={c},u={u}) rel-L2 {rel:.3e}"


# ------------------------------------------------------------------------------------------------------------------
# NEXT-4: RoPE + QKV split fused into the append
# ------------------------------------------------------------------------------------------------------------------
def rope_case(b, theta):
    t = wl.make_tensors(b, DEV, poison_unused=True)
    qkv = torch.cat([t.q.reshape(b.T, -1), t.k_new.reshape(b.T, -1), t.v_new.reshape(b.T, -1)], dim=1).contiguous()
    k0, v0 = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    h = binding.handle_for(b, t)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    q_rot = h.qkv_rope_append(qkv, bt, qsl, ctx, theta)
    out = binding.mixed_attention(h, q_rot, bt, qsl, ctx, b.scale)
    torch.cuda.synchronize()
    q_ref = oracle.rope_qkv_append(wl.to_u16(qkv), k0, v0, b.block_table, b.query_start_loc, b.ctx_lens, b.num_q_heads, theta)
    assert np.array_equal(wl.to_u16(t.v_cache), v0), "v_cache: the fused append must copy V bit for bit"
    assert_same_bf16_bits(wl.to_u16(q_rot), q_ref, "rotated q")
    assert_same_bf16_bits(wl.to_u16(t.k_cache), k0, "k_cache (rotated k; untouched slots identical)")
    ref, _, _ = oracle.mixed_attention(q_ref, k0, v0, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    if b.T:
        check_attention(b, out, ref)
    return h


@pytest.mark.parametrize("shape,model", [((8, 2, 128), "llama3"), ((28, 4, 128), "qwen2.5"), ((4, 4, 64), "llama3"),
                                         ((16, 4, 64), "qwen2.5"), ((64, 8, 128), "llama3")])
def test_rope_qkv_append_random_batches(shape, model):
    Hq, Hkv, D = shape
    for seed in (0, 1):
        b = wl.random_batch(3100 + 7 * seed + Hq, Hq=Hq, Hkv=Hkv, D=D, n_prefill=2, n_decode=5, max_c=200, max_u=900)
        rope_case(b, THETA[model])


def test_rope_long_positions_and_c2():
    """Positions up to 30 000 (cos / sin range reduction) and BASELINE.json configs[1] with the fused append."""
    reqs = [(1, 29999), (130, 20000), (1, 12345), (1, 0), (17, 0)]
    rope_case(wl.make_batch("rope-long", 32, 8, 128, reqs, 41, with_append=True), THETA["llama3"])
    b = wl.config_c2()
    rope_case(wl.Batch(**{**b.__dict__, "with_append": True}), THETA["llama3"])


def test_rope_position_zero_is_a_bit_copy():
    b = wl.make_batch("p0", 8, 2, 128, [(1, 0), (1, 0), (1, 0)], 42, with_append=True)
    t = wl.make_tensors(b, DEV)
    qkv = torch.cat([t.q.reshape(b.T, -1), t.k_new.reshape(b.T, -1), t.v_new.reshape(b.T, -1)], dim=1).contiguous()
    h = binding.handle_for(b, t)
    kp, vp = t.k_cache.clone(), t.v_cache.clone()
    q_rot = h.qkv_rope_append(qkv, dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens), 10000.0)
    h2 = binding.SlidingAttn(8, 2, 128, kp, vp, b.R, b.T, b.max_pages_per_req)
    binding.kv_append(h2, t.k_new, t.v_new, dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens))
    torch.cuda.synchronize()
    assert torch.equal(q_rot, t.q) and torch.equal(t.k_cache, kp) and torch.equal(t.v_cache, vp)


def test_rope_theta_must_be_finite_and_above_one():
    b = wl.make_batch("bad", 8, 2, 128, [(1, 5)], 43, with_append=True)
    t = wl.make_tensors(b, DEV)
    qkv = torch.zeros(1, 12 * 128, dtype=torch.bfloat16, device=DEV)
    h = binding.handle_for(b, t)
    for bad in (0.0, 1.0, -5.0, float("nan"), float("inf")):
        with pytest.raises(binding.SlidingAttnError) as ei:
            h.qkv_rope_append(qkv, dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens), bad)
        assert ei.value.status == binding.SS_ERR_INVALID_ARG


# ------------------------------------------------------------------------------------------------------------------
# NEXT-3: FP8 E4M3 KV cache (a1 quantising append, a4 decode over FP8 tiles, a3 prefill on fp16 copies of the FP8 tiles)
# ------------------------------------------------------------------------------------------------------------------
def fp8_scales(Hkv, seed):
    rng = np.random.default_rng(seed)
    return (rng.uniform(0.008, 0.02, size=Hkv).astype(np.float32), rng.uniform(0.008, 0.02, size=Hkv).astype(np.float32))


def quantise_pool(cache_bf16, scale):
    """Initial cache contents (an INPUT of the test, any codes would do): the N(0,1) pool quantised with torch, poisoned
    unused slots (bf16 NaN) become E4M3 NaN codes."""
    s = torch.from_numpy(scale).to(cache_bf16.device).view(1, -1, 1, 1)
    return (cache_bf16.float() / s).clamp(-448.0, 448.0).to(torch.float8_e4m3fn).view(torch.uint8).contiguous()


def fp8_case(b, seed=0, check_rows=None):
    t = wl.make_tensors(b, DEV, poison_unused=True)
    ks, vs = fp8_scales(b.num_kv_heads, 500 + seed)
    kc, vc = quantise_pool(t.k_cache, ks), quantise_pool(t.v_cache, vs)
    k0, v0 = kc.cpu().numpy().copy(), vc.cpu().numpy().copy()
    h = binding.handle_for(b, t, fp8_caches=(kc, vc), kv_scales=(dev(ks), dev(vs)))
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    if b.with_append:
        binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx)
        oracle.kv_append_fp8(k0, v0, wl.to_u16(t.k_new), wl.to_u16(t.v_new), ks, vs, b.block_table, b.query_start_loc, b.ctx_lens)
    out = binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale)
    torch.cuda.synchronize()
    if b.with_append:
        assert np.array_equal(kc.cpu().numpy(), k0), "FP8 k_cache codes differ from the oracle's"
        assert np.array_equal(vc.cpu().numpy(), v0), "FP8 v_cache codes differ from the oracle's"
    rows = None if check_rows is None else np.asarray(check_rows, dtype=np.int32)
    ref, _ = oracle.mixed_attention_fp8(wl.to_u16(t.q), k0, v0, ks, vs, b.block_table, b.query_start_loc, b.ctx_lens, b.scale, rows=rows)
    if rows is None:
        check_attention(b, out, ref)
    else:
        got = out.to(torch.float64).cpu().numpy()
        assert not np.isnan(got).any()
        err = np.abs(got[rows] - ref)
        assert err.max() <= MAX_ABS and err.mean() <= MEAN_ABS, (err.max(), err.mean())
        rel = np.linalg.norm(got[rows] - ref, axis=(1, 2)) / np.maximum(np.linalg.norm(ref, axis=(1, 2)), 1e-30)
        assert rel.max() <= REL_L2, rel.max()
    return h


def test_fp8_append_every_bf16_pattern():
    """Quantisation decision on every bf16 input (NaN payloads, +-inf, denormals, -0, ties) at several scales: bit-exact."""
    Hkv, D = 2, 128
    pats = np.arange(65536, dtype=np.uint16)
    T = 65536 // (Hkv * D)
    b = wl.make_batch("fp8-all", 4, Hkv, D, [(T, 5)], 77, with_append=True)
    t = wl.make_tensors(b, DEV)
    k_new = torch.from_numpy(pats.view(np.int16).reshape(T, Hkv, D).copy()).to(DEV).view(torch.bfloat16)
    v_new = torch.from_numpy(np.roll(pats, 12345).view(np.int16).reshape(T, Hkv, D).copy()).to(DEV).view(torch.bfloat16)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    for scales in ([1.0, 0.0123], [3.7, 2.0 ** -10], [1e-3, 448.0], [0.3333333, 1e-30]):
        ks, vs = np.asarray(scales, dtype=np.float32), np.asarray(scales[::-1], dtype=np.float32)
        kc = torch.full(t.k_cache.shape, 0x55, dtype=torch.uint8, device=DEV)
        vc = torch.full(t.v_cache.shape, 0xAA, dtype=torch.uint8, device=DEV)
        k0, v0 = kc.cpu().numpy().copy(), vc.cpu().numpy().copy()
        h = binding.handle_for(b, t, fp8_caches=(kc, vc), kv_scales=(dev(ks), dev(vs)))
        binding.kv_append(h, k_new, v_new, bt, qsl, ctx)
        torch.cuda.synchronize()
        oracle.kv_append_fp8(k0, v0, wl.to_u16(k_new), wl.to_u16(v_new), ks, vs, b.block_table, b.query_start_loc, b.ctx_lens)
        assert np.array_equal(kc.cpu().numpy(), k0) and np.array_equal(vc.cpu().numpy(), v0), f"scales {scales}"


@pytest.mark.parametrize("shape", [(8, 2, 128), (28, 4, 128), (32, 8, 128), (64, 8, 128), (16, 1, 128), (4, 4, 128)])
def test_fp8_random_mixed_batches(shape):
    Hq, Hkv, D = shape
    for seed in (0, 1):
        b = wl.random_batch(4100 + 11 * seed + Hq, Hq=Hq, Hkv=Hkv, D=D, n_prefill=2, n_decode=9, max_c=150, max_u=1500)
        fp8_case(wl.Batch(**{**b.__dict__, "with_append": True}), seed)


def test_fp8_decode_long_contexts_and_splits():
    """Split-KV over FP8 tiles: contexts to 12 345 keys (several splits), ragged tails, a single cached key."""
    reqs = [(1, 12345), (1, 4095), (1, 4096), (1, 63), (1, 64), (1, 65), (1, 0), (1, 1), (1, 15), (1, 16), (1, 8191), (1, 777)]
    fp8_case(wl.make_batch("fp8-long", 32, 8, 128, reqs, 78, with_append=True))
    fp8_case(wl.make_batch("fp8-long-g8", 64, 8, 128, reqs, 79, with_append=True), 1)


def test_fp8_pure_decode_batch_all_rows():
    b = wl.config_c3(0, 1, 128)                          # PD-128: 128 decodes, lognormal contexts
    fp8_case(wl.Batch(**{**b.__dict__, "with_append": True}))


def test_fp8_needs_scales_and_head_dim_128():
    b = wl.make_batch("fp8-bad", 8, 2, 128, [(1, 5)], 80, with_append=True)
    t = wl.make_tensors(b, DEV)
    kc = torch.zeros(t.k_cache.shape, dtype=torch.uint8, device=DEV)
    h = binding.handle_for(b, t, fp8_caches=(kc, kc.clone()))
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    with pytest.raises(binding.SlidingAttnError) as ei:
        binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx)
    assert ei.value.status == binding.SS_ERR_INVALID_ARG
    with pytest.raises(binding.SlidingAttnError) as ei:
        binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale)
    assert ei.value.status == binding.SS_ERR_INVALID_ARG
    b64 = wl.config_tiny()
    t64 = wl.make_tensors(b64, DEV)
    kc64 = torch.zeros(t64.k_cache.shape, dtype=torch.uint8, device=DEV)
    with pytest.raises(binding.SlidingAttnError) as ei:
        binding.handle_for(b64, t64, fp8_caches=(kc64, kc64.clone()))
    assert ei.value.status == binding.SS_ERR_INVALID_ARG


def test_fp8_debug_checks_catch_bad_scales():
    """the header says every FP8 scale is finite and > 0; with SS_FLAG_DEBUG_CHECKS the device check now
    enforces it (a zero or negative k_scale breaks the running max of the raw scores silently)."""
    b = wl.make_batch("fp8-scales", 8, 2, 128, [(1, 300), (40, 10)], 81, with_append=True)
    t = wl.make_tensors(b, DEV)
    ks, vs = fp8_scales(2, 7)
    kc, vc = quantise_pool(t.k_cache, ks), quantise_pool(t.v_cache, vs)
    k_dev, v_dev = dev(ks), dev(vs)
    h = binding.handle_for(b, t, fp8_caches=(kc, vc), kv_scales=(k_dev, v_dev), debug_checks=True)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    kc0 = kc.clone()
    for which, idx, bad in ((k_dev, 1, 0.0), (k_dev, 0, -0.01), (v_dev, 1, float("nan")), (v_dev, 0, float("inf"))):
        good = float(which[idx])
        which[idx] = bad
        out = torch.full_like(t.q, 7.0)
        binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx)
        binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=out)
        with pytest.raises(binding.SlidingAttnError, match="device check 5") as ei:
            h.poll_device_error()
        assert f"request {idx + (2 if which is v_dev else 0)}," in str(ei.value)
        assert torch.equal(kc, kc0) and bool((out == 7.0).all())
        which[idx] = good
    binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx)
    out = binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=torch.full_like(t.q, float("nan")))
    h.poll_device_error()
    assert not torch.isnan(out.float()).any() and not torch.equal(kc, kc0)


def test_fp8_bitwise_reproducible_whatever_ran_before():
    """The split of an item's keys between the decode warpgroups must not depend on the CTA's history (dynamic queue):
    repeated calls, and the same batch after a different batch on the same handle, give identical bits."""
    b = wl.config_c3(0, 1, 128)
    t = wl.make_tensors(b, DEV, caches=False)
    kc, vc, ks, vs = wl.make_fp8_caches(b, DEV)
    h = binding.handle_for(b, t, fp8_caches=(kc, vc), kv_scales=(ks, vs))
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    outs = [binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale).clone() for _ in range(4)]
    ctx2 = torch.clamp(ctx - 37, min=0)                       # another batch in between: other tile counts per item
    binding.mixed_attention(h, t.q, bt, qsl, ctx2, b.scale)
    outs.append(binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale).clone())
    torch.cuda.synchronize()
    assert all(torch.equal(outs[0], o) for o in outs[1:])


def test_fp8_two_launch_route_more_requests_than_the_in_kernel_plan_holds():
    """R > 256: the stand-alone work-list kernel plans the batch (single-head prefill items) and the FP8 main kernel
    reads its items."""
    rng = np.random.default_rng(81)
    reqs = [(1, int(u)) for u in rng.integers(1, 700, size=290)] + [(37, 100), (2, 0)]
    b = wl.make_batch("fp8-r292", 8, 2, 128, reqs, 82, with_append=True)
    h = fp8_case(b)
    assert h.last_launch_count() == 2                        # work list + main


def _edge_rows(b, per_req=24, seed=0):
    """Rows worth checking one by one: first / last of every request and of every 128-row tile, plus a random share."""
    rng = np.random.default_rng(seed)
    rows = set()
    for r, (c, u) in enumerate(b.reqs):
        s = int(b.query_start_loc[r])
        for j in {0, c - 1, *range(127, c, 128), *range(128, c, 128), *(int(x) for x in rng.integers(0, max(c, 1), size=min(per_req, c)))}:
            if 0 <= j < c:
                rows.add(s + j)
    return sorted(rows)


@pytest.mark.parametrize("reqs,shape", [
    ([(300, 0), (1, 77)], (8, 2, 128)),                       # 3 row tiles, odd and even ring-tile counts (padding tile)
    ([(128, 128), (129, 63), (127, 1), (2, 0), (1, 500)], (32, 8, 128)),
    ([(65, 4031), (64, 64), (1, 4095)], (28, 4, 128)),        # G = 7: odd group, single-head items
    ([(2048, 4096)], (32, 8, 128)),                           # PP-b
    ([(1024, 0), (1024, 6000), (1, 3000), (1, 9000)], (64, 8, 128)),   # 70B shape, PP-f + decodes
    ([(700, 300), (300, 0), (1, 2000), (1, 17)], (28, 4, 128)),        # G = 7 with head pairs: 3 pair items + 1 single-head item per kv head
    ([(640, 0), (1, 100)], (6, 2, 128)),                               # G = 3, too few items to pair: single-head items only
])
def test_fp8_prefill_on_tensor_cores(reqs, shape):
    """Prefill chunks over the FP8 cache: tcgen05 on fp16 copies of the staged tiles (converter warpgroup); single-head items
    while one wave of CTAs holds them all, head pairs (two chains on one converted tile) from the second wave on."""
    Hq, Hkv, D = shape
    b = wl.make_batch("fp8-prefill", Hq, Hkv, D, reqs, 90 + len(reqs), with_append=True)
    fp8_case(b, seed=len(reqs), check_rows=_edge_rows(b) if b.T > 700 else None)


@pytest.mark.parametrize("fp8", [False, True])
def test_single_head_item_as_long_as_the_ring_then_a_pair_item(fp8):
    """G = 7, forty 128-row chunks whose items cover exactly as many ring tiles as the ring has slots (5 over the bf16 cache;
    5 + the padding tile = 6 over the FP8 cache): chain B sits out every fourth item and then takes a pair item whose
    first tile reuses the slot of the skipped item's first tile - its issuer must have seen every Q phase for the parity
    waits on the ring to be exact (a race the build before the fix did not lose on this batch either: the test pins the
    shape, the argument is in attn_mixed.cu).  Five launches, all rows against the oracle."""
    rng = np.random.default_rng(4242)
    reqs = [(128, int(u)) for u in rng.integers(130, 192, size=40, endpoint=True)] + [(1, 300), (1, 5000)]
    b = wl.make_batch("single-then-pair", 28, 4, 128, reqs, 4242, with_append=True)
    if fp8:
        fp8_case(b, seed=42)
        return
    t = wl.make_tensors(b, DEV, poison_unused=True)
    k0, v0 = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    h = binding.handle_for(b, t)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx)
    outs = [binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale).clone() for _ in range(5)]
    torch.cuda.synchronize()
    oracle.kv_append(k0, v0, wl.to_u16(t.k_new), wl.to_u16(t.v_new), b.block_table, b.query_start_loc, b.ctx_lens)
    ref, _, _ = oracle.mixed_attention(wl.to_u16(t.q), k0, v0, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    for out in outs:
        check_attention(b, out, ref)


def test_randomized_shapes_and_mixes_bf16_and_fp8():
    """48 seeded random batches over ten layer shapes (G = 1, 2, 3, 4, 7, 8, 16; head_dim 64 and 128), 0-3 prefill chunks and
    0-39 decodes of random lengths each, alternately over the bf16 and the FP8 cache: append bit-exact, every row against
    the fp64 oracle."""
    shapes = [(8, 2, 128), (32, 8, 128), (28, 4, 128), (64, 8, 128), (16, 1, 128), (4, 4, 64), (16, 4, 64), (8, 8, 64),
              (14, 2, 128), (12, 4, 128)]
    rng = np.random.default_rng(12345)
    for it in range(48):
        Hq, Hkv, D = shapes[it % len(shapes)]
        npf, nd = int(rng.integers(0, 4)), int(rng.integers(0, 40))
        nd = max(nd, 1 if npf == 0 else 0)
        b = wl.random_batch(70000 + it, Hq=Hq, Hkv=Hkv, D=D, n_prefill=npf, n_decode=nd, max_c=int(rng.integers(2, 400)),
                            max_u=int(rng.integers(1, 5000)))
        b = wl.Batch(**{**b.__dict__, "with_append": True})
        if D == 128 and it % 2 == 1:
            fp8_case(b, seed=it)
            continue
        t = wl.make_tensors(b, DEV, poison_unused=True)
        k0, v0 = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
        h = binding.handle_for(b, t)
        bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
        binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx)
        out = binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale)
        torch.cuda.synchronize()
        oracle.kv_append(k0, v0, wl.to_u16(t.k_new), wl.to_u16(t.v_new), b.block_table, b.query_start_loc, b.ctx_lens)
        assert np.array_equal(wl.to_u16(t.k_cache), k0) and np.array_equal(wl.to_u16(t.v_cache), v0)
        ref, _, _ = oracle.mixed_attention(wl.to_u16(t.q), k0, v0, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
        check_attention(b, out, ref)


@pytest.mark.parametrize("shape,model", [((8, 2, 128), "llama3"), ((28, 4, 128), "qwen2.5"), ((64, 8, 128), "llama3")])
def test_fp8_rope_qkv_append(shape, model):
    """Fused RoPE + QKV split over an FP8 cache: q as on a bf16 handle; k rotated and rounded to bf16 once, THEN quantised
    like ss_kv_append; v quantised.  Oracle = its RoPE append into scratch bf16 caches, then its FP8 append of those bits.
    q, K codes and V codes bit-exact (round 3: the rotation is the oracle's double arithmetic, so the bf16 value that
    gets quantised is the oracle's)."""
    Hq, Hkv, D = shape
    b = wl.random_batch(5100 + Hq, Hq=Hq, Hkv=Hkv, D=D, n_prefill=2, n_decode=6, max_c=180, max_u=900)
    b = wl.Batch(**{**b.__dict__, "with_append": True})
    t = wl.make_tensors(b, DEV, poison_unused=True)
    ks, vs = fp8_scales(Hkv, 600 + Hq)
    kc, vc = quantise_pool(t.k_cache, ks), quantise_pool(t.v_cache, vs)
    k0, v0 = kc.cpu().numpy().copy(), vc.cpu().numpy().copy()
    qkv = torch.cat([t.q.reshape(b.T, -1), t.k_new.reshape(b.T, -1), t.v_new.reshape(b.T, -1)], dim=1).contiguous()
    h = binding.handle_for(b, t, fp8_caches=(kc, vc), kv_scales=(dev(ks), dev(vs)))
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    q_rot = h.qkv_rope_append(qkv, bt, qsl, ctx, THETA[model])
    out = binding.mixed_attention(h, q_rot, bt, qsl, ctx, b.scale)
    torch.cuda.synchronize()
    # oracle: RoPE append into scratch bf16 caches, gather the rotated k rows, FP8 append of those bits
    sk = np.zeros(tuple(t.k_cache.shape), dtype=np.uint16)
    sv = np.zeros_like(sk)
    q_ref = oracle.rope_qkv_append(wl.to_u16(qkv), sk, sv, b.block_table, b.query_start_loc, b.ctx_lens, Hq, THETA[model])
    k_rot = np.zeros((b.T, Hkv, D), dtype=np.uint16)
    for r, (c, u) in enumerate(b.reqs):
        for j in range(c):
            pos = u + j
            k_rot[int(b.query_start_loc[r]) + j] = sk[int(b.block_table[r][pos // 16]), :, pos % 16, :]
    oracle.kv_append_fp8(k0, v0, k_rot, wl.to_u16(t.v_new), ks, vs, b.block_table, b.query_start_loc, b.ctx_lens)
    assert_same_bf16_bits(wl.to_u16(q_rot), q_ref, "rotated q")
    assert np.array_equal(vc.cpu().numpy(), v0), "FP8 v codes differ"
    assert np.array_equal(kc.cpu().numpy(), k0), "FP8 k codes differ"
    # attention: the oracle on ITS OWN q and codes (nothing the CUDA path produced)
    ref, _ = oracle.mixed_attention_fp8(q_ref, k0, v0, ks, vs, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    check_attention(b, out, ref)
