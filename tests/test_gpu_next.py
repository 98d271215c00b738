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


def assert_within_one_bf16_ulp(got_u16, want_u16, what):
    g, w = u16_to_f64(got_u16), u16_to_f64(want_u16)
    odd = ~np.isfinite(w)                                   # poisoned unused slots (NaN payloads): must be untouched bits
    assert np.array_equal(got_u16[odd], want_u16[odd]), f"{what}: non-finite patterns differ"
    g, w = np.where(odd, 0.0, g), np.where(odd, 0.0, w)
    assert np.isfinite(g).all(), f"{what}: non-finite values"
    diff = np.abs(g - w)
    ulp = np.maximum(np.abs(g), np.abs(w)) * 2.0 ** -7 + 3e-6
    assert (diff <= ulp).all(), f"{what}: more than one bf16 ulp (+ 3e-6) apart (max {diff.max():.3e})"
    frac = float((got_u16 != want_u16).mean())
    assert frac < 2e-3, f"{what}: {frac:.2%} of the elements differ"


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
    assert_within_one_bf16_ulp(wl.to_u16(q_rot), q_ref, "rotated q")
    assert_within_one_bf16_ulp(wl.to_u16(t.k_cache), k0, "k_cache (rotated k; untouched slots identical)")
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
