"""ss_mixed_attention_static: the attention step for callers that cannot allocate device memory.

Who cannot: a serving engine that gave all free HBM to its paged KV cache at start-up (a later cudaMalloc fails, or at
best stalls the device), and code hosted inside another framework's memory pool.  They get one call that takes no
handle and no workspace; its scratch is an 8 MiB array inside the library, shared by every call on the device and
never cleared between calls except for the counters the call zeroes itself.

What is checked: the new entry point against the existing route (ss_create + ss_mixed_attention with a torch
workspace) on the same inputs, within the tolerance of tests/test_gpu_parity.py, for calls made back to back on the
shared array - with a different head layout in between, so the second and third call find the previous call's work
list, partials and counters lying where theirs now go.  The batches have long decode contexts, so the split-KV
partials and arrival counters (the scratch that must not be stale) are really used.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests.  It makes no assumption about what ran before it - it passes alone in a fresh process (where its first call
performs the per-device set-up) and after the whole suite.
"""
import numpy as np
import pytest
import torch

from paper_2606_05933_b200 import binding, workloads as wl

pytestmark = pytest.mark.gpu

MAX_ABS, MEAN_ABS = 2e-2, 2e-3          # tests/test_gpu_parity.py
DEV = "cuda:0"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def both_routes(b):
    """(existing route, static-scratch route, lse of each) on one batch whose cache already holds every token."""
    t = wl.make_tensors(b, DEV, poison_unused=True)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    h = binding.handle_for(b, t)
    if b.with_append:
        binding.kv_append(h, t.k_new, t.v_new, bt, qsl, ctx)
    lse_ref = torch.full((b.T, b.num_q_heads), float("nan"), dtype=torch.float32, device=DEV)
    ref = binding.mixed_attention(h, t.q, bt, qsl, ctx, b.scale, out=torch.full_like(t.q, float("nan")), lse=lse_ref)
    lse_got = torch.full_like(lse_ref, float("nan"))
    got = binding.mixed_attention_static(t.k_cache, t.v_cache, t.q, bt, qsl, ctx, b.scale,
                                         out=torch.full_like(t.q, float("nan")), lse=lse_got)
    torch.cuda.synchronize()
    h.close()
    return ref, got, lse_ref, lse_got


def assert_same(b, ref, got, lse_ref, lse_got):
    r, g = ref.to(torch.float64).cpu().numpy(), got.to(torch.float64).cpu().numpy()
    assert not np.isnan(r).any(), "existing route left rows unwritten"
    assert not np.isnan(g).any(), "static-scratch route left rows unwritten"
    err = np.abs(g - r)
    assert err.max() <= MAX_ABS and err.mean() <= MEAN_ABS, (b.name, err.max(), err.mean())
    assert np.abs(lse_got.cpu().numpy() - lse_ref.cpu().numpy()).max() <= 2e-2, b.name


def batch_a():
    # Llama-3-8B heads; decodes long enough to be split over several CTAs, two prefill chunks, an empty request
    reqs = [(1, 9000), (1, 5), (1, 12345), (300, 4000), (1, 0), (0, 40), (1, 4095), (130, 0), (1, 4096), (1, 511)]
    return wl.make_batch("static-a", 32, 8, 128, reqs, 501, with_append=True)


def batch_b():
    # other head count, group size and head_dim: every region of the scratch sits at a different offset than for batch_a
    reqs = [(1, 7000), (200, 1000), (1, 3), (1, 6200), (1, 2048), (17, 33)]
    return wl.make_batch("static-b", 8, 2, 64, reqs, 502, with_append=True)


def test_static_scratch_matches_existing_route_on_calls_in_a_row():
    for b in (batch_a(), batch_b(), batch_a(), batch_a()):
        assert_same(b, *both_routes(b))


def test_static_scratch_same_batch_twice_is_bitwise_reproducible():
    """Two calls in a row on identical inputs: the second starts from the first one's leftovers and must not see them."""
    b = batch_a()
    t = wl.make_tensors(b, DEV)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    outs = []
    for _ in range(2):
        out = torch.full_like(t.q, float("nan"))
        binding.mixed_attention_static(t.k_cache, t.v_cache, t.q, bt, qsl, ctx, b.scale, out=out)
        outs.append(out)
    torch.cuda.synchronize()
    assert torch.equal(outs[0].view(torch.int16), outs[1].view(torch.int16))


def test_static_scratch_refuses_configs_beyond_its_maximum():
    """A config whose worst case needs more than the 8 MiB array is refused up front, with both sizes in the message,
    and `out` is left untouched."""
    b = wl.config_tiny()
    t = wl.make_tensors(b, DEV)
    bt, qsl, ctx = dev(b.block_table), dev(b.query_start_loc), dev(b.ctx_lens)
    out = torch.full_like(t.q, float("nan"))
    with pytest.raises(binding.SlidingAttnError, match="SS_ERR_WORKSPACE_TOO_SMALL.*8388608") as ei:
        binding.mixed_attention_static(t.k_cache, t.v_cache, t.q, bt, qsl, ctx, b.scale, out=out,
                                       max_requests=2048, max_tokens=1 << 24)
    assert ei.value.status == -2
    torch.cuda.synchronize()
    assert torch.isnan(out.float()).all()
    # the same batch with bounds that fit goes through
    binding.mixed_attention_static(t.k_cache, t.v_cache, t.q, bt, qsl, ctx, b.scale, out=out)
    torch.cuda.synchronize()
    assert not torch.isnan(out.float()).any()
