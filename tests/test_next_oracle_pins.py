"""Pins of oracle/next_oracle.c (CPU only): RoPE + QKV-split fused into the append and the
FP8 E4M3 KV cache (NEXT-3).  Each pin checks the oracle against something other than itself: closed forms, invariants,
the complex-multiplication statement of RoPE evaluated with numpy, torch's own cos/sin/rotate_half formula and
float8_e4m3fn type, the OCP value table written out by hand, exhaustive neighbour/midpoint arithmetic."""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2606_05933_b200 import workloads as wl
from helpers import f64_to_u16, u16_to_f64

THETA = 500000.0          # Llama-3's rope_theta; Qwen2.5 uses 1e6 (public model configs)


# ------------------------------------------------------------------------------------------------------------------
# double -> bf16, one rounding to nearest even
# ------------------------------------------------------------------------------------------------------------------
def _all_finite_bf16():
    bits = np.arange(0x10000, dtype=np.uint32).astype(np.uint16)
    vals = u16_to_f64(bits)
    keep = np.isfinite(vals)
    return bits[keep], vals[keep]


def test_bf16_rounding_is_exact_on_representable_values_and_ties_to_even():
    bits, vals = _all_finite_bf16()
    assert np.array_equal(oracle.f64_to_bf16(vals)[vals != 0], bits[vals != 0])          # every bf16 value round-trips
    pos = np.sort(vals[vals > 0])
    lo, hi = pos[:-1], pos[1:]
    mid = (lo + hi) / 2                                    # exact in double
    lo_bits, hi_bits = f64_to_u16(lo), f64_to_u16(hi)
    want_tie = np.where(lo_bits % 2 == 0, lo_bits, hi_bits)                               # ties go to the even pattern
    assert np.array_equal(oracle.f64_to_bf16(mid), want_tie)
    eps = (hi - lo) * 2.0 ** -20                           # far below fp32 resolution: a double->float->bf16 path fails here
    assert np.array_equal(oracle.f64_to_bf16(mid + eps), hi_bits)
    assert np.array_equal(oracle.f64_to_bf16(mid - eps), lo_bits)
    assert np.array_equal(oracle.f64_to_bf16(-(mid + eps)), hi_bits | 0x8000)


# ------------------------------------------------------------------------------------------------------------------
# RoPE
# ------------------------------------------------------------------------------------------------------------------
def test_rope_position_zero_is_the_identity_and_pairs_keep_their_norm():
    rng = np.random.default_rng(0)
    for D in (64, 128):
        x = rng.standard_normal(D)
        assert np.array_equal(oracle.rope_rotate(x, 0, THETA), x)
        for pos in (1, 17, 4096, 32767, 131071):
            y = oracle.rope_rotate(x, pos, THETA)
            h = D // 2
            assert np.allclose(y[:h] ** 2 + y[h:] ** 2, x[:h] ** 2 + x[h:] ** 2, rtol=1e-13, atol=0)


def test_rope_equals_complex_multiplication_by_unit_phasors():
    """(x_i + i x_{i+D/2}) * exp(i pos theta^(-2i/D)): the textbook statement, evaluated with numpy complex arithmetic."""
    rng = np.random.default_rng(1)
    D = 128
    x = rng.standard_normal(D)
    for pos in (3, 1000, 30000):
        z = (x[:D // 2] + 1j * x[D // 2:]) * np.exp(1j * pos * THETA ** (-2.0 * np.arange(D // 2) / D))
        y = oracle.rope_rotate(x, pos, THETA)
        assert np.allclose(y[:D // 2], z.real, rtol=0, atol=1e-12) and np.allclose(y[D // 2:], z.imag, rtol=0, atol=1e-12)


def test_rope_matches_the_rotate_half_formula_in_torch_fp64():
    """q*cos + rotate_half(q)*sin with cos/sin = cat(freqs, freqs) - the public formulation of the model families the
    paper serves, written with torch ops."""
    g = torch.Generator().manual_seed(2)
    D = 128
    x = torch.randn(D, dtype=torch.float64, generator=g)
    for pos in (5, 2047, 20000):
        inv = 1.0 / (THETA ** (torch.arange(0, D, 2, dtype=torch.float64) / D))
        emb = torch.cat([pos * inv, pos * inv])
        rot = torch.cat([-x[D // 2:], x[:D // 2]])
        want = x * emb.cos() + rot * emb.sin()
        got = oracle.rope_rotate(x.numpy(), pos, THETA)
        assert np.allclose(got, want.numpy(), rtol=0, atol=1e-12)


def test_rope_scores_depend_on_relative_position_only():
    rng = np.random.default_rng(3)
    D = 64
    q, k = rng.standard_normal(D), rng.standard_normal(D)
    base = oracle.rope_rotate(q, 900, THETA) @ oracle.rope_rotate(k, 650, THETA)
    for shift in (1, 77, 5000):
        s = oracle.rope_rotate(q, 900 + shift, THETA) @ oracle.rope_rotate(k, 650 + shift, THETA)
        assert abs(s - base) < 1e-9
    assert abs(oracle.rope_rotate(q, 900, THETA) @ oracle.rope_rotate(k, 651, THETA) - base) > 1e-6


def _qkv_case(seed, Hq=8, Hkv=2, D=128):
    b = wl.random_batch(seed, Hq=Hq, Hkv=Hkv, D=D, n_prefill=2, n_decode=4, max_c=70, max_u=300)
    t = wl.make_tensors(b, "cpu")
    qkv = torch.cat([t.q.reshape(b.T, -1), t.k_new.reshape(b.T, -1), t.v_new.reshape(b.T, -1)], dim=1).contiguous()
    return b, t, wl.to_u16(qkv)


def test_rope_qkv_append_places_every_token_like_kv_append_and_rotates_by_its_position():
    b, t, qkv = _qkv_case(11)
    k0, v0 = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    k1, v1 = k0.copy(), v0.copy()
    q_out = oracle.rope_qkv_append(qkv, k1, v1, b.block_table, b.query_start_loc, b.ctx_lens, b.num_q_heads, THETA)
    # V: exactly what the plain kv_append writes, and nothing else is touched (same slots as K)
    kp, vp = k0.copy(), v0.copy()
    oracle.kv_append(kp, vp, wl.to_u16(t.k_new), wl.to_u16(t.v_new), b.block_table, b.query_start_loc, b.ctx_lens)
    assert np.array_equal(v1, vp)
    touched = np.zeros(k0.shape[:3], dtype=bool)
    for r, (c, u) in enumerate(b.reqs):
        for j in range(c):
            pos, tok = u + j, int(b.query_start_loc[r]) + j
            page, slot = int(b.block_table[r, pos // 16]), pos % 16
            touched[page, :, slot] = True
            for h in range(b.num_q_heads):
                want = oracle.f64_to_bf16(oracle.rope_rotate(u16_to_f64(wl.to_u16(t.q[tok, h])), pos, THETA))
                assert np.array_equal(q_out[tok, h], want)
            for g in range(b.num_kv_heads):
                want = oracle.f64_to_bf16(oracle.rope_rotate(u16_to_f64(wl.to_u16(t.k_new[tok, g])), pos, THETA))
                assert np.array_equal(k1[page, g, slot], want)
    assert np.array_equal(k1[~touched], k0[~touched])


def test_rope_with_zero_context_single_token_is_a_plain_append():
    """u = 0, c = 1: position 0, the rotation is the identity -> bit copies of q and k."""
    b = wl.make_batch("p0", 4, 2, 64, [(1, 0), (1, 0)], 5, with_append=True)
    t = wl.make_tensors(b, "cpu")
    qkv = wl.to_u16(torch.cat([t.q.reshape(b.T, -1), t.k_new.reshape(b.T, -1), t.v_new.reshape(b.T, -1)], dim=1).contiguous())
    k1, v1 = wl.to_u16(t.k_cache), wl.to_u16(t.v_cache)
    kp, vp = k1.copy(), v1.copy()
    q_out = oracle.rope_qkv_append(qkv, k1, v1, b.block_table, b.query_start_loc, b.ctx_lens, 4, THETA)
    oracle.kv_append(kp, vp, wl.to_u16(t.k_new), wl.to_u16(t.v_new), b.block_table, b.query_start_loc, b.ctx_lens)
    assert np.array_equal(q_out, wl.to_u16(t.q)) and np.array_equal(k1, kp) and np.array_equal(v1, vp)


# ------------------------------------------------------------------------------------------------------------------
# FP8 E4M3
# ------------------------------------------------------------------------------------------------------------------
def test_e4m3_decode_matches_the_ocp_value_table():
    codes = np.arange(256, dtype=np.uint8)
    got = oracle.e4m3_to_f64(codes)
    for c in range(256):
        s, e, m = c >> 7, (c >> 3) & 15, c & 7
        if e == 15 and m == 7:
            assert math.isnan(got[c])
            continue
        want = (m / 8.0) * 2.0 ** -6 if e == 0 else (1 + m / 8.0) * 2.0 ** (e - 7)
        assert got[c] == (-want if s else want)
    assert got[0x7E] == 448.0 and got[0x08] == 2.0 ** -6 and got[0x01] == 2.0 ** -9 and got[0x38] == 1.0
    # torch's own float8_e4m3fn agrees on every code
    tv = torch.from_numpy(codes.copy()).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    assert np.array_equal(np.isnan(tv), np.isnan(got)) and np.array_equal(tv[~np.isnan(tv)], got[~np.isnan(got)])


def test_e4m3_encode_round_trips_ties_to_even_and_saturates():
    codes = np.array([c for c in range(256) if (c & 0x7F) != 0x7F], dtype=np.uint8)
    vals = oracle.e4m3_to_f64(codes)
    back = oracle.f32_to_e4m3(vals.astype(np.float32))
    assert np.array_equal(back[vals != 0], codes[vals != 0])
    pos_codes = np.arange(0, 0x7E, dtype=np.uint8)
    lo, hi = oracle.e4m3_to_f64(pos_codes), oracle.e4m3_to_f64(pos_codes + 1)
    mid = ((lo + hi) / 2).astype(np.float32)                # exact in fp32 (few significant bits)
    want = np.where(pos_codes % 2 == 0, pos_codes, pos_codes + 1)
    assert np.array_equal(oracle.f32_to_e4m3(mid), want)
    up = np.nextafter(mid, np.float32(np.inf)).astype(np.float32)
    dn = np.nextafter(mid, np.float32(-np.inf)).astype(np.float32)
    assert np.array_equal(oracle.f32_to_e4m3(up), pos_codes + 1) and np.array_equal(oracle.f32_to_e4m3(dn), pos_codes)
    sat = oracle.f32_to_e4m3(np.array([448.0, 449.0, 464.0, 1e30, np.inf, -500.0, -np.inf], dtype=np.float32))
    assert list(sat) == [0x7E, 0x7E, 0x7E, 0x7E, 0x7E, 0xFE, 0xFE]
    assert oracle.f32_to_e4m3(np.array([np.nan], dtype=np.float32))[0] & 0x7F == 0x7F


def test_e4m3_encode_agrees_with_torch_on_every_bf16_input():
    bits, vals = _all_finite_bf16()
    keep = np.abs(vals) <= 448.0                            # torch's cast does not saturate; inside the range it is RNE
    x = vals[keep].astype(np.float32)
    want = torch.from_numpy(x).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    got = oracle.f32_to_e4m3(x)
    nz = x != 0
    assert np.array_equal(got[nz], want[nz])
    assert np.array_equal(got[~nz] & 0x7F, want[~nz] & 0x7F)


def _fp8_case(seed, Hq=8, Hkv=2, D=128):
    b = wl.random_batch(seed, Hq=Hq, Hkv=Hkv, D=D, n_prefill=1, n_decode=5, max_c=40, max_u=200)
    t = wl.make_tensors(b, "cpu")
    return b, t


def test_fp8_append_quantises_with_the_per_head_scale_and_touches_only_its_slots():
    b, t = _fp8_case(21)
    shape = tuple(t.k_cache.shape)
    k8 = np.full(shape, 0x5A, dtype=np.uint8)
    v8 = np.full(shape, 0xA5, dtype=np.uint8)
    ks, vs = np.array([0.5, 0.0625], dtype=np.float32), np.array([2.0, 0.25], dtype=np.float32)
    oracle.kv_append_fp8(k8, v8, wl.to_u16(t.k_new), wl.to_u16(t.v_new), ks, vs, b.block_table, b.query_start_loc, b.ctx_lens)
    touched = np.zeros(shape[:3], dtype=bool)
    for r, (c, u) in enumerate(b.reqs):
        for j in range(c):
            pos, tok = u + j, int(b.query_start_loc[r]) + j
            page, slot = int(b.block_table[r, pos // 16]), pos % 16
            touched[page, :, slot] = True
            for g in range(2):
                xk = t.k_new[tok, g].to(torch.float32) / float(ks[g])
                xv = t.v_new[tok, g].to(torch.float32) / float(vs[g])
                wk = xk.clamp(-448, 448).to(torch.float8_e4m3fn).view(torch.uint8).numpy()     # torch: RNE inside the range
                wv = xv.clamp(-448, 448).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
                assert np.array_equal(k8[page, g, slot], wk) and np.array_equal(v8[page, g, slot], wv)
    assert (k8[~touched] == 0x5A).all() and (v8[~touched] == 0xA5).all()


def test_fp8_attention_with_unit_scale_on_representable_inputs_equals_the_bf16_oracle():
    """K, V drawn from the e4m3 grid are exact in both formats: the FP8 oracle at scale 1 must reproduce the bf16 oracle
    bit for bit (same arithmetic, same order), and a power-of-two scale on pre-scaled codes must give the same values."""
    b, t = _fp8_case(22)
    rng = np.random.default_rng(22)
    shape = tuple(t.k_cache.shape)
    k8 = rng.integers(0, 0x78, size=shape, dtype=np.uint8) | (rng.integers(0, 2, size=shape, dtype=np.uint8) << 7)
    v8 = rng.integers(0, 0x78, size=shape, dtype=np.uint8) | (rng.integers(0, 2, size=shape, dtype=np.uint8) << 7)
    kb, vb = f64_to_u16(oracle.e4m3_to_f64(k8)), f64_to_u16(oracle.e4m3_to_f64(v8))
    assert np.array_equal(u16_to_f64(kb), oracle.e4m3_to_f64(k8))                          # exact in bf16
    one = np.ones(2, dtype=np.float32)
    q = wl.to_u16(t.q)
    ref, lse_ref, _ = oracle.mixed_attention(q, kb, vb, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    got, lse = oracle.mixed_attention_fp8(q, k8, v8, one, one, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    assert np.array_equal(got, ref) and np.array_equal(lse, lse_ref)
    # scale 4 on the same codes == bf16 oracle on 4x the values (power of two: exact)
    four = np.full(2, 4.0, dtype=np.float32)
    ref4, _, _ = oracle.mixed_attention(q, f64_to_u16(4 * oracle.e4m3_to_f64(k8)), f64_to_u16(4 * oracle.e4m3_to_f64(v8)),
                                        b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    got4, _ = oracle.mixed_attention_fp8(q, k8, v8, four, four, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    assert np.allclose(got4, ref4, rtol=1e-13, atol=1e-15)


def test_fp8_attention_closed_forms():
    """Q = 0 -> every row is the prefix mean of the dequantised V; a single cached key returns dequantised V exactly."""
    b = wl.make_batch("cf", 4, 2, 64, [(1, 0), (1, 37), (6, 10)], 23, with_append=False)
    t = wl.make_tensors(b, "cpu")
    rng = np.random.default_rng(23)
    shape = tuple(t.k_cache.shape)
    k8 = rng.integers(0, 0x70, size=shape, dtype=np.uint8)
    v8 = rng.integers(0, 0x70, size=shape, dtype=np.uint8) | (rng.integers(0, 2, size=shape, dtype=np.uint8) << 7)
    ks, vs = np.array([0.3, 1.7], dtype=np.float32), np.array([0.11, 2.5], dtype=np.float32)
    q0 = np.zeros((b.T, 4, 64), dtype=np.uint16)
    out, lse = oracle.mixed_attention_fp8(q0, k8, v8, ks, vs, b.block_table, b.query_start_loc, b.ctx_lens, b.scale)
    for r, (c, u) in enumerate(b.reqs):
        for j in range(c):
            n, row = u + j + 1, int(b.query_start_loc[r]) + j
            for h in range(4):
                g = h // 2
                vv = np.stack([oracle.e4m3_to_f64(v8[int(b.block_table[r, p // 16]), g, p % 16]) for p in range(n)]) * float(vs[g])
                assert np.allclose(out[row, h], vv.mean(0), rtol=1e-12, atol=1e-15)
                assert abs(lse[row, h] - math.log(n)) < 1e-12
    qr = wl.to_u16(t.q)
    out1, _ = oracle.mixed_attention_fp8(qr, k8, v8, ks, vs, b.block_table, b.query_start_loc, b.ctx_lens, b.scale, rows=np.array([0]))
    page = int(b.block_table[0, 0])
    for h in range(4):
        assert np.array_equal(out1[0, h], oracle.e4m3_to_f64(v8[page, h // 2, 0]) * float(vs[h // 2]))
