"""fp64 CPU oracle for the mixed prefill+decode paged-attention path — TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It shares no code with ``paper_2606_05933_b200`` (the CUDA product) and
never imports it.  The arithmetic lives in ``attn_oracle.c`` (plain C, fp64, OpenMP over query rows);
this file only compiles it with gcc and marshals numpy arrays through ctypes.

What it computes and which passage of the paper each function follows is stated in ``attn_oracle.c``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRCS = [_HERE / "attn_oracle.c", _HERE / "next_oracle.c"]
_LIB = _HERE / "liboracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile attn_oracle.c + next_oracle.c -> oracle/liboracle.so with gcc (-O2 -fopenmp, no fast-math)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < max(s.stat().st_mtime for s in _SRCS):
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=gnu11", "-fno-fast-math", "-ffp-contract=off",
               "-o", str(tmp), *map(str, _SRCS), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        vp, i32, i64p = ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_int64)
        lib.oracle_kv_append.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32]
        lib.oracle_kv_append.restype = i32
        lib.oracle_mixed_attention.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32,
                                               ctypes.c_float, vp, i32, vp, vp, i64p]
        lib.oracle_mixed_attention.restype = i32
        lib.oracle_num_threads.restype = i32
        f64, i64 = ctypes.c_double, ctypes.c_int64
        lib.oracle_rope_rotate.argtypes = [vp, i32, i64, f64, vp]
        lib.oracle_rope_qkv_append.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, f64]
        lib.oracle_rope_qkv_append.restype = i32
        lib.oracle_kv_append_fp8.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32]
        lib.oracle_kv_append_fp8.restype = i32
        lib.oracle_mixed_attention_fp8.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, i32,
                                                   ctypes.c_float, vp, i32, vp, vp]
        lib.oracle_mixed_attention_fp8.restype = i32
        lib.oracle_f64_to_bf16_array.argtypes = [vp, i64, vp]
        lib.oracle_f32_to_e4m3_array.argtypes = [vp, i64, vp]
        lib.oracle_e4m3_to_f64_array.argtypes = [vp, i64, vp]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _u16(a, name):
    a = np.ascontiguousarray(a)
    if a.dtype != np.uint16:
        raise TypeError(f"{name}: expected uint16 bf16 bit patterns, got {a.dtype}")
    return a


def _i32(a, name):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a


def kv_append(k_cache, v_cache, k_new, v_new, block_table, query_start_loc, ctx_lens):
    """In-place oracle append.  k_cache/v_cache: uint16 [P,Hkv,page,D]; k_new/v_new: uint16 [T,Hkv,D]."""
    lib = _load()
    for c in (k_cache, v_cache):
        if c.dtype != np.uint16 or not c.flags.c_contiguous or not c.flags.writeable:
            raise TypeError("caches must be writable C-contiguous uint16 arrays")
    k_new, v_new = _u16(k_new, "k_new"), _u16(v_new, "v_new")
    bt, qsl, ctx = _i32(block_table, "bt"), _i32(query_start_loc, "qsl"), _i32(ctx_lens, "ctx")
    _, Hkv, page, D = k_cache.shape
    R = ctx.shape[0]
    rc = lib.oracle_kv_append(k_cache.ctypes.data, v_cache.ctypes.data, k_new.ctypes.data,
                              v_new.ctypes.data, bt.ctypes.data, qsl.ctypes.data, ctx.ctypes.data,
                              R, bt.shape[1] if bt.ndim == 2 else 0, Hkv, D, page)
    if rc != 0:
        raise RuntimeError(f"oracle_kv_append failed: {rc}")


def mixed_attention(q, k_cache, v_cache, block_table, query_start_loc, ctx_lens, scale, rows=None):
    """fp64 attention.  q: uint16 [T,Hq,D]; caches uint16 [P,Hkv,page,D].

    Returns (out float64 [n,Hq,D], lse float64 [n,Hq], pairs int) with n = len(rows) or T."""
    lib = _load()
    q, k_cache, v_cache = _u16(q, "q"), _u16(k_cache, "k_cache"), _u16(v_cache, "v_cache")
    bt, qsl, ctx = _i32(block_table, "bt"), _i32(query_start_loc, "qsl"), _i32(ctx_lens, "ctx")
    T, Hq, D = q.shape
    _, Hkv, page, Dk = k_cache.shape
    assert Dk == D and v_cache.shape == k_cache.shape
    R = ctx.shape[0]
    assert qsl.shape[0] == R + 1 and (R == 0 or int(qsl[R]) == T)
    if rows is not None:
        rows = _i32(rows, "rows")
        n = rows.shape[0]
        rows_p = rows.ctypes.data
    else:
        n, rows_p = T, None
    out = np.empty((n, Hq, D), dtype=np.float64)
    lse = np.empty((n, Hq), dtype=np.float64)
    pairs = ctypes.c_int64(0)
    rc = lib.oracle_mixed_attention(q.ctypes.data, k_cache.ctypes.data, v_cache.ctypes.data,
                                    bt.ctypes.data, qsl.ctypes.data, ctx.ctypes.data, R,
                                    bt.shape[1] if bt.ndim == 2 else 0, Hq, Hkv, D, page,
                                    ctypes.c_float(np.float32(scale)), rows_p, n,
                                    out.ctypes.data, lse.ctypes.data, ctypes.byref(pairs))
    if rc != 0:
        raise RuntimeError(f"oracle_mixed_attention failed: {rc}")
    return out, lse, int(pairs.value)


# ------------------------------------------------------------------------------------------------------------------
# next_oracle.c: RoPE + QKV split fused into the append (NEXT-4), FP8 E4M3 KV cache (NEXT-3)
# ------------------------------------------------------------------------------------------------------------------
def f64_to_bf16(x) -> np.ndarray:
    """double -> bf16 bit patterns, one rounding to nearest even."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    out = np.empty(x.shape, dtype=np.uint16)
    _load().oracle_f64_to_bf16_array(x.ctypes.data, x.size, out.ctypes.data)
    return out


def f32_to_e4m3(x) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float32)
    out = np.empty(x.shape, dtype=np.uint8)
    _load().oracle_f32_to_e4m3_array(x.ctypes.data, x.size, out.ctypes.data)
    return out


def e4m3_to_f64(codes) -> np.ndarray:
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    out = np.empty(codes.shape, dtype=np.float64)
    _load().oracle_e4m3_to_f64_array(codes.ctypes.data, codes.size, out.ctypes.data)
    return out


def rope_rotate(x, pos: int, theta: float) -> np.ndarray:
    """RoPE of one head vector (float64 in, float64 out)."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    out = np.empty_like(x)
    _load().oracle_rope_rotate(x.ctypes.data, x.shape[0], int(pos), float(theta), out.ctypes.data)
    return out


def rope_qkv_append(qkv, k_cache, v_cache, block_table, query_start_loc, ctx_lens, Hq: int, theta: float):
    """qkv uint16 [T,(Hq+2Hkv)*D]; caches uint16 [P,Hkv,page,D] updated in place; returns q_out uint16 [T,Hq,D]."""
    lib = _load()
    qkv = _u16(qkv, "qkv")
    for c in (k_cache, v_cache):
        if c.dtype != np.uint16 or not c.flags.c_contiguous or not c.flags.writeable:
            raise TypeError("caches must be writable C-contiguous uint16 arrays")
    bt, qsl, ctx = _i32(block_table, "bt"), _i32(query_start_loc, "qsl"), _i32(ctx_lens, "ctx")
    _, Hkv, page, D = k_cache.shape
    T = qkv.shape[0]
    assert qkv.shape[1] == (Hq + 2 * Hkv) * D
    q_out = np.zeros((T, Hq, D), dtype=np.uint16)
    rc = lib.oracle_rope_qkv_append(qkv.ctypes.data, q_out.ctypes.data, k_cache.ctypes.data, v_cache.ctypes.data,
                                    bt.ctypes.data, qsl.ctypes.data, ctx.ctypes.data, ctx.shape[0],
                                    bt.shape[1] if bt.ndim == 2 else 0, Hq, Hkv, D, page, float(theta))
    if rc != 0:
        raise RuntimeError(f"oracle_rope_qkv_append failed: {rc}")
    return q_out


def kv_append_fp8(k_cache, v_cache, k_new, v_new, k_scale, v_scale, block_table, query_start_loc, ctx_lens):
    """In-place FP8 append.  caches uint8 [P,Hkv,page,D] (e4m3 codes); k_new/v_new uint16 [T,Hkv,D]; scales fp32 [Hkv]."""
    lib = _load()
    for c in (k_cache, v_cache):
        if c.dtype != np.uint8 or not c.flags.c_contiguous or not c.flags.writeable:
            raise TypeError("FP8 caches must be writable C-contiguous uint8 arrays")
    k_new, v_new = _u16(k_new, "k_new"), _u16(v_new, "v_new")
    ks, vs = np.ascontiguousarray(k_scale, dtype=np.float32), np.ascontiguousarray(v_scale, dtype=np.float32)
    bt, qsl, ctx = _i32(block_table, "bt"), _i32(query_start_loc, "qsl"), _i32(ctx_lens, "ctx")
    _, Hkv, page, D = k_cache.shape
    rc = lib.oracle_kv_append_fp8(k_cache.ctypes.data, v_cache.ctypes.data, k_new.ctypes.data, v_new.ctypes.data,
                                  ks.ctypes.data, vs.ctypes.data, bt.ctypes.data, qsl.ctypes.data, ctx.ctypes.data,
                                  ctx.shape[0], bt.shape[1] if bt.ndim == 2 else 0, Hkv, D, page)
    if rc != 0:
        raise RuntimeError(f"oracle_kv_append_fp8 failed: {rc}")


def mixed_attention_fp8(q, k_cache, v_cache, k_scale, v_scale, block_table, query_start_loc, ctx_lens, scale, rows=None):
    """fp64 attention over an FP8 E4M3 cache (codes uint8 [P,Hkv,page,D], scales fp32 [Hkv]).  Returns (out, lse)."""
    lib = _load()
    q = _u16(q, "q")
    k_cache, v_cache = np.ascontiguousarray(k_cache, dtype=np.uint8), np.ascontiguousarray(v_cache, dtype=np.uint8)
    ks, vs = np.ascontiguousarray(k_scale, dtype=np.float32), np.ascontiguousarray(v_scale, dtype=np.float32)
    bt, qsl, ctx = _i32(block_table, "bt"), _i32(query_start_loc, "qsl"), _i32(ctx_lens, "ctx")
    T, Hq, D = q.shape
    _, Hkv, page, _ = k_cache.shape
    if rows is not None:
        rows = _i32(rows, "rows")
        n, rows_p = rows.shape[0], rows.ctypes.data
    else:
        n, rows_p = T, None
    out = np.empty((n, Hq, D), dtype=np.float64)
    lse = np.empty((n, Hq), dtype=np.float64)
    rc = lib.oracle_mixed_attention_fp8(q.ctypes.data, k_cache.ctypes.data, v_cache.ctypes.data, ks.ctypes.data,
                                        vs.ctypes.data, bt.ctypes.data, qsl.ctypes.data, ctx.ctypes.data, ctx.shape[0],
                                        bt.shape[1] if bt.ndim == 2 else 0, Hq, Hkv, D, page,
                                        ctypes.c_float(np.float32(scale)), rows_p, n, out.ctypes.data, lse.ctypes.data)
    if rc != 0:
        raise RuntimeError(f"oracle_mixed_attention_fp8 failed: {rc}")
    return out, lse
