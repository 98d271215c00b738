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
_SRC = _HERE / "attn_oracle.c"
_LIB = _HERE / "liboracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile attn_oracle.c -> oracle/liboracle.so with gcc (-O2 -fopenmp, no fast-math)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-fno-fast-math",
               "-o", str(tmp), str(_SRC), "-lm"]
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
