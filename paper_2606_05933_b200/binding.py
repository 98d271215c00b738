"""ctypes binding of libslidingattn.so (include/slidingattn.h).  Argument marshalling only: every step of
the path runs in the CUDA kernels.  There is no CPU fallback — if the compiled library is missing or no
sm_100 device is present the calls raise."""
from __future__ import annotations

import ctypes
from pathlib import Path
from typing import Optional

import numpy as np
import torch

_PKG = Path(__file__).resolve().parent
LIB_PATH = _PKG / "libslidingattn.so"
_lib = None

SS_OK = 0
SS_ERR_INVALID_ARG = -1
SS_ERR_DEVICE_CHECK = -6
SS_FLAG_DEBUG_CHECKS = 1
SS_FLAG_KV_FP8 = 2
# include/slidingattn.h (the product boundary) ...
EXPORTS = ["ss_version", "ss_status_string", "ss_last_error_string", "ss_create", "ss_destroy",
           "ss_workspace_bytes", "ss_set_kv_scales", "ss_kv_append", "ss_qkv_rope_append", "ss_mixed_attention",
           "ss_mixed_attention_static", "ss_iteration_host",
           "ss_poll_device_error", "ss_reset"]
# ... and include/slidingattn_debug.h (test / tuning / measurement aids)
DEBUG_EXPORTS = ["ss_build_worklist", "ss_last_launch_count", "ss_debug_force_simple_path",
                 "ss_debug_set_param", "ss_debug_set_trace", "ss_set_kernel_timing", "ss_last_kernel_time_us",
                 "ss_debug_stream_read"]


class ss_config(ctypes.Structure):
    _fields_ = [("num_q_heads", ctypes.c_int32), ("num_kv_heads", ctypes.c_int32),
                ("head_dim", ctypes.c_int32), ("page_size", ctypes.c_int32),
                ("num_pages", ctypes.c_int64), ("max_requests", ctypes.c_int32),
                ("max_tokens", ctypes.c_int32), ("max_pages_per_req", ctypes.c_int32),
                ("flags", ctypes.c_uint32)]


class ss_work_item(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in
                ("kind", "req", "head", "row0", "nrows", "kv_begin", "kv_end", "split", "nsplit",
                 "partial", "q_pos0", "nheads")]


WORK_ITEM_DTYPE = np.dtype([(n, np.int32) for n, _ in ss_work_item._fields_])


class SlidingAttnError(RuntimeError):
    pass


def load():
    """dlopen the in-tree library; raises (never falls back) if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise SlidingAttnError(f"{LIB_PATH} not built: run `python -m paper_2606_05933_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
    lib = ctypes.CDLL(str(LIB_PATH))
    vp, i32, f32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_float
    lib.ss_version.restype = ctypes.c_int
    lib.ss_status_string.restype = ctypes.c_char_p
    lib.ss_status_string.argtypes = [ctypes.c_int]
    lib.ss_last_error_string.restype = ctypes.c_char_p
    lib.ss_last_error_string.argtypes = [vp]
    lib.ss_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(ss_config), vp, vp]
    lib.ss_destroy.argtypes = [vp]
    lib.ss_workspace_bytes.argtypes = [vp]
    lib.ss_workspace_bytes.restype = ctypes.c_size_t
    lib.ss_set_kv_scales.argtypes = [vp, vp, vp]
    lib.ss_kv_append.argtypes = [vp, vp, vp, vp, vp, vp, i32, i32, vp]
    lib.ss_qkv_rope_append.argtypes = [vp, vp, vp, vp, vp, i32, i32, f32, vp, vp]
    lib.ss_mixed_attention.argtypes = [vp, vp, vp, vp, vp, i32, i32, f32, vp, vp, vp, ctypes.c_size_t, vp]
    lib.ss_mixed_attention_static.argtypes = [ctypes.POINTER(ss_config), vp, vp, vp, vp, vp, vp, i32, i32, f32, vp, vp,
                                              vp, ctypes.c_char_p, ctypes.c_size_t]
    lib.ss_build_worklist.argtypes = [vp, vp, vp, i32, i32, vp, ctypes.c_size_t, vp, i32,
                                      ctypes.POINTER(i32 * 3), vp]
    lib.ss_iteration_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, i32, i32, f32, vp, vp]
    lib.ss_last_launch_count.argtypes = [vp]
    lib.ss_poll_device_error.argtypes = [vp, vp]
    lib.ss_reset.argtypes = [vp, vp]
    lib.ss_debug_force_simple_path.argtypes = [vp, ctypes.c_int]
    lib.ss_debug_set_param.argtypes = [vp, ctypes.c_int, ctypes.c_int]
    lib.ss_debug_set_trace.argtypes = [vp, vp, i32]
    lib.ss_debug_stream_read.argtypes = [vp, vp, ctypes.c_size_t, vp]
    lib.ss_set_kernel_timing.argtypes = [vp, ctypes.c_int]
    lib.ss_last_kernel_time_us.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    for name in EXPORTS + DEBUG_EXPORTS:
        if name not in ("ss_status_string", "ss_last_error_string", "ss_workspace_bytes"):
            getattr(lib, name).restype = ctypes.c_int
    _lib = lib
    return lib


def _ptr(t: Optional[torch.Tensor]) -> Optional[int]:
    return None if t is None else t.data_ptr()


def _want(t: torch.Tensor, name: str, dtype, cuda: bool = True, shape=None):
    """The C ABI takes raw pointers: a wrong dtype (torch's default int64 indices!), a strided view or a host
    tensor would be read as garbage with no error, so refuse them here."""
    if not isinstance(t, torch.Tensor):
        raise SlidingAttnError(f"{name}: expected a torch.Tensor")
    if t.dtype != dtype:
        raise SlidingAttnError(f"{name}: expected {dtype}, got {t.dtype}")
    if cuda != t.is_cuda:
        raise SlidingAttnError(f"{name}: expected a {'CUDA' if cuda else 'host'} tensor")
    if not t.is_contiguous():
        raise SlidingAttnError(f"{name}: must be contiguous")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise SlidingAttnError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream or None


class SlidingAttn:
    """Handle bound to one pair of paged caches [num_pages, Hkv, 16, D] on the current device: bf16, or uint8 E4M3
    codes (SS_FLAG_KV_FP8; then `kv_scales` = (k_scale, v_scale), float32 CUDA tensors of Hkv entries each)."""

    def __init__(self, num_q_heads: int, num_kv_heads: int, head_dim: int, k_cache: torch.Tensor,
                 v_cache: torch.Tensor, max_requests: int, max_tokens: int, max_pages_per_req: int,
                 debug_checks: bool = False, kv_scales=None):
        self.lib = load()
        if not (k_cache.is_cuda and v_cache.is_cuda):
            raise SlidingAttnError("caches must be CUDA tensors (no CPU path exists)")
        fp8 = k_cache.dtype == torch.uint8
        assert (fp8 or k_cache.dtype == torch.bfloat16) and v_cache.dtype == k_cache.dtype
        assert k_cache.is_contiguous() and v_cache.is_contiguous() and k_cache.shape == v_cache.shape
        P, Hkv, page, D = k_cache.shape
        assert Hkv == num_kv_heads and D == head_dim
        flags = (SS_FLAG_DEBUG_CHECKS if debug_checks else 0) | (SS_FLAG_KV_FP8 if fp8 else 0)
        self.cfg = ss_config(num_q_heads, num_kv_heads, head_dim, page, P, max_requests, max_tokens,
                             max_pages_per_req, flags)
        self.k_cache, self.v_cache = k_cache, v_cache
        self._h = ctypes.c_void_p()
        self._check(self.lib.ss_create(ctypes.byref(self._h), ctypes.byref(self.cfg), k_cache.data_ptr(),
                                       v_cache.data_ptr()), create=True)
        self.workspace_bytes = int(self.lib.ss_workspace_bytes(self._h))
        self.workspace = torch.empty(self.workspace_bytes, dtype=torch.uint8, device=k_cache.device)
        if kv_scales is not None:
            self.set_kv_scales(*kv_scales)

    def set_kv_scales(self, k_scale: torch.Tensor, v_scale: torch.Tensor):
        """FP8 handles: per kv head fp32 scales (device tensors; the handle keeps them alive and the kernels read them)."""
        _want(k_scale, "k_scale", torch.float32, True, (self.cfg.num_kv_heads,))
        _want(v_scale, "v_scale", torch.float32, True, (self.cfg.num_kv_heads,))
        self.k_scale, self.v_scale = k_scale, v_scale
        self._check(self.lib.ss_set_kv_scales(self._h, k_scale.data_ptr(), v_scale.data_ptr()))

    def _check(self, rc: int, create: bool = False):
        if rc != SS_OK:
            detail = b"" if create or not self._h else self.lib.ss_last_error_string(self._h)
            err = SlidingAttnError(f"{self.lib.ss_status_string(rc).decode()} ({rc}) {detail.decode()}")
            err.status = rc
            raise err

    def close(self):
        if getattr(self, "_h", None):
            self.lib.ss_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the two calls of the path -------------------------------------------------------------
    def _check_batch(self, block_table, query_start_loc, ctx_lens, cuda=True):
        R = ctx_lens.shape[0]
        _want(ctx_lens, "ctx_lens", torch.int32, cuda, (R,))
        _want(query_start_loc, "query_start_loc", torch.int32, cuda, (R + 1,))
        _want(block_table, "block_table", torch.int32, cuda, (R, self.cfg.max_pages_per_req))
        return R

    def kv_append(self, k_new, v_new, block_table, query_start_loc, ctx_lens, stream=None):
        R, T = self._check_batch(block_table, query_start_loc, ctx_lens), k_new.shape[0]
        kv_shape = (T, self.cfg.num_kv_heads, self.cfg.head_dim)
        _want(k_new, "k_new", torch.bfloat16, True, kv_shape)
        _want(v_new, "v_new", torch.bfloat16, True, kv_shape)
        self._check(self.lib.ss_kv_append(self._h, _ptr(k_new), _ptr(v_new), _ptr(block_table),
                                          _ptr(query_start_loc), _ptr(ctx_lens), R, T, _stream_ptr(stream)))

    def qkv_rope_append(self, qkv, block_table, query_start_loc, ctx_lens, rope_theta, q_out=None, stream=None):
        """RoPE + QKV split fused into the append (NEXT-4): returns the rotated q [T, Hq, D]."""
        R, T = self._check_batch(block_table, query_start_loc, ctx_lens), qkv.shape[0]
        c = self.cfg
        _want(qkv, "qkv", torch.bfloat16, True, (T, (c.num_q_heads + 2 * c.num_kv_heads) * c.head_dim))
        if q_out is None:
            q_out = torch.empty(T, c.num_q_heads, c.head_dim, dtype=torch.bfloat16, device=qkv.device)
        _want(q_out, "q_out", torch.bfloat16, True, (T, c.num_q_heads, c.head_dim))
        self._check(self.lib.ss_qkv_rope_append(self._h, _ptr(qkv), _ptr(block_table), _ptr(query_start_loc),
                                                _ptr(ctx_lens), R, T, float(rope_theta), _ptr(q_out),
                                                _stream_ptr(stream)))
        return q_out

    def mixed_attention(self, q, block_table, query_start_loc, ctx_lens, scale, out=None, lse=None,
                        stream=None):
        R, T = self._check_batch(block_table, query_start_loc, ctx_lens), q.shape[0]
        q_shape = (T, self.cfg.num_q_heads, self.cfg.head_dim)
        _want(q, "q", torch.bfloat16, True, q_shape)
        if out is None:
            out = torch.empty_like(q)
        _want(out, "out", torch.bfloat16, True, q_shape)
        if lse is not None:
            _want(lse, "lse", torch.float32, True)
            if lse.numel() < T * self.cfg.num_q_heads:
                raise SlidingAttnError("lse: needs at least T * Hq elements")
        self._check(self.lib.ss_mixed_attention(self._h, _ptr(q), _ptr(block_table), _ptr(query_start_loc),
                                                _ptr(ctx_lens), R, T, float(scale), _ptr(out), _ptr(lse),
                                                self.workspace.data_ptr(), self.workspace_bytes,
                                                _stream_ptr(stream)))
        return out

    # ---- aids ----------------------------------------------------------------------------------
    def build_worklist(self, query_start_loc, ctx_lens, stream=None):
        R = ctx_lens.shape[0]
        T = int(self.cfg.max_tokens)
        counts = (ctypes.c_int32 * 3)()
        self._check(self.lib.ss_build_worklist(self._h, _ptr(query_start_loc), _ptr(ctx_lens), R, T,
                                               self.workspace.data_ptr(), self.workspace_bytes, None, 0,
                                               ctypes.byref(counts), _stream_ptr(stream)))
        n = counts[0] + counts[1]
        items = np.zeros(n, dtype=WORK_ITEM_DTYPE)
        if n:
            self._check(self.lib.ss_build_worklist(self._h, _ptr(query_start_loc), _ptr(ctx_lens), R, T,
                                                   self.workspace.data_ptr(), self.workspace_bytes,
                                                   items.ctypes.data, n, ctypes.byref(counts),
                                                   _stream_ptr(stream)))
        return items, tuple(counts)

    def iteration_host(self, q, k_new, v_new, block_table, query_start_loc, ctx_lens, scale, out, stream=None):
        """Host (pinned) tensors in, host tensor out; H2D + append + attention + D2H + sync inside."""
        R, T = self._check_batch(block_table, query_start_loc, ctx_lens, cuda=False), q.shape[0]
        _want(q, "q", torch.bfloat16, False, (T, self.cfg.num_q_heads, self.cfg.head_dim))
        _want(out, "out", torch.bfloat16, False, (T, self.cfg.num_q_heads, self.cfg.head_dim))
        for name, x in (("k_new", k_new), ("v_new", v_new)):
            if x is not None:
                _want(x, name, torch.bfloat16, False, (T, self.cfg.num_kv_heads, self.cfg.head_dim))
        self._check(self.lib.ss_iteration_host(self._h, _ptr(q), _ptr(k_new), _ptr(v_new), _ptr(block_table),
                                               _ptr(query_start_loc), _ptr(ctx_lens), R, T, float(scale),
                                               _ptr(out), _stream_ptr(stream)))
        return out

    def poll_device_error(self, stream=None) -> None:
        """Synchronises; raises SlidingAttnError(SS_ERR_DEVICE_CHECK ...) if a debug check tripped since the last poll."""
        self._check(self.lib.ss_poll_device_error(self._h, _stream_ptr(stream)))

    def reset(self, stream=None) -> None:
        self._check(self.lib.ss_reset(self._h, _stream_ptr(stream)))

    def last_launch_count(self) -> int:
        return int(self.lib.ss_last_launch_count(self._h))

    def set_kernel_timing(self, on: bool):
        self._check(self.lib.ss_set_kernel_timing(self._h, int(on)))

    def last_kernel_time_us(self) -> float:
        v = ctypes.c_float()
        self._check(self.lib.ss_last_kernel_time_us(self._h, ctypes.byref(v)))
        return float(v.value)

    def force_simple_path(self, on: bool):
        self._check(self.lib.ss_debug_force_simple_path(self._h, int(on)))

    def debug_set_param(self, which: int, value: int):
        """1 = main-launch CTAs, 2 = decode-first CTAs, 3 = decode split keys, 4 = force the two-launch route; 0 = automatic."""
        self._check(self.lib.ss_debug_set_param(self._h, int(which), int(value)))


    def stream_read(self, buf: torch.Tensor, stream=None):
        """Measurement aid: one read-only streaming pass over a contiguous CUDA tensor (bench.py's HBM read peak)."""
        assert buf.is_cuda and buf.is_contiguous()
        self._check(self.lib.ss_debug_stream_read(self._h, buf.data_ptr(), buf.numel() * buf.element_size(),
                                                  _stream_ptr(stream)))

    def set_trace(self, buf: Optional[torch.Tensor], words_per_cta: int = 0):
        """Per-CTA timeline of the main launch into a CUDA int64 tensor [num_ctas, words_per_cta]; None = off."""
        self._trace_buf = buf
        self._check(self.lib.ss_debug_set_trace(self._h, _ptr(buf), int(words_per_cta)))


def kv_append(handle: SlidingAttn, k_new, v_new, block_table, query_start_loc, ctx_lens, stream=None):
    """north_star kv_append(k_new, v_new, block_table, slot offsets): slot offsets = ctx_lens + query_start_loc."""
    return handle.kv_append(k_new, v_new, block_table, query_start_loc, ctx_lens, stream)


def mixed_attention(handle: SlidingAttn, q, block_table, query_start_loc, ctx_lens, scale, out=None,
                    lse=None, stream=None):
    """north_star mixed_attention(q, k_cache, v_cache, block_table, query_start_loc, ctx_lens, scale, out);
    the caches are the ones the handle was created on."""
    return handle.mixed_attention(q, block_table, query_start_loc, ctx_lens, scale, out, lse, stream)


STATIC_SCRATCH_BYTES = 8 << 20      # SS_STATIC_SCRATCH_BYTES


def mixed_attention_static(k_cache, v_cache, q, block_table, query_start_loc, ctx_lens, scale, max_requests=None,
                           max_tokens=None, out=None, lse=None, stream=None):
    """ss_mixed_attention_static: mixed_attention with no handle and no workspace, for callers that cannot allocate
    device memory (an engine whose KV cache already owns all of HBM, code inside another framework's pool).  The
    scratch is a STATIC_SCRATCH_BYTES array inside the library, shared by every call on the device: calls must not
    overlap on the GPU, and a config needing more raises SlidingAttnError (SS_ERR_WORKSPACE_TOO_SMALL).  bf16 caches
    only.  The binding itself allocates `out` only when the caller does not pass one - pass `out` to allocate nothing."""
    lib = load()
    if not (k_cache.is_cuda and k_cache.dtype == torch.bfloat16):
        raise SlidingAttnError("k_cache: expected a CUDA bfloat16 tensor")
    P, Hkv, page, D = k_cache.shape
    _want(v_cache, "v_cache", torch.bfloat16, True, k_cache.shape)
    R, T, Hq = ctx_lens.shape[0], q.shape[0], q.shape[1]
    _want(q, "q", torch.bfloat16, True, (T, Hq, D))
    _want(ctx_lens, "ctx_lens", torch.int32, True, (R,))
    _want(query_start_loc, "query_start_loc", torch.int32, True, (R + 1,))
    _want(block_table, "block_table", torch.int32, True, (R, block_table.shape[1]))
    if out is None:
        out = torch.empty_like(q)
    _want(out, "out", torch.bfloat16, True, (T, Hq, D))
    if lse is not None:
        _want(lse, "lse", torch.float32, True)
        if lse.numel() < T * Hq:
            raise SlidingAttnError("lse: needs at least T * Hq elements")
    cfg = ss_config(Hq, Hkv, D, page, P, max(max_requests or R, 1), max(max_tokens or T, 1), block_table.shape[1], 0)
    msg = ctypes.create_string_buffer(512)
    rc = lib.ss_mixed_attention_static(ctypes.byref(cfg), k_cache.data_ptr(), v_cache.data_ptr(), _ptr(q),
                                       _ptr(block_table), _ptr(query_start_loc), _ptr(ctx_lens), R, T, float(scale),
                                       _ptr(out), _ptr(lse), _stream_ptr(stream), msg, len(msg))
    if rc != SS_OK:
        err = SlidingAttnError(f"{lib.ss_status_string(rc).decode()} ({rc}) {msg.value.decode()}")
        err.status = rc
        raise err
    return out


def handle_for(batch, tensors, extra_tokens: int = 0, debug_checks: bool = False, fp8_caches=None, kv_scales=None) -> SlidingAttn:
    """Convenience: a handle sized for one workloads.Batch (fp8_caches = (k_codes, v_codes) uint8 tensors for an FP8 handle)."""
    kc, vc = fp8_caches if fp8_caches is not None else (tensors.k_cache, tensors.v_cache)
    return SlidingAttn(batch.num_q_heads, batch.num_kv_heads, batch.head_dim, kc, vc,
                       max_requests=max(batch.R, 1), max_tokens=max(batch.T + extra_tokens, 1),
                       max_pages_per_req=batch.max_pages_per_req, debug_checks=debug_checks, kv_scales=kv_scales)
