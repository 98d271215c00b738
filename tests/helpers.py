"""Test-only helpers: independent de-paging and bf16 widening (via torch, a library routine), used to
pin the oracle against dense textbook formulas.  Nothing here is imported by the product."""
import numpy as np
import torch

from paper_2606_05933_b200 import workloads as wl


def u16_to_f64(a: np.ndarray) -> np.ndarray:
    """uint16 bf16 bits -> float64 through torch's own bf16 type (independent of the oracle's shift)."""
    t = torch.from_numpy(a.astype(np.int16, copy=True).reshape(-1)).view(torch.bfloat16)
    return t.to(torch.float64).numpy().reshape(a.shape)


def f64_to_u16(a: np.ndarray) -> np.ndarray:
    t = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16).reshape(a.shape)


def depage(b: wl.Batch, cache_u16: np.ndarray, r: int, n: int) -> np.ndarray:
    """Dense [n, Hkv, D] float64 view of request r's first n cached tokens.  cache: [P,Hkv,page,D]."""
    out = np.empty((n, b.num_kv_heads, b.head_dim), dtype=np.float64)
    for t in range(n):
        page = int(b.block_table[r, t // b.page_size])
        out[t] = u16_to_f64(cache_u16[page, :, t % b.page_size, :])
    return out


def host_arrays(b: wl.Batch, t: wl.Tensors):
    return dict(q=wl.to_u16(t.q), k_new=wl.to_u16(t.k_new), v_new=wl.to_u16(t.v_new),
                k_cache=wl.to_u16(t.k_cache), v_cache=wl.to_u16(t.v_cache))


def oracle_run(b: wl.Batch, arrs, scale=None, rows=None, append=None):
    """append (default b.with_append) + attention through the oracle on host arrays (copies caches)."""
    import oracle
    k = arrs["k_cache"].copy()
    v = arrs["v_cache"].copy()
    if b.with_append if append is None else append:
        oracle.kv_append(k, v, arrs["k_new"], arrs["v_new"], b.block_table, b.query_start_loc, b.ctx_lens)
    out, lse, pairs = oracle.mixed_attention(arrs["q"], k, v, b.block_table, b.query_start_loc,
                                             b.ctx_lens, b.scale if scale is None else scale, rows=rows)
    return out, lse, pairs, k, v
