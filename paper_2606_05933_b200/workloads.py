"""Seeded synthetic batches for the mixed prefill+decode attention path.

This module serves BOTH the CUDA path's tests/bench and the fp64 oracle's tests, so it holds none of
the method's arithmetic: it only draws batch metadata ``B = {(c_i, u_i)}`` (§3.2), lays
the requests' logical pages out over a randomly permuted physical pool, and fills tensors with
N(0,1) values rounded to bf16.  The recipes stand in for the paper's ShareGPT / arXiv-summarization
workloads (Table 2), which are not available here; only their shapes are taken
(SURVEY.md §8(d)).

It imports neither ``oracle`` nor the CUDA extension.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np
import torch

PAGE_SIZE = 16


@dataclass
class Batch:
    """One continuous-batching iteration: requests (c_i, u_i) plus their paging metadata."""
    name: str
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    reqs: List[Tuple[int, int]]            # (c_i = q_len, u_i = ctx_len) in batch order
    num_pages: int                          # physical pool size (pages per tensor)
    block_table: np.ndarray                 # [R, max_pages_per_req] int32, unused tail = -1 sentinel
    query_start_loc: np.ndarray             # [R+1] int32
    ctx_lens: np.ndarray                    # [R] int32
    seed: int
    with_append: bool = False               # timed/parity region includes kv_append of the new tokens
    page_size: int = PAGE_SIZE
    meta: dict = field(default_factory=dict)

    @property
    def R(self) -> int:
        return len(self.reqs)

    @property
    def T(self) -> int:
        return int(self.query_start_loc[-1])

    @property
    def max_pages_per_req(self) -> int:
        return int(self.block_table.shape[1])

    @property
    def scale(self) -> float:
        return float(np.float32(1.0 / math.sqrt(self.head_dim)))

    def used_pages(self) -> np.ndarray:
        """Sorted unique physical page ids referenced by the block table."""
        ids = []
        for r, (c, u) in enumerate(self.reqs):
            n = -(-(c + u) // self.page_size)
            ids.append(self.block_table[r, :n])
        if not ids:
            return np.zeros((0,), dtype=np.int64)
        return np.unique(np.concatenate(ids).astype(np.int64))


def make_batch(name: str, Hq: int, Hkv: int, D: int, reqs: Sequence[Tuple[int, int]], seed: int,
               num_pages: Optional[int] = None, with_append: bool = False,
               rng: Optional[np.random.Generator] = None, shuffle_requests: bool = False,
               max_pages_per_req: Optional[int] = None, page_size: int = PAGE_SIZE,
               meta: Optional[dict] = None) -> Batch:
    """Assign physical pages: a random permutation of the pool consumed sequentially, so consecutive
    logical pages of a request are never adjacent in HBM."""
    rng = rng if rng is not None else np.random.default_rng(seed)
    reqs = [(int(c), int(u)) for c, u in reqs]
    if shuffle_requests and len(reqs) > 1:
        order = rng.permutation(len(reqs))
        reqs = [reqs[i] for i in order]
    need = [-(-(c + u) // page_size) for c, u in reqs]
    total = int(sum(need))
    if num_pages is None:
        num_pages = max(2 * total, 4)
    if total > num_pages:
        raise ValueError(f"pool too small: need {total} pages, have {num_pages}")
    mp = max(max(need, default=1), 1) if max_pages_per_req is None else max_pages_per_req
    perm = rng.permutation(num_pages)
    bt = np.full((len(reqs), mp), -1, dtype=np.int32)
    cur = 0
    for r, n in enumerate(need):
        bt[r, :n] = perm[cur:cur + n]
        cur += n
    qsl = np.zeros(len(reqs) + 1, dtype=np.int32)
    qsl[1:] = np.cumsum([c for c, _ in reqs])
    ctx = np.array([u for _, u in reqs], dtype=np.int32).reshape(len(reqs))
    return Batch(name, Hq, Hkv, D, reqs, int(num_pages), bt, qsl, ctx, seed, with_append,
                 page_size, dict(meta or {}))


# --------------------------------------------------------------------------------------------
# BASELINE.json configs (C1..C5) and the scene-edge points of SURVEY.md §8(d)
# --------------------------------------------------------------------------------------------
LOGNORMAL_SIGMA = 0.75       # not given by BASELINE.json; reading stated in DESIGN.md

# Layer shapes (Hq, Hkv, D) of the models the paper serves ("Llama3-8B and Qwen2.5-7B", tensor parallel
# degree 2 on its 2-GPU boxes), from the public model configs; SURVEY.md section 8(f) NEXT-3.  Qwen2.5-7B has 28 query
# and 4 KV heads: G = 7, the first non-power-of-two group (TP2 slice: 14/2, also G = 7).
MODEL_SHAPES = {
    "llama3-8b": (32, 8, 128), "llama3-70b": (64, 8, 128), "qwen2.5-7b": (28, 4, 128),
    "llama3-8b-tp2": (16, 4, 128), "qwen2.5-7b-tp2": (14, 2, 128),
}


def _lognormal_ctx(rng, median, size, cap):
    return np.clip(np.rint(rng.lognormal(math.log(median), LOGNORMAL_SIGMA, size=size)), 1, cap
                   ).astype(np.int64)


def config_tiny(seed: int = 1) -> Batch:
    """C1: 4/4/64, one 64-token chunk on 32 cached + decodes at ctx 17, 40, 100; 64-page pool."""
    return make_batch("C1-tiny", 4, 4, 64, [(64, 32), (1, 17), (1, 40), (1, 100)], seed,
                      num_pages=64, with_append=True)


def config_c2(seed: int = 2, shuffle: bool = False) -> Batch:
    """C2: Llama-3-8B-shaped layer, 512-token chunk at ctx 1024 + 64 decodes ctx U{512..4096}."""
    rng = np.random.default_rng(seed)
    dec = rng.integers(512, 4096, size=64, endpoint=True)
    reqs = [(512, 1024)] + [(1, int(u)) for u in dec]
    return make_batch("C2-8B-mixed", 32, 8, 128, reqs, seed, rng=rng, shuffle_requests=shuffle)


def c3_split(C: int, n: int) -> List[int]:
    return [C // n + (1 if i < C % n else 0) for i in range(n)]


def config_c3(C: int, n: int, N_d: int, ctx_median: int = 1500, shuffle: bool = False,
              model: str = "llama3-8b") -> Batch:
    """C3 grid point: chunk budget C over n prefill requests (ctx U{0..4096}) + N_d decodes
    (ctx lognormal, median 1500 unless swept, cap 8192).  C may be 0 (pure decode).  `model` picks the layer shape
    (BASELINE.json configs[2] is the Llama-3-8B shape; the other shapes reuse the recipe with their own seeds)."""
    seed = 3000 + (100 if N_d == 128 else 0) + (10 * int(round(math.log2(C / 256))) if C > 0 else 90) + n
    if ctx_median != 1500:
        seed += 7 * ctx_median
    if model != "llama3-8b":
        seed += 100000 * (1 + sorted(MODEL_SHAPES).index(model))
    Hq, Hkv, D = MODEL_SHAPES[model]
    rng = np.random.default_rng(seed)
    pu = rng.integers(0, 4096, size=n, endpoint=True)
    du = _lognormal_ctx(rng, ctx_median, N_d, 8192)
    reqs = ([(c, int(u)) for c, u in zip(c3_split(C, n), pu)] if C > 0 else []) + \
           [(1, int(u)) for u in du]
    tag = "" if model == "llama3-8b" else f"-{model}"
    return make_batch(f"C3-C{C}-n{n}-Nd{N_d}-m{ctx_median}{tag}", Hq, Hkv, D, reqs, seed, rng=rng,
                      shuffle_requests=shuffle,
                      meta={"chunk": C, "n_prefill": n if C > 0 else 0, "n_decode": N_d,
                            "ctx_median": ctx_median})


def config_dense(C: int, n: int, N_d: int, ctx_median: int = 1500) -> Batch:
    """Extra points of the latency surface between the C3 grid lines (same recipe as config_c3, own seeds): any chunk
    budget C >= 0 over n prefill requests (ctx U{0..4096}) + N_d >= 0 decodes (ctx lognormal, cap 8192)."""
    seed = 500000 + 17 * C + 1009 * n + 31 * N_d + 7 * ctx_median
    rng = np.random.default_rng(seed)
    pu = rng.integers(0, 4096, size=max(n, 1), endpoint=True)
    du = _lognormal_ctx(rng, ctx_median, N_d, 8192) if N_d > 0 else np.zeros(0, dtype=np.int64)
    reqs = ([(c, int(u)) for c, u in zip(c3_split(C, n), pu) if c > 0] if C > 0 else []) + [(1, int(u)) for u in du]
    return make_batch(f"DN-C{C}-n{n}-Nd{N_d}-m{ctx_median}", 32, 8, 128, reqs, seed, rng=rng,
                      meta={"chunk": C, "n_prefill": n if C > 0 else 0, "n_decode": N_d, "ctx_median": ctx_median})


def config_c4(seed: int = 4, num_requests: int = 256, pool_pages: int = 610352) -> Batch:
    """C4: 256 decodes, ctx U{1024..16384}, pages scattered over a 2 x 20 GB pool."""
    rng = np.random.default_rng(seed)
    dec = rng.integers(1024, 16384, size=num_requests, endpoint=True)
    return make_batch("C4-decode-heavy", 32, 8, 128, [(1, int(u)) for u in dec], seed,
                      num_pages=pool_pages, rng=rng)


def config_c5(seed: int = 5, shuffle: bool = False) -> Batch:
    """C5: Llama-3-70B-shaped layer, 2x1024 chunk tokens at ctx 0 and 6000 + 192 decodes lognormal
    (median 4000, cap 32768), with kv_append of the 2240 new tokens."""
    rng = np.random.default_rng(seed)
    dec = _lognormal_ctx(rng, 4000, 192, 32768)
    reqs = [(1024, 0), (1024, 6000)] + [(1, int(u)) for u in dec]
    return make_batch("C5-70B-mixed", 64, 8, 128, reqs, seed, rng=rng, with_append=True,
                      shuffle_requests=shuffle)


def config_model_mixed(model: str, seed: int = 6, chunk: int = 512, chunk_ctx: int = 1024, n_decode: int = 64,
                       shuffle: bool = False) -> Batch:
    """C2's recipe (one chunk + decodes ctx U{512..4096}) on another model's layer shape."""
    Hq, Hkv, D = MODEL_SHAPES[model]
    rng = np.random.default_rng(seed)
    dec = rng.integers(512, 4096, size=n_decode, endpoint=True)
    reqs = [(chunk, chunk_ctx)] + [(1, int(u)) for u in dec]
    return make_batch(f"MX-{model}", Hq, Hkv, D, reqs, seed, rng=rng, shuffle_requests=shuffle, with_append=True)


SCENE_EDGES = {
    "PP-a": (32, 8, [(2048, 0)]),
    "PP-b": (32, 8, [(2048, 4096)]),
    "PP-c": (32, 8, [(2048, 8192)]),
    "PP-d": (32, 8, [(512, 4096)]),
    "PP-e": (32, 8, [(8192, 0)]),
    "PP-f": (64, 8, [(1024, 0), (1024, 6000)]),
    "PP-g": (64, 8, [(4096, 4096)]),
    "PP-q": (28, 4, [(2048, 4096)]),        # PP-b on the Qwen2.5-7B shape (G = 7)
}


def config_scene_edge(name: str) -> Batch:
    Hq, Hkv, reqs = SCENE_EDGES[name]
    seed = 7000 + sorted(SCENE_EDGES).index(name)
    return make_batch(name, Hq, Hkv, 128, reqs, seed)


def config_decode_only(name: str) -> Batch:
    """PD-* scene edges: the decode set of a named mixed config alone (C = 0).
    PD-C2 / PD-C5: the decodes of C2 / C5; PD-32 / PD-128: the C3 decode sets (median 1500)."""
    if name == "PD-C2":
        src = config_c2()
    elif name == "PD-C5":
        src = config_c5()
    elif name in ("PD-32", "PD-128"):
        return config_c3(0, 1, int(name[3:]))
    else:
        raise KeyError(name)
    reqs = [(c, u) for c, u in src.reqs if c == 1]
    return make_batch(name, src.num_q_heads, src.num_kv_heads, src.head_dim, reqs, 7100 + len(reqs))


def random_batch(seed: int, Hq: int = 8, Hkv: int = 2, D: int = 128, n_prefill: int = 2,
                 n_decode: int = 5, max_c: int = 200, max_u: int = 600, n_empty: int = 1,
                 with_append: bool = True) -> Batch:
    """Small ragged batch for property tests: prefill chunks (c>1), decodes (c==1), c==0 requests,
    u==0 cases, lengths straddling page (16) and tile (128) edges, shuffled request order."""
    rng = np.random.default_rng(seed)
    edge = [1, 15, 16, 17, 31, 32, 33, 127, 128, 129, 255, 256, 257]
    reqs = []
    for _ in range(n_prefill):
        c = int(rng.choice(edge[1:])) if rng.random() < 0.5 else int(rng.integers(2, max_c, endpoint=True))
        u = 0 if rng.random() < 0.25 else (int(rng.choice(edge)) if rng.random() < 0.4
                                          else int(rng.integers(1, max_u, endpoint=True)))
        reqs.append((min(c, max_c), min(u, max_u)))
    for _ in range(n_decode):
        u = 0 if rng.random() < 0.15 else (int(rng.choice(edge)) if rng.random() < 0.4
                                          else int(rng.integers(1, max_u, endpoint=True)))
        reqs.append((1, min(u, max_u)))
    for _ in range(n_empty):
        reqs.append((0, int(rng.integers(0, max_u, endpoint=True))))
    return make_batch(f"rand-{seed}", Hq, Hkv, D, reqs, seed, rng=rng, shuffle_requests=True,
                      with_append=with_append)


# --------------------------------------------------------------------------------------------
# tensors
# --------------------------------------------------------------------------------------------
@dataclass
class Tensors:
    q: torch.Tensor          # [T,Hq,D] bf16
    k_new: torch.Tensor      # [T,Hkv,D] bf16
    v_new: torch.Tensor      # [T,Hkv,D] bf16
    k_cache: torch.Tensor    # [P,Hkv,page,D] bf16
    v_cache: torch.Tensor    # [P,Hkv,page,D] bf16


def _randn_bf16(shape, gen: torch.Generator, device, chunk_elems: int = 1 << 27) -> torch.Tensor:
    n = int(np.prod(shape)) if len(shape) else 1
    out = torch.empty(n, dtype=torch.bfloat16, device=device)
    for s in range(0, n, chunk_elems):
        e = min(n, s + chunk_elems)
        out[s:e] = torch.randn(e - s, generator=gen, device=device, dtype=torch.float32).to(torch.bfloat16)
    return out.view(*shape)


def make_fp8_caches(b: Batch, device, seed_offset: int = 0):
    """FP8 E4M3 cache pools for timing runs (SS_FLAG_KV_FP8): uniformly random codes, the two NaN codes (0x7F, 0xFF)
    mapped to zero, and per kv head fp32 scales in [0.008, 0.02] (code magnitudes are log-uniform over 2^-9 .. 448, so
    values reach ~ +-9).  Pure input generation: no quantisation arithmetic lives here.
    Returns (k_codes, v_codes, k_scale, v_scale), caches uint8 [P,Hkv,page,D], scales float32 [Hkv] on `device`."""
    device = torch.device(device)
    gen = torch.Generator(device=device)
    gen.manual_seed(1000003 * b.seed + 29 + seed_offset)
    shape = (b.num_pages, b.num_kv_heads, b.page_size, b.head_dim)
    caches = []
    for _ in range(2):
        c = torch.empty(shape, dtype=torch.uint8, device=device)
        flat = c.view(-1)
        for s in range(0, flat.numel(), 1 << 28):
            e = min(flat.numel(), s + (1 << 28))
            r = torch.randint(0, 256, (e - s,), generator=gen, device=device, dtype=torch.int16)
            r[(r & 0x7F) == 0x7F] = 0
            flat[s:e] = r.to(torch.uint8)
        caches.append(c)
    rng = np.random.default_rng(b.seed + 4242 + seed_offset)
    ks = torch.from_numpy(rng.uniform(0.008, 0.02, size=b.num_kv_heads).astype(np.float32)).to(device)
    vs = torch.from_numpy(rng.uniform(0.008, 0.02, size=b.num_kv_heads).astype(np.float32)).to(device)
    return caches[0], caches[1], ks, vs


def make_tensors(b: Batch, device="cpu", poison_unused: bool = False, caches: bool = True) -> Tensors:
    """N(0,1) bf16 everywhere (every cache page, used or not).  With ``poison_unused`` the slots no
    request may read (pages outside every block table, slots past u+c in last pages) get bf16 NaN /
    +-3e38 bit patterns to prove the path never touches them (SURVEY.md §8(c) reading 7).

    For ``with_append`` batches the cache positions u..u+c-1 hold OLD data that kv_append must
    overwrite; otherwise the cache is taken to hold all u+c tokens already."""
    device = torch.device(device)
    gen = torch.Generator(device=device)
    gen.manual_seed(1000003 * b.seed + 17)
    T = max(b.T, 0)
    q = _randn_bf16((T, b.num_q_heads, b.head_dim), gen, device)
    k_new = _randn_bf16((T, b.num_kv_heads, b.head_dim), gen, device)
    v_new = _randn_bf16((T, b.num_kv_heads, b.head_dim), gen, device)
    cshape = (b.num_pages, b.num_kv_heads, b.page_size, b.head_dim)
    if not caches:                                   # FP8 runs bring their own pools (make_fp8_caches)
        return Tensors(q, k_new, v_new, None, None)
    k_cache = _randn_bf16(cshape, gen, device)
    v_cache = _randn_bf16(cshape, gen, device)
    if poison_unused:
        poison_unused_slots(b, k_cache, v_cache)
    return Tensors(q, k_new, v_new, k_cache, v_cache)


_POISON_BITS = (0x7FC0, 0x7F7F, 0xFF7F, 0xFFC1)   # NaN, +3.39e38, -3.39e38, NaN with payload


def poison_unused_slots(b: Batch, k_cache: torch.Tensor, v_cache: torch.Tensor) -> None:
    used = torch.zeros(b.num_pages, b.page_size, dtype=torch.bool)
    for r, (c, u) in enumerate(b.reqs):
        n = c + u
        for lp in range(-(-n // b.page_size)):
            cnt = min(b.page_size, n - lp * b.page_size)
            used[int(b.block_table[r, lp]), :cnt] = True
    mask = (~used).to(k_cache.device)[:, None, :, None]       # [P,1,page,1]
    pat = torch.tensor(_POISON_BITS, dtype=torch.int32).to(torch.int16)
    idx = torch.arange(b.head_dim) % len(_POISON_BITS)
    row = pat[idx].to(k_cache.device)
    for cache in (k_cache, v_cache):
        bits = cache.view(torch.int16)
        bits.copy_(torch.where(mask, row.view(1, 1, 1, -1), bits))


def to_u16(t: torch.Tensor) -> np.ndarray:
    """bf16 tensor -> numpy uint16 bit patterns on host (exact)."""
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)


def compact_pool(b: Batch, *caches: torch.Tensor):
    """Gather only the pages named in the block table to the host and remap the table, so the oracle
    can run on batches whose pool (e.g. C4's 40 GB) does not fit host memory.  Pure data movement;
    legal because attention is invariant to a physical-page permutation (pinned in the oracle tests).

    Returns (remapped_block_table int32 [R,max_pages], [uint16 arrays [n_used,Hkv,page,D] ...])."""
    used = b.used_pages()
    remap = np.full(b.num_pages, -1, dtype=np.int64)
    remap[used] = np.arange(used.shape[0])
    bt = b.block_table.astype(np.int64)
    new_bt = np.where(bt >= 0, remap[np.clip(bt, 0, None)], -1).astype(np.int32)
    outs = []
    for cache in caches:
        idx = torch.from_numpy(used).to(cache.device)
        outs.append(to_u16(cache.index_select(0, idx)))
    return new_bt, outs
