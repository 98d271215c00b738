"""slidingattn for B200 (sm_100a): one continuous-batching iteration's mixed chunked-prefill + decode
attention over a paged KV cache — the batch execution that SlidingServe's latency predictor models
(PAPER.md:99 §3.1 step 9, :107 §3.2).  Hand-written CUDA behind a C ABI (include/slidingattn.h);
this package is only the ctypes binding plus host-side bookkeeping.  There is no CPU fallback: the
binding raises if the compiled library is missing."""
__all__ = ["features", "binding", "workloads", "accounting"]
