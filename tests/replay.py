"""Test-side model of a stream's WHOLE history, independent of any paging (uses only numpy + oracle/).

The pager (slack_cache_*, A0 / A5) and the kernels see a stream through a bounded, paged, re-numbered cache; the paper's
statement of what a chunk attends to is about the stream itself ("appended to a rolling KV cache for
subsequent chunks", "preserves the first few chunks as a global sink and keeps KV entries only for the most recent W
chunks").  TrueStream keeps every token a stream ever produced and answers, for the chunk being generated, (a) which
TRUE token indices are visible and (b) what the attention output is, by running the oracle on an unpaged private copy
(identity page table, base 0, no gap, all earlier tokens cached).  Neither answer touches a descriptor made by the pager.
"""
from __future__ import annotations

import numpy as np

import oracle
from paper_2606_15319_b200 import workloads as W


class TrueStream:
    def __init__(self, window: int, sink: int, n_heads: int, head_dim: int, dtype: str, seed: int, amp: float = 0.5):
        self.window, self.sink = window, sink
        self.H, self.D, self.dtype = n_heads, head_dim, dtype
        self.rng = np.random.default_rng(seed)
        self.amp = amp
        store = np.uint16 if dtype == "bf16" else np.float32
        self.k = np.zeros((0, n_heads, head_dim), dtype=store)   # committed tokens, true order
        self.v = np.zeros((0, n_heads, head_dim), dtype=store)

    @property
    def committed(self) -> int:
        return int(self.k.shape[0])

    def draw(self, q_len: int):
        """Seeded Q / K_new / V_new of one denoising step of the next chunk (storage dtype)."""
        d = lambda: W._draw(self.rng, (q_len, self.H, self.D), self.amp, self.dtype)
        return d(), d(), d()

    def visible_true(self, q_len: int) -> np.ndarray:
        """True token indices the chunk [N - q_len, N) attends to: the sink and the last `window` tokens (own chunk included)."""
        n = self.committed + q_len
        lo = max(0, n - self.window) if self.window > 0 else 0
        sink = min(self.sink, n)
        return np.concatenate([np.arange(0, sink), np.arange(max(lo, sink), n)]).astype(np.int64)

    def reference_attention(self, q, k_new, v_new, scale: float, page_size: int = 64):
        """Oracle output of the chunk against the whole history, through an identity-paged private pool."""
        q_len = q.shape[0]
        n = self.committed + q_len
        n_pages = -(-n // page_size)
        shape = (max(n_pages, 1), self.H, page_size, self.D)
        kp = np.zeros(shape, dtype=self.k.dtype)
        vp = np.zeros(shape, dtype=self.k.dtype)
        table = np.arange(max(n_pages, 1), dtype=np.int32)
        if self.committed:
            hist = W.StreamSpec(self.committed, 0, 0, 0, 0, table)
            oracle.kv_append(kp, vp, [hist], self.k, self.v)
        s = W.StreamSpec(q_len, self.committed, 0, self.window, self.sink, table)
        oracle.kv_append(kp, vp, [s], k_new, v_new)
        return oracle.chunk_attention(kp, vp, [s], q, scale, self.dtype)

    def commit(self, k_new, v_new) -> None:
        self.k = np.concatenate([self.k, k_new])
        self.v = np.concatenate([self.v, v_new])


def check_cache_invariants(cache, n_pages: int, descs) -> None:
    """No physical page is listed twice over all open streams' tables, and free + owned = pool size."""
    owned = np.concatenate([np.asarray(d.page_table, dtype=np.int64) for d in descs]) if descs else np.zeros(0, np.int64)
    assert owned.size == np.unique(owned).size, "a physical page is owned twice"
    assert owned.size == 0 or (owned.min() >= 0 and owned.max() < n_pages)
    assert cache.free_pages + owned.size == n_pages, "free list + page tables must cover the pool exactly"
