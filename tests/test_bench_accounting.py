"""CPU checks of bench.py's bookkeeping (no GPU, no timing): the flop / byte counts the reported TFLOP/s and GB/s are
built from must equal brute-force counts on small workloads (visible keys only; block-sparse: selected
(query, key) pairs only)."""
import numpy as np

import bench
from paper_2606_15319_b200 import metrics, workloads as W


def brute_pairs(w, masks=None, rows=None):
    total = 0
    for si, s in enumerate(w.streams):
        n = s.cache_len + s.q_len
        lo = max(0, n - s.window) if s.window > 0 else 0
        sink = min(s.sink_len, n)
        vis = [t for t in range(n) if t < sink or t >= max(lo, sink)]
        r = range(s.q_len) if rows is None else [int(x) for x in rows[si]]
        for i in r:
            if masks is None:
                total += len(vis) * w.n_heads
            else:
                m = masks[si]
                for h in range(w.n_heads):
                    total += sum(1 for t in vis if m[h, i // W.MASK_BLOCK_Q, (s.base + t) // W.MASK_BLOCK_K])
    return total


def test_dense_flops_and_bytes():
    for w in (W.small_ragged(head_dim=16), W.sink_ragged(head_dim=16)):
        assert metrics.attention_flops(w.streams, w.n_heads, w.head_dim) == 4.0 * w.head_dim * brute_pairs(w)
        vk = metrics.visible_keys(w.streams)
        assert metrics.attention_min_bytes(w.streams, w.n_heads, w.head_dim, 2) == \
            sum((2 * s.q_len + 2 * k) * w.n_heads * w.head_dim * 2 for s, k in zip(w.streams, vk))
        assert metrics.append_bytes(w.streams, w.n_heads, w.head_dim, 2) == 8.0 * w.total_q * w.n_heads * w.head_dim


def test_selected_pairs_matches_brute_force():
    w = W.sink_ragged(head_dim=16, seed=4)
    masks = W.random_block_masks(w, 0.6, seed=3)
    assert bench.selected_pairs(w, masks) == brute_pairs(w, masks)
    rows = bench.sample_rows(w.streams, 40)
    assert bench.selected_pairs(w, masks, rows) == brute_pairs(w, masks, rows)
    ones = [np.ones_like(m) if m is not None else None for m in masks]
    assert 4.0 * w.head_dim * bench.selected_pairs(w, ones) == metrics.attention_flops(w.streams, w.n_heads, w.head_dim)


def test_sample_rows_are_valid_and_seeded():
    w = W.small_ragged(head_dim=16)
    a, b = bench.sample_rows(w.streams, 64), bench.sample_rows(w.streams, 64)
    for s, r, r2 in zip(w.streams, a, b):
        assert np.array_equal(r, r2) and len(np.unique(r)) == len(r)
        assert (len(r) == 0) == (s.q_len == 0) and all(0 <= x < s.q_len for x in r)
