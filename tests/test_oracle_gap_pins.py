"""Pins for the oracle's reading of `gap_slots` (reading A18; include/slack.h token -> slot rule; PAPER.md P:86
"preserves the first few chunks as a global sink and keeps KV entries only for the most recent W chunks").

A bounded sink + local cache DROPS the tokens between the sink and the window: they leave the numbering, their pages
leave the table, and the hole that remains inside partially used pages is `gap_slots`.  Pinned against things other than
the oracle's own position formula:
* pure-Python brute force with its own index arithmetic (tests/test_oracle_pins.py brute_force);
* the closed form K = 0 -> mean of V over the visible tokens, V placed in the pool by hand-written slot arithmetic;
* the defining property: a stream whose out-of-window tokens were dropped (pages removed, gap set) gives bit-identical
  results to the same stream holding everything (the window hides those tokens anyway);
* the append writes behind the hole (read back through hand-written arithmetic, nothing else changes).
CPU only."""
import numpy as np
import pytest

import oracle
from paper_2606_15319_b200 import workloads as W
from test_oracle_pins import brute_force


def gapped(seed, dtype="f32", P=4, H=2, D=4, sink=3, gap=6, held_local=9, q_len=5, window=11, base=1):
    """One stream: `sink` sink tokens, a hole of `gap` slots, then held_local + q_len tokens; random page ids."""
    rng = np.random.default_rng(seed)
    cache_len = sink + held_local
    end_pos = base + gap + cache_len + q_len
    n_tab = -(-end_pos // P)
    n_pages = n_tab + 3
    table = rng.permutation(n_pages)[:n_tab].astype(np.int32)
    s = W.StreamSpec(q_len, cache_len, base, window, sink, table, gap)
    store = np.float32 if dtype == "f32" else np.uint16
    draw = lambda n: W._draw(rng, (n, H, D), 1.0, dtype)
    k_all, v_all = draw(cache_len + q_len), draw(cache_len + q_len)
    kp = np.full((n_pages, H, P, D), np.nan if dtype == "f32" else 0x7FC1, dtype=store)
    vp = kp.copy()
    for t in range(cache_len + q_len):                     # hand-written slot arithmetic (not the oracle's)
        pos = base + t if t < sink else base + gap + t
        kp[table[pos // P], :, pos % P, :] = k_all[t]
        vp[table[pos // P], :, pos % P, :] = v_all[t]
    w = W.Workload("gapped", dtype, H, D, P, n_pages, 0.37, [s], draw(q_len), k_all[cache_len:], v_all[cache_len:],
                   [k_all[:cache_len]], [v_all[:cache_len]], seed)
    return w, kp, vp


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("gap,window", [(6, 11), (1, 0), (9, 5), (4, 14), (0, 11)])
def test_brute_force_with_gap(dtype, gap, window):
    w, kp, vp = gapped(3, dtype=dtype, gap=gap, window=window)
    out, lse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    bo, bl = brute_force(w, kp, vp)
    for (r, h), vec in bo:
        np.testing.assert_allclose(out[r, h], vec, rtol=1e-13, atol=1e-15)
    for (r, h), val in bl:
        assert abs(lse[h, r] - val) < 1e-13


@pytest.mark.parametrize("gap", [0, 2, 7])
@pytest.mark.parametrize("window", [0, 5, 8, 14, 17, 40])
def test_k_zero_gives_mean_over_sink_and_window(gap, window):
    w, kp, vp = gapped(5, gap=gap, window=window)
    kp[...] = np.where(np.isnan(kp), np.nan, 0.0)          # K = 0 wherever a token lives; unowned slots stay NaN
    s = w.streams[0]
    n = s.cache_len + s.q_len
    lo = max(0, n - window) if window else 0
    keys = [t for t in range(n) if t < s.sink_len or t >= max(lo, s.sink_len)]
    v_all = np.concatenate([w.v_prior[0], w.v_new]).astype(np.float64)
    out, lse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    np.testing.assert_allclose(out, np.broadcast_to(v_all[keys].mean(axis=0), out.shape), rtol=1e-14, atol=1e-15)
    np.testing.assert_allclose(lse, np.log(len(keys)), rtol=1e-14)


@pytest.mark.parametrize("P", [4, 8])
@pytest.mark.parametrize("cut", ["pages", "tokens"])
def test_dropping_out_of_window_tokens_changes_nothing(P, cut):
    """Full stream (everything held, gap 0) vs the same stream after the tokens between sink and window were dropped."""
    rng = np.random.default_rng(11)
    H, D, sink, window, q_len, hist = 2, 4, 5, 13, 6, 41
    n = hist + q_len
    table = rng.permutation(-(-n // P) + 2)[:-(-n // P)].astype(np.int32)
    n_pages = int(table.max()) + 3
    full = W.StreamSpec(q_len, hist, 0, window, sink, table)
    k_all = rng.standard_normal((n, H, D)).astype(np.float32)
    v_all = rng.standard_normal((n, H, D)).astype(np.float32)
    q = rng.standard_normal((q_len, H, D)).astype(np.float32)
    kp = np.full((n_pages, H, P, D), np.nan, np.float32)
    vp = kp.copy()
    oracle.kv_append(kp, vp, [W.StreamSpec(n, 0, 0, 0, 0, table)], k_all, v_all)
    want, want_lse = oracle.chunk_attention(kp, vp, [full], q, 0.5, "f32")
    # drop by hand: pages wholly inside (sink, lo) leave the table; the numbering closes up
    lo = n - window
    first_free = -(-sink // P)
    keep_page = lo // P
    k_pages = max(0, keep_page - first_free)
    keep_pos = lo if cut == "tokens" else max(sink, keep_page * P if k_pages else sink)
    dropped = keep_pos - sink
    new_table = np.concatenate([table[:first_free], table[first_free + k_pages:]])
    gap = keep_pos - k_pages * P - sink
    for page in table[first_free:first_free + k_pages]:   # recycled pages get poisoned: nobody may read them
        kp[page] = np.nan
        vp[page] = np.nan
    trimmed = W.StreamSpec(q_len, hist - dropped, 0, window, sink, new_table, gap)
    got, got_lse = oracle.chunk_attention(kp, vp, [trimmed], q, 0.5, "f32")
    assert np.array_equal(got, want) and np.array_equal(got_lse, want_lse)


def test_append_lands_behind_the_hole():
    w, kp, vp = gapped(7, gap=6)
    s = w.streams[0]
    k0, v0 = kp.copy(), vp.copy()
    new_k = (np.arange(s.q_len * w.n_heads * w.head_dim, dtype=np.float32) + 1000).reshape(s.q_len, w.n_heads, w.head_dim)
    oracle.kv_append(kp, vp, [s], new_k, -new_k)
    for i in range(s.q_len):
        pos = s.base + s.gap_slots + s.cache_len + i
        page, slot = s.page_table[pos // w.page_size], pos % w.page_size
        assert np.array_equal(kp[page, :, slot, :], new_k[i]) and np.array_equal(vp[page, :, slot, :], -new_k[i])
        k0[page, :, slot, :] = new_k[i]
        v0[page, :, slot, :] = -new_k[i]
    assert np.array_equal(kp, k0, equal_nan=True) and np.array_equal(vp, v0, equal_nan=True)
