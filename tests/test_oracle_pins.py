"""Pins for the fp64 oracle (`oracle/`): every check here is against something OTHER than the oracle's own
formula - pure-Python brute force, closed forms, library routines (torch SDPA, scipy logsumexp), a dense
block-causal mask over the whole sequence, and invariances (SURVEY.md §8(c) "What pins each part").
CPU only; runs in seconds."""
import copy
import math

import numpy as np
import pytest
import scipy.special
import torch

import oracle
from paper_2606_15319_b200 import workloads as W
from helpers import empty_pools, oracle_pools, prior_streams, stream_rows


def tiny(seed=1, dtype="f32", **kw):
    args = dict(dtype=dtype, n_heads=2, head_dim=4, page_size=4, q_lens=[5, 3, 1], cache_lens=[6, 0, 9],
                windows=[0, 0, 7], bases=[0, 3, 2], seed=seed, spare_pages=2)
    args.update(kw)
    return W.make_workload("tiny", **args)


# ------------------------------------------------------------------ (i) brute force, written independently
def brute_force(w, k_pool, v_pool):
    """Triple loop in pure Python floats with math.fsum; own index arithmetic (no oracle helpers)."""
    H, D, P = w.n_heads, w.head_dim, w.page_size
    dec = (lambda x: float(np.array([int(x) << 16], dtype=np.uint32).view(np.float32)[0])) if w.dtype == "bf16" \
        else (lambda x: float(x))
    outs, lses, row = [], [], 0
    for s in w.streams:
        n = s.cache_len + s.q_len
        lo = 0
        if s.window > 0 and n - s.window > 0:
            lo = n - s.window
        sink = min(s.sink_len, n)
        keys = [t for t in range(n) if t < sink or t >= max(lo, sink)]
        for i in range(s.q_len):
            for h in range(H):
                qv = [dec(w.q[row + i, h, d]) for d in range(D)]
                logits = []
                vals = []
                for t in keys:
                    pos = s.base + t
                    if t >= s.sink_len:
                        pos += s.gap_slots               # hole behind the sink left by dropped tokens (slack.h)
                    page = int(s.page_table[pos // P])
                    slot = pos % P
                    kv = [dec(k_pool[page, h, slot, d]) for d in range(D)]
                    vals.append([dec(v_pool[page, h, slot, d]) for d in range(D)])
                    logits.append(w.scale * math.fsum(a * b for a, b in zip(qv, kv)))
                mx = max(logits)
                e = [math.exp(x - mx) for x in logits]
                den = math.fsum(e)
                outs.append(((row + i, h), [math.fsum(e[j] * vals[j][d] for j in range(len(keys))) / den
                                            for d in range(D)]))
                lses.append(((row + i, h), mx + math.log(den)))
        row += s.q_len
    return outs, lses


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("sink", [0, 2])
def test_brute_force_tiny(dtype, sink):
    w = tiny(seed=3, dtype=dtype, sink_lens=[sink, 0, sink])
    kp, vp = oracle_pools(w)
    out, lse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    bo, bl = brute_force(w, kp, vp)
    assert len(bo) == w.total_q * w.n_heads
    for (r, h), vec in bo:
        np.testing.assert_allclose(out[r, h], vec, rtol=1e-13, atol=1e-15)
    for (r, h), val in bl:
        assert abs(lse[h, r] - val) < 1e-13


# ------------------------------------------------------------------ closed forms
def _set_all_kv(w, k_val=None, v_val=None):
    """Overwrite K and/or V of every token (prior + new) with a constant array generator."""
    for arrs, val in ((w.k_prior + [w.k_new], k_val), (w.v_prior + [w.v_new], v_val)):
        if val is not None:
            for a in arrs:
                a[...] = val


def test_v_all_ones_gives_ones():           # (ii) softmax rows sum to 1
    w = tiny(seed=5)
    _set_all_kv(w, v_val=1.0)
    kp, vp = oracle_pools(w)
    out, _ = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    np.testing.assert_allclose(out, 1.0, rtol=0, atol=1e-15)


def test_one_hot_v_is_probability_row():    # (iii)
    w = W.make_workload("onehot", dtype="f32", n_heads=1, head_dim=16, page_size=4, q_lens=[4], cache_lens=[9],
                        windows=[0], bases=[1], seed=9)
    n = 13
    eye = np.zeros((n, 1, 16), np.float32)
    eye[np.arange(n), 0, np.arange(n)] = 1.0
    w.v_prior[0][...] = eye[:9]
    w.v_new[...] = eye[9:]
    kp, vp = oracle_pools(w)
    out, lse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    p = out[:, 0, :]
    assert np.all(p[:, :n] > 0) and np.all(p[:, n:] == 0)
    np.testing.assert_allclose(p.sum(axis=1), 1.0, atol=1e-15)
    # the probability row must be softmax of the logits computed by hand in fp64
    k = np.concatenate([w.k_prior[0], w.k_new])[:, 0, :].astype(np.float64)
    s = w.scale * (w.q[:, 0, :].astype(np.float64) @ k.T)
    np.testing.assert_allclose(p[:, :n], scipy.special.softmax(s, axis=1), rtol=1e-13)
    np.testing.assert_allclose(lse[0], scipy.special.logsumexp(s, axis=1), rtol=1e-14)   # LSE pin


@pytest.mark.parametrize("base", [0, 1, 3])
@pytest.mark.parametrize("wsel", ["none", "Lq", "n-1", "n", "n+1", "1"])
def test_k_zero_gives_window_mean(base, wsel):   # (iv) pins lo / base / slot arithmetic
    Lq, Lc = 5, 9
    n = Lq + Lc
    win = {"none": 0, "Lq": Lq, "n-1": n - 1, "n": n, "n+1": n + 1, "1": 1}[wsel]
    w = W.make_workload("k0", dtype="f32", n_heads=2, head_dim=4, page_size=4, q_lens=[Lq], cache_lens=[Lc],
                        windows=[win], bases=[base], seed=21, spare_pages=1)
    _set_all_kv(w, k_val=0.0)
    kp, vp = oracle_pools(w, fill=np.nan)
    out, lse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    v_all = np.concatenate([w.v_prior[0], w.v_new]).astype(np.float64)      # logical order, by construction
    lo = 0 if win == 0 else max(0, n - win)
    want = v_all[lo:n].mean(axis=0)
    for i in range(Lq):
        np.testing.assert_allclose(out[i], want, rtol=1e-14, atol=1e-16)
    np.testing.assert_allclose(lse, math.log(n - lo), rtol=1e-14)
    if wsel == "1":                                                          # (v) single visible key -> out = v
        np.testing.assert_array_equal(out[0], v_all[n - 1])


def test_single_key_returns_v():            # (v) with non-zero K
    w = W.make_workload("one", dtype="bf16", n_heads=2, head_dim=8, page_size=4, q_lens=[1], cache_lens=[0],
                        windows=[0], bases=[2], seed=4)
    kp, vp = oracle_pools(w)
    out, lse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    np.testing.assert_array_equal(out[0], oracle.to_f64(w.v_new[0], "bf16"))


def test_logit_shift_invariance():          # (vi)
    c = 3.25
    w = tiny(seed=8, head_dim=4)
    kp, vp = oracle_pools(w)
    out0, lse0 = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    w2 = copy.deepcopy(w)
    w2.head_dim = 5
    ext = lambda a, val: np.concatenate([a, np.full(a.shape[:2] + (1,), val, np.float32)], axis=2)
    w2.q = ext(w.q, 1.0)
    w2.k_new = ext(w.k_new, c)
    w2.v_new = ext(w.v_new, 0.0)
    w2.k_prior = [ext(a, c) for a in w.k_prior]
    w2.v_prior = [ext(a, 0.0) for a in w.v_prior]
    kp2, vp2 = oracle_pools(w2)
    out1, lse1 = oracle.chunk_attention(kp2, vp2, w2.streams, w2.q, w2.scale, w2.dtype)
    np.testing.assert_allclose(out1[:, :, :4], out0, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(lse1, lse0 + w.scale * c, rtol=1e-13)


# ------------------------------------------------------------------ (vii) library special case
@pytest.mark.parametrize("cfg", ["cfg1", "ragged"])
def test_matches_torch_sdpa_fp64(cfg):
    w = W.config1() if cfg == "cfg1" else W.small_ragged(seed=13, dtype="bf16", head_dim=64, page_size=16)
    for s in w.streams:
        s.window = 0
    kp, vp = oracle_pools(w)
    out, _ = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    dec = lambda a: torch.from_numpy(oracle.to_f64(a, w.dtype))
    for (r0, r1), s, kpri, vpri in zip(stream_rows(w), w.streams, w.k_prior, w.v_prior):
        if s.q_len == 0:
            continue
        q = dec(w.q[r0:r1]).permute(1, 0, 2)
        k = torch.cat([dec(kpri), dec(w.k_new[r0:r1])]).permute(1, 0, 2)
        v = torch.cat([dec(vpri), dec(w.v_new[r0:r1])]).permute(1, 0, 2)
        ref = torch.nn.functional.scaled_dot_product_attention(q, k, v, scale=w.scale).permute(1, 0, 2).numpy()
        np.testing.assert_allclose(out[r0:r1], ref, rtol=1e-11, atol=1e-14)


# ------------------------------------------------------------------ block-causal semantics over the full sequence
@pytest.mark.parametrize("win_chunks", [0, 1, 2, 3])
def test_block_causal_full_sequence_replay(win_chunks):
    """Replay a stream chunk by chunk through the oracle (append, attend) and compare every chunk's rows with
    dense masked softmax over the whole sequence, mask = chunk(j) <= chunk(i) and chunk(j) > chunk(i) - Wc."""
    rng = np.random.default_rng(17)
    C, Lq, H, D, P = 4, 6, 2, 8, 4
    T = C * Lq
    q = rng.standard_normal((T, H, D), dtype=np.float32)
    k = rng.standard_normal((T, H, D), dtype=np.float32)
    v = rng.standard_normal((T, H, D), dtype=np.float32)
    scale = 0.3
    table = rng.permutation(T // P + 2).astype(np.int32)
    kp = np.full((len(table), H, P, D), np.nan, np.float32)
    vp = kp.copy()
    got = np.zeros((T, H, D))
    for c in range(C):
        s = W.StreamSpec(Lq, c * Lq, 1, win_chunks * Lq, 0, table)
        oracle.kv_append(kp, vp, [s], k[c * Lq:(c + 1) * Lq], v[c * Lq:(c + 1) * Lq])
        o, _ = oracle.chunk_attention(kp, vp, [s], q[c * Lq:(c + 1) * Lq], scale, "f32")
        got[c * Lq:(c + 1) * Lq] = o
    chunk = np.arange(T) // Lq
    mask = chunk[None, :] <= chunk[:, None]
    if win_chunks:
        mask &= chunk[None, :] > chunk[:, None] - win_chunks
    for h in range(H):
        s_ = scale * (q[:, h].astype(np.float64) @ k[:, h].astype(np.float64).T)
        s_[~mask] = -np.inf
        want = scipy.special.softmax(s_, axis=1) @ v[:, h].astype(np.float64)
        np.testing.assert_allclose(got[:, h], want, rtol=1e-12, atol=1e-15)


# ------------------------------------------------------------------ page-table gather
def test_page_permutation_invariance_and_poison():
    w = W.small_ragged(seed=19, dtype="bf16", head_dim=16, page_size=16)
    kp, vp = oracle_pools(w)
    out0, lse0 = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    perm = np.random.default_rng(5).permutation(w.n_pages)       # new physical id of old page p is perm[p]
    w2 = copy.deepcopy(w)
    for s in w2.streams:
        s.page_table = perm[s.page_table].astype(np.int32)
    kp2, vp2 = np.empty_like(kp), np.empty_like(vp)
    kp2[perm], vp2[perm] = kp, vp
    out1, lse1 = oracle.chunk_attention(kp2, vp2, w2.streams, w2.q, w2.scale, w2.dtype)
    np.testing.assert_array_equal(out0, out1)
    np.testing.assert_array_equal(lse0, lse1)
    # identity table == shuffled table (same logical data)
    w3 = W.small_ragged(seed=19, dtype="bf16", head_dim=16, page_size=16)
    ident = np.arange(w3.n_pages, dtype=np.int32)
    at = 0
    for s in w3.streams:
        s.page_table = ident[at:at + len(s.page_table)].copy()
        at += len(s.page_table)
    kp3, vp3 = oracle_pools(w3)
    out3, _ = oracle.chunk_attention(kp3, vp3, w3.streams, w3.q, w3.scale, w3.dtype)
    np.testing.assert_array_equal(out0, out3)


def test_unowned_slots_poisoned_with_nan_do_not_leak():
    w = W.small_ragged(seed=23, dtype="f32", head_dim=16, page_size=16)
    kp, vp = oracle_pools(w, fill=np.nan)        # every slot never appended stays NaN
    out, lse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    assert np.all(np.isfinite(out)) and np.all(np.isfinite(lse))
    # window-clipped streams: poisoning the invisible (evicted-but-resident) tokens changes nothing
    w2 = copy.deepcopy(w)
    for s, kpri, vpri in zip(w2.streams, w2.k_prior, w2.v_prior):
        n = s.cache_len + s.q_len
        lo = max(0, n - s.window) if s.window else 0
        kpri[:min(lo, s.cache_len)] = np.nan
        vpri[:min(lo, s.cache_len)] = np.nan
    kp2, vp2 = oracle_pools(w2, fill=np.nan)
    out2, _ = oracle.chunk_attention(kp2, vp2, w2.streams, w2.q, w2.scale, w2.dtype)
    np.testing.assert_array_equal(out, out2)


# ------------------------------------------------------------------ append
@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_append_pins(dtype):
    w = W.small_ragged(seed=29, dtype=dtype, head_dim=8, page_size=16)
    sentinel = 0xABCD if dtype == "bf16" else np.float32(-777.25)
    kp, vp = oracle_pools(w, fill=sentinel, with_new=False)
    kb, vb = kp.copy(), vp.copy()
    oracle.kv_append(kp, vp, w.streams, w.k_new, w.v_new)
    # source bytes == bytes read back through the page table (independent index arithmetic)
    row = 0
    written = np.zeros(kp.shape[:1] + kp.shape[2:3], bool)       # [page, slot]
    for s in w.streams:
        for i in range(s.q_len):
            pos = s.base + s.cache_len + i
            pg, sl = int(s.page_table[pos // w.page_size]), pos % w.page_size
            assert not written[pg, sl]
            written[pg, sl] = True
            np.testing.assert_array_equal(kp[pg, :, sl, :], w.k_new[row + i])
            np.testing.assert_array_equal(vp[pg, :, sl, :], w.v_new[row + i])
        row += s.q_len
    # nothing else was written (whole-pool compare against the pre-append image)
    untouched = ~written
    np.testing.assert_array_equal(kp.transpose(0, 2, 1, 3)[untouched], kb.transpose(0, 2, 1, 3)[untouched])
    np.testing.assert_array_equal(vp.transpose(0, 2, 1, 3)[untouched], vb.transpose(0, 2, 1, 3)[untouched])
    # re-append is idempotent; two halves == at once
    k2, v2 = kp.copy(), vp.copy()
    oracle.kv_append(k2, v2, w.streams, w.k_new, w.v_new)
    np.testing.assert_array_equal(k2, kp)
    k3, v3 = kb.copy(), vb.copy()
    first, second, rows_a, rows_b = [], [], [], []
    for (r0, r1), s in zip(stream_rows(w), w.streams):
        h = s.q_len // 2
        a, b = copy.copy(s), copy.copy(s)
        a.q_len = h
        b.q_len, b.cache_len = s.q_len - h, s.cache_len + h
        first.append(a), second.append(b)
        rows_a.append(np.arange(r0, r0 + h)), rows_b.append(np.arange(r0 + h, r1))
    ia, ib = np.concatenate(rows_a), np.concatenate(rows_b)
    oracle.kv_append(k3, v3, first, w.k_new[ia], w.v_new[ia])
    oracle.kv_append(k3, v3, second, w.k_new[ib], w.v_new[ib])
    np.testing.assert_array_equal(k3, kp)
    np.testing.assert_array_equal(v3, vp)


# ------------------------------------------------------------------ batching
def test_batched_equals_each_stream_alone():
    w = W.small_ragged(seed=31, dtype="bf16", head_dim=16, page_size=16)
    kp, vp = oracle_pools(w)
    out, lse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    for (r0, r1), s in zip(stream_rows(w), w.streams):
        o1, l1 = oracle.chunk_attention(kp, vp, [s], w.q[r0:r1], w.scale, w.dtype)
        np.testing.assert_array_equal(out[r0:r1], o1)
        np.testing.assert_array_equal(lse[:, r0:r1], l1)


def test_row_sampling_is_exact():
    w = W.small_ragged(seed=37, dtype="bf16", head_dim=16, page_size=16)
    kp, vp = oracle_pools(w)
    out, lse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    rows = [np.array([0, s.q_len - 1]) if s.q_len else np.array([], dtype=np.int64) for s in w.streams]
    o2, l2 = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype, rows=rows, row_block=1)
    m = ~np.isnan(o2)
    assert m.sum() == sum(len(np.unique(r)) for r in rows) * w.n_heads * w.head_dim
    np.testing.assert_allclose(o2[m], out[m], rtol=1e-13, atol=1e-16)


# ------------------------------------------------------------------ split-KV merge formula (A4)
def test_lse_merge_equals_unsplit():
    rng = np.random.default_rng(41)
    R, D, Lk = 7, 5, 50
    q, k, v = rng.standard_normal((R, D)), rng.standard_normal((Lk, D)) * 3, rng.standard_normal((Lk, D))
    full, lse_full = oracle.attend_rows(q, k, v, 0.7)
    for cuts in ([0, 50], [0, 1, 50], [0, 13, 14, 37, 50]):
        parts = [oracle.attend_rows(q, k[a:b], v[a:b], 0.7) for a, b in zip(cuts[:-1], cuts[1:])]
        o, l = oracle.lse_merge([p[0] for p in parts], [p[1] for p in parts])
        np.testing.assert_allclose(o, full, rtol=1e-13, atol=1e-15)
        np.testing.assert_allclose(l, lse_full, rtol=1e-14)
    np.testing.assert_allclose(lse_full, scipy.special.logsumexp(0.7 * q @ k.T, axis=1), rtol=1e-14)


# ------------------------------------------------------------------ storage decoding and input rounding
def test_bf16_roundtrip_matches_torch():
    x = np.random.default_rng(43).standard_normal(4096, dtype=np.float32) * 3
    x[:4] = [0.0, -0.0, 1.00390625, 1.01171875]          # ties: round to even
    bits = W.f32_to_bf16_bits(x)
    tb = torch.from_numpy(x).to(torch.bfloat16)
    np.testing.assert_array_equal(bits, tb.view(torch.int16).numpy().view(np.uint16))
    np.testing.assert_array_equal(oracle.to_f64(bits, "bf16"), tb.double().numpy())
    np.testing.assert_array_equal(W.bf16_bits_to_f32(bits), tb.float().numpy())


def test_error_metrics():
    want = np.array([[3.0, 4.0], [np.nan, np.nan]])
    got = np.array([[3.0, 4.5], [99.0, 99.0]])
    ma, rf = oracle.error_metrics(got, want)
    assert ma == 0.5 and abs(rf - 0.1) < 1e-15
    assert oracle.error_metrics(np.array([[np.nan, 1.0], [0, 0]]), want)[0] == float("inf")
