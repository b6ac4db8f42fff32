"""Pins for the oracle's block-sparse variant (PAPER.md P:88 knob (2): "skips nonselected attention
blocks with sparse masks").  As in test_oracle_pins.py every check is against something other than the oracle's own
formula: a pure-Python brute force with its own index arithmetic, torch SDPA with an element-wise boolean mask, the
K = 0 closed form, and invariances.  CPU only."""
import math

import numpy as np
import pytest
import torch

import oracle
from paper_2606_15319_b200 import workloads as W
from helpers import oracle_pools, stream_rows


def tiny(seed=1, dtype="f32", **kw):
    args = dict(dtype=dtype, n_heads=2, head_dim=4, page_size=4, q_lens=[5, 3, 1], cache_lens=[6, 0, 9],
                windows=[0, 0, 7], bases=[0, 3, 2], seed=seed, spare_pages=2)
    args.update(kw)
    return W.make_workload("tiny", **args)


def rand_masks(w, bq, bk, seed, p_keep=0.5):
    """Unstructured random masks (rows may end up empty): [H, n_qb, n_kb] per stream."""
    rng = np.random.default_rng(seed)
    out = []
    for s in w.streams:
        n_qb, n_kb = -(-s.q_len // bq), -(-(s.base + s.cache_len + s.q_len) // bk)
        out.append(rng.random((w.n_heads, max(n_qb, 1), n_kb)) < p_keep)
    return out


def token_mask(w, s, m, bq, bk):
    """Element-wise boolean [H, Lq, n] 'query i may use key token t', written out from the definition."""
    n = s.cache_len + s.q_len
    lo = max(0, n - s.window) if s.window > 0 else 0
    sink = min(s.sink_len, n)
    ok = np.zeros((w.n_heads, s.q_len, n), dtype=bool)
    for h in range(w.n_heads):
        for i in range(s.q_len):
            for t in range(n):
                vis = t < sink or t >= max(lo, sink)
                ok[h, i, t] = vis and bool(m[h, i // bq, (s.base + t) // bk])
    return ok


# ------------------------------------------------------------------ all-ones mask == dense (same key sets; BLAS row blocking differs)
def test_all_ones_mask_is_dense():
    w = W.small_ragged(seed=5, dtype="bf16", head_dim=16)
    kp, vp = oracle_pools(w)
    dense, dlse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype)
    ones = [np.ones((w.n_heads, -(-s.q_len // 256) or 1, -(-(s.base + s.n) // 128)), dtype=bool) for s in w.streams]
    sp, slse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype, block_masks=ones)
    np.testing.assert_allclose(sp, dense, rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(slse, dlse, rtol=1e-13)


# ------------------------------------------------------------------ brute force, written independently
@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("bq,bk", [(2, 3), (1, 4), (4, 2)])
def test_brute_force_tiny_sparse(dtype, bq, bk):
    w = tiny(seed=4, dtype=dtype, sink_lens=[2, 0, 1])
    kp, vp = oracle_pools(w)
    masks = rand_masks(w, bq, bk, seed=9)
    out, lse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype, block_masks=masks, block_q=bq, block_k=bk)
    H, D, P = w.n_heads, w.head_dim, w.page_size
    dec = (lambda x: float(np.array([int(x) << 16], dtype=np.uint32).view(np.float32)[0])) if dtype == "bf16" else float
    row = 0
    n_empty = 0
    for s, m in zip(w.streams, masks):
        n = s.cache_len + s.q_len
        lo = n - s.window if (s.window > 0 and n > s.window) else 0
        sink = min(s.sink_len, n)
        for i in range(s.q_len):
            for h in range(H):
                keys = [t for t in range(n) if (t < sink or t >= max(lo, sink)) and m[h][i // bq][(s.base + t) // bk]]
                if not keys:
                    n_empty += 1
                    assert np.all(out[row + i, h] == 0.0) and lse[h, row + i] == -np.inf
                    continue
                qv = [dec(w.q[row + i, h, d]) for d in range(D)]
                logits, vals = [], []
                for t in keys:
                    pos = s.base + t
                    page, slot = int(s.page_table[pos // P]), pos % P
                    logits.append(w.scale * math.fsum(qv[d] * dec(kp[page, h, slot, d]) for d in range(D)))
                    vals.append([dec(vp[page, h, slot, d]) for d in range(D)])
                mx = max(logits)
                e = [math.exp(x - mx) for x in logits]
                den = math.fsum(e)
                want = [math.fsum(e[j] * vals[j][d] for j in range(len(keys))) / den for d in range(D)]
                np.testing.assert_allclose(out[row + i, h], want, rtol=1e-13, atol=1e-15)
                assert abs(lse[h, row + i] - (mx + math.log(den))) < 1e-13
        row += s.q_len
    assert not np.isnan(out).any()


# ------------------------------------------------------------------ library routine with a different masking mechanism
@pytest.mark.parametrize("base", [0, 1, 127])
def test_matches_torch_sdpa_with_boolean_mask(base):
    w = W.make_workload("sdpa", dtype="bf16", n_heads=2, head_dim=16, page_size=128, q_lens=[300, 70], cache_lens=[500, 260],
                        windows=[0, 200], bases=[base, (base + 5) % 128], sink_lens=[0, 40], seed=21, amp=1.0, spare_pages=1)
    kp, vp = oracle_pools(w)
    masks = W.random_block_masks(w, 0.5, seed=3)
    out, _ = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype, block_masks=masks)
    for s, m, (r0, r1) in zip(w.streams, masks, stream_rows(w)):
        n = s.cache_len + s.q_len
        toks = np.arange(n)
        pos = s.base + toks
        k = oracle.to_f64(kp[s.page_table[pos // 128], :, pos % 128, :], "bf16")      # [n, H, D], all tokens
        v = oracle.to_f64(vp[s.page_table[pos // 128], :, pos % 128, :], "bf16")
        q = oracle.to_f64(w.q[r0:r1], "bf16")
        ok = token_mask(w, s, m, 256, 128)
        ref = torch.nn.functional.scaled_dot_product_attention(
            torch.from_numpy(q).permute(1, 0, 2), torch.from_numpy(k).permute(1, 0, 2), torch.from_numpy(v).permute(1, 0, 2),
            attn_mask=torch.from_numpy(ok), scale=w.scale).permute(1, 0, 2).numpy()
        np.testing.assert_allclose(out[r0:r1], ref, rtol=1e-10, atol=1e-12)


# ------------------------------------------------------------------ closed form: K = 0 -> mean of V over the used keys
@pytest.mark.parametrize("base", [0, 1, 3])
@pytest.mark.parametrize("window", [0, 5, 11, 12])
def test_k_zero_gives_mean_of_used_values(base, window):
    w = W.make_workload("kz", dtype="f32", n_heads=1, head_dim=3, page_size=4, q_lens=[5], cache_lens=[7], windows=[window],
                        bases=[base], sink_lens=[2], seed=2, spare_pages=1)
    w.k_new[:] = 0
    w.k_prior[0][:] = 0
    kp, vp = oracle_pools(w)
    bq, bk = 2, 3
    masks = rand_masks(w, bq, bk, seed=base * 10 + window, p_keep=0.6)
    out, lse = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype, block_masks=masks, block_q=bq, block_k=bk)
    s = w.streams[0]
    v_all = np.concatenate([w.v_prior[0], w.v_new]).astype(np.float64)[:, 0, :]      # token order
    ok = token_mask(w, s, masks[0], bq, bk)[0]
    for i in range(s.q_len):
        if ok[i].any():
            np.testing.assert_allclose(out[i, 0], v_all[ok[i]].mean(axis=0), rtol=1e-14)
            assert abs(lse[0, i] - math.log(ok[i].sum())) < 1e-14
        else:
            assert np.all(out[i, 0] == 0) and lse[0, i] == -np.inf


# ------------------------------------------------------------------ invariances
def test_disjoint_masks_merge_to_union():
    w = W.small_ragged(seed=8, dtype="bf16", head_dim=16)
    kp, vp = oracle_pools(w)
    full = W.random_block_masks(w, 0.3, seed=1)
    rng = np.random.default_rng(0)
    a, b = [], []
    for m in full:
        if m is None:
            a.append(None); b.append(None)
            continue
        pick = rng.random(m.shape) < 0.5
        a.append(m & pick); b.append(m & ~pick)
    o_u, l_u = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype, block_masks=full)
    o_a, l_a = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype, block_masks=a)
    o_b, l_b = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype, block_masks=b)
    # rows empty in one part contribute weight e^{-inf} = 0
    L = np.stack([l_a, l_b]); m = L.max(axis=0)
    wgt = np.exp(L - m)
    den = wgt.sum(axis=0)                                      # [H, rows]
    merged = (wgt[0].T[:, :, None] * o_a + wgt[1].T[:, :, None] * o_b) / den.T[:, :, None]
    np.testing.assert_allclose(merged, o_u, rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(m + np.log(den), l_u, rtol=1e-13)


def test_bits_of_invisible_blocks_are_ignored():
    w = W.sink_ragged(seed=6, dtype="bf16", head_dim=16)
    kp, vp = oracle_pools(w)
    masks = W.random_block_masks(w, 0.6, seed=2)
    o1, l1 = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype, block_masks=masks)
    flipped = []
    for s, m in zip(w.streams, masks):
        m2 = m.copy()
        vis = W.visible_key_blocks(s)
        inv = np.setdiff1d(np.arange(m.shape[2]), vis)
        m2[:, :, inv] = True
        flipped.append(m2)
    o2, l2 = oracle.chunk_attention(kp, vp, w.streams, w.q, w.scale, w.dtype, block_masks=flipped)
    assert np.array_equal(o1, o2) and np.array_equal(l1, l2)


def test_generator_sparsity_and_packing():
    w = W.small_ragged(seed=3, dtype="bf16", head_dim=16)
    for rho in (0.0, 0.6, 0.9):
        masks = W.random_block_masks(w, rho, seed=4)
        for s, m in zip(w.streams, masks):
            if m is None:
                continue
            vis = W.visible_key_blocks(s)
            kept = m[:, :, vis].sum(axis=2)
            want = vis.size - min(int(round(rho * vis.size)), vis.size - 1)
            assert np.all(kept == want) and np.all(m[:, :, vis[-1]])
        packed = W.pack_block_masks(w, masks)
        assert packed.dtype == np.uint32 and packed.shape[1] == w.n_heads
        row = 0
        for s, m in zip(w.streams, masks):
            for qb in range(-(-s.q_len // 256)):
                for h in range(w.n_heads):
                    for kb in range(m.shape[2]):
                        assert bool((packed[row, h, kb // 32] >> np.uint32(kb % 32)) & np.uint32(1)) == bool(m[h, qb, kb])
                row += 1
        assert row == packed.shape[0]
