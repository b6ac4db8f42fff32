"""-m gpu tests of the state-plane page transfer (slack_kv_transfer, PAPER.md P:255, P:259-270,
P:660-662) against the oracle's exact copy: bit-exact whole-pool compare (integer / byte work), between two pools in HBM
and through a pinned host pool (eviction and restore), head partitions, layer-major events, and attention of the
migrated stream through its new page table."""
import copy

import numpy as np
import pytest
import torch

import oracle
from paper_2606_15319_b200 import binding, workloads as W
import gpu_harness as G
from helpers import oracle_pools

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    c = binding.Context(0)
    yield c
    c.close()


def sentinel_pool(w, n_pages, where="cuda"):
    shape = (n_pages, w.n_heads, w.page_size, w.head_dim)
    host = np.full(shape, G.host_fill(w), dtype=w.storage)
    k = binding.to_torch(host, w.dtype, DEV if where == "cuda" else "cpu", pin=(where == "pinned"))
    v = k.clone()
    if where == "pinned":
        v = v.pin_memory()
    return binding.Pool(k, v, n_pages, w.n_heads, w.head_dim, w.page_size, w.dtype), host.copy(), host.copy()


def bits(a):
    return a.view(np.uint32) if a.dtype == np.float32 else a


@pytest.mark.parametrize("make,heads", [(lambda: W.small_ragged(page_size=256), (0, 2)),
                                        (lambda: W.small_ragged(page_size=256), (1, 2)),
                                        (lambda: W.small_ragged(dtype="f32", head_dim=64, page_size=16), (0, 1))])
def test_transfer_bit_exact_between_hbm_pools(ctx, make, heads):
    w = make()
    src = G.make_pool(w)
    G.gpu_append_all(ctx, w, src)
    ko, vo = oracle_pools(w, fill=G.host_fill(w))
    n_dst = w.n_pages + 7
    dst, dk, dv = sentinel_pool(w, n_dst)
    rng = np.random.default_rng(5)
    perm = rng.permutation(n_dst)
    at = 0
    for s in w.streams[:3]:                                 # three separate requests (one stream each)
        sp = np.asarray(s.page_table, dtype=np.int32)
        dp = perm[at:at + sp.size].astype(np.int32)
        at += sp.size
        ctx.slack_kv_transfer([src], [dst], sp, dp, heads[0], heads[1])
        oracle.kv_transfer(ko, vo, dk, dv, sp, dp, heads[0], heads[1])
    torch.cuda.synchronize()
    assert np.array_equal(bits(binding.to_numpy(dst.k_pool, w.dtype)), bits(dk))
    assert np.array_equal(bits(binding.to_numpy(dst.v_pool, w.dtype)), bits(dv))
    assert G.pools_equal_oracle(w, src)                     # the source is read-only


def test_evict_to_pinned_host_and_restore(ctx):
    """Credit-aware eviction and later re-admission: HBM -> pinned host pool -> other pages of the HBM pool."""
    w = W.small_ragged(page_size=256, seed=31)
    src = G.make_pool(w)
    G.gpu_append_all(ctx, w, src)
    s = w.streams[0]
    sp = np.asarray(s.page_table, dtype=np.int32)
    host_pool, hk, hv = sentinel_pool(w, sp.size + 2, where="pinned")
    hp = np.arange(sp.size, dtype=np.int32)[::-1].copy()
    ctx.slack_kv_transfer([src], [host_pool], sp, hp, 0, w.n_heads)
    torch.cuda.synchronize()
    ko, vo = oracle_pools(w, fill=G.host_fill(w))
    oracle.kv_transfer(ko, vo, hk, hv, sp, hp, 0, w.n_heads)
    assert np.array_equal(binding.to_numpy(host_pool.k_pool, w.dtype), hk)
    assert np.array_equal(binding.to_numpy(host_pool.v_pool, w.dtype), hv)
    back, bk, bv = sentinel_pool(w, w.n_pages)
    rp = np.random.default_rng(2).permutation(w.n_pages)[:sp.size].astype(np.int32)
    ctx.slack_kv_transfer([host_pool], [back], hp, rp, 0, w.n_heads)
    torch.cuda.synchronize()
    oracle.kv_transfer(hk, hv, bk, bv, hp, rp, 0, w.n_heads)
    assert np.array_equal(binding.to_numpy(back.k_pool, w.dtype), bk)
    assert np.array_equal(binding.to_numpy(back.v_pool, w.dtype), bv)


def test_layer_major_events_and_attention_after_rehoming(ctx):
    """Re-homing: three layers move on a side stream in layer-major order; the consumer of layer l waits for event
    l only and attends through the new page table; results must equal the oracle on the source placement."""
    L = 3
    ws = [W.small_ragged(page_size=256, seed=40)]
    for l in range(1, L):                                   # same descriptors and page ids in every layer, other values
        wl = copy.deepcopy(ws[0])
        wl.q, wl.k_new, wl.v_new = (np.roll(a, 7 * l, axis=0) for a in (ws[0].q, ws[0].k_new, ws[0].v_new))
        wl.k_prior = [np.roll(a, 3 * l, axis=0) for a in ws[0].k_prior]
        wl.v_prior = [np.roll(a, 5 * l, axis=0) for a in ws[0].v_prior]
        ws.append(wl)
    srcs = []
    for w in ws:
        p = G.make_pool(w)
        G.gpu_append_all(ctx, w, p)
        srcs.append(p)
    w0 = ws[0]
    n_dst = w0.n_pages + 4
    dsts = [sentinel_pool(w0, n_dst)[0] for _ in range(L)]
    rng = np.random.default_rng(9)
    perm = rng.permutation(n_dst)
    moved, at = [], 0
    side = torch.cuda.Stream(DEV)
    events = [[torch.cuda.Event() for _ in range(L)] for _ in w0.streams]
    for e in sum(events, []):
        e.record(side)                                      # materialise the CUDA handles
    with torch.cuda.stream(side):
        for si, s in enumerate(w0.streams):
            sp = np.asarray(s.page_table, dtype=np.int32)
            dp = perm[at:at + sp.size].astype(np.int32)
            at += sp.size
            ctx.slack_kv_transfer(srcs, dsts, sp, dp, 0, w0.n_heads, stream=side, layer_done_events=events[si])
            m = copy.copy(s)
            m.page_table = dp
            moved.append(m)
    main = torch.cuda.current_stream()
    for l in range(L):
        for si in range(len(w0.streams)):
            main.wait_event(events[si][l])                  # layer l of every stream has arrived; later layers may not have
        w = copy.copy(ws[l])
        w.streams = moved
        w.n_pages = n_dst
        out, lse, plan, _ = G.gpu_attention(ctx, w, dsts[l])
        want, want_lse = G.oracle_attention(ws[l])
        G.check_attention(ws[l], out, lse, want, want_lse)
        assert plan.kernel_kind == G.TC_KIND


def test_transfer_argument_errors(ctx):
    w = W.small_ragged(page_size=256)
    src = G.make_pool(w)
    dst, _, _ = sentinel_pool(w, w.n_pages)
    ids = np.arange(3, dtype=np.int32)
    with pytest.raises(binding.SlackError):
        ctx.slack_kv_transfer([src], [dst], ids, np.array([0, 0, 1], dtype=np.int32), 0, w.n_heads)       # duplicate destination
    with pytest.raises(binding.SlackError):
        ctx.slack_kv_transfer([src], [dst], ids, np.array([0, 1, w.n_pages], dtype=np.int32), 0, w.n_heads)  # out of range
    with pytest.raises(binding.SlackError):
        ctx.slack_kv_transfer([src], [dst], ids, ids, 1, 1)                                                # empty head range
    ctx.slack_kv_transfer([src], [dst], ids[:0], ids[:0], 0, w.n_heads)                                     # empty list: no-op
    assert ctx.last_launch_count == 0


def test_back_to_back_transfers_on_two_streams(ctx):
    """the page-id lists of a transfer are staged per call and released behind its last kernel, so two
    transfers queued back to back on different streams cannot overwrite each other's lists."""
    w = W.small_ragged(page_size=256)
    src = G.make_pool(w)
    G.gpu_append_all(ctx, w, src)
    ko, vo = oracle_pools(w, fill=G.host_fill(w))
    s0, s1 = w.streams[0], w.streams[3]
    sp0, sp1 = np.asarray(s0.page_table, np.int32), np.asarray(s1.page_table, np.int32)
    n_dst = int(sp0.size + sp1.size + 3)
    dst, dk, dv = sentinel_pool(w, n_dst)
    perm = np.random.default_rng(9).permutation(n_dst).astype(np.int32)
    dp0, dp1 = perm[:sp0.size], perm[sp0.size:sp0.size + sp1.size]
    a, b = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    for _ in range(10):
        ctx.slack_kv_transfer([src] * 4, [dst] * 4, sp0, dp0, 0, w.n_heads, stream=a)
        ctx.slack_kv_transfer([src] * 4, [dst] * 4, sp1, dp1, 0, w.n_heads, stream=b)
    torch.cuda.synchronize()
    oracle.kv_transfer(ko, vo, dk, dv, sp0, dp0, 0, w.n_heads)
    oracle.kv_transfer(ko, vo, dk, dv, sp1, dp1, 0, w.n_heads)
    assert np.array_equal(bits(binding.to_numpy(dst.k_pool, w.dtype)), bits(dk))
    assert np.array_equal(bits(binding.to_numpy(dst.v_pool, w.dtype)), bits(dv))


def test_transfer_inside_one_pool_rejects_read_write_overlap(ctx):
    w = W.small_ragged(page_size=256)
    pool = G.make_pool(w)
    ids = np.asarray(w.streams[0].page_table, np.int32)
    assert ids.size >= 2
    with pytest.raises(binding.SlackError) as e:
        ctx.slack_kv_transfer([pool], [pool], ids[:2], ids[1:3] if ids.size >= 3 else ids[::-1][:2], 0, w.n_heads)
    assert e.value.status == binding.SLACK_EINVAL
