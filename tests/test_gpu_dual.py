"""-m gpu parity tests of DUAL items (DevItem::dual / slack_work_item.dual): two single-tile items (<= 128 query rows each,
same number of key tiles) walked by one CTA, one per query-tile slot, each with its own K/V tiles - the decode-like
short-chunk case of BASELINE.json north_star.  Same oracle and tolerances as tests/test_gpu_parity.py; BASELINE's
supplementary decode-like config (64 streams x 72 queries x 8190 keys) is compared in full by tests/test_gpu_full_size.py."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_15319_b200 import binding, workloads as W
import gpu_harness as G
from helpers import oracle_pools

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    c = binding.Context(0)
    yield c
    c.close()


def decode_like(seed, n=10, heads=4, page_size=128):
    """Many short chunks (1..128 queries) over ragged caches, some windowed, bases anywhere in the first page."""
    rng = np.random.default_rng(seed)
    q = [int(x) for x in rng.integers(1, 129, size=n)]
    c = [int(x) for x in rng.integers(0, 1500, size=n)]
    wdw = [0 if i % 3 else 700 for i in range(n)]
    b = [int(x) for x in rng.integers(0, page_size, size=n)]
    return W.make_workload("decode_like_small", dtype="bf16", n_heads=heads, head_dim=128, page_size=page_size, q_lens=q,
                           cache_lens=c, windows=wdw, bases=b, seed=seed, amp=0.5, spare_pages=2)


def run(ctx, w, **opts):
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    out, lse, plan, launches = G.gpu_attention(ctx, w, pool, cta_pairs=1, **opts)
    want, want_lse = G.oracle_attention(w)
    G.check_attention(w, out, lse, want, want_lse)
    assert np.isfinite(out).all()
    return plan, out, pool


@pytest.mark.parametrize("seed", [1, 2, 3])
@pytest.mark.parametrize("sm_count", [0, 8, 3])
def test_decode_like_batches_use_dual_items(ctx, seed, sm_count):
    plan, *_ = run(ctx, decode_like(seed), sm_count=sm_count)
    items = plan.items()
    assert sum(i["dual"] for i in items) >= len(items) // 4, "short chunks should pair up"


def test_dual_items_with_split_rows_and_sinks(ctx):
    """Few queues, long caches: dual rows are cut into pieces (both members get partial slots and a combine entry)."""
    w = W.make_workload("decode_long", dtype="bf16", n_heads=4, head_dim=128, page_size=256, q_lens=[72, 100, 1, 128],
                        cache_lens=[5000, 5000, 3000, 2500], windows=[0, 4000, 0, 0], bases=[3, 0, 255, 17],
                        sink_lens=[0, 200, 0, 0], seed=9, amp=0.5, spare_pages=1)
    plan, *_ = run(ctx, w, sm_count=12)
    items = plan.items()
    assert any(i["dual"] and i["partial_slot"] >= 0 for i in items)


def test_one_head_leaves_singles_unpaired(ctx):
    plan, *_ = run(ctx, decode_like(4, heads=1), sm_count=4)      # one row per stream: nothing to pair within a stream


def test_other_kernels_walk_dual_items_one_by_one(ctx):
    """The block-sparse call gets the same (dual) plan and treats the two members as ordinary items."""
    w = decode_like(5)
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    plan = ctx.slack_plan(pool, w.streams, cta_pairs=1)
    assert any(i["dual"] for i in plan.items())
    masks = W.random_block_masks(w, 0.5, seed=2)
    q = binding.to_torch(w.q, w.dtype, "cuda:0")
    out = torch.full_like(q, float("nan"))
    md = torch.from_numpy(W.pack_block_masks(w, masks).view(np.int32)).to("cuda:0")
    ws = torch.empty(max(plan.sparse_workspace_bytes, 16), dtype=torch.uint8, device="cuda:0")
    ctx.slack_chunk_attention_sparse(plan, pool, q, out, w.scale, md, workspace=ws)
    torch.cuda.synchronize()
    ko, vo = oracle_pools(w, fill=G.host_fill(w))
    want, _ = oracle.chunk_attention(ko, vo, w.streams, w.q, w.scale, w.dtype, block_masks=masks)
    G.check_attention(w, out.float().cpu().numpy().astype(np.float64), None, want, None)


def test_repeated_launches_are_bit_identical(ctx):
    w = decode_like(6)
    plan, ref, pool = run(ctx, w)
    q = binding.to_torch(w.q, w.dtype, "cuda:0")
    ws = torch.full((max(plan.workspace_bytes, 16),), 0xFF, dtype=torch.uint8, device="cuda:0")
    for _ in range(20):
        out = torch.full_like(q, float("nan"))
        ws.fill_(0xFF)
        ctx.slack_chunk_attention(plan, pool, q, out, w.scale, workspace=ws)
        torch.cuda.synchronize()
        assert np.array_equal(out.float().cpu().numpy().astype(np.float64), ref)
