"""-m gpu: streams replayed chunk by chunk through the C ABI with the library's own page bookkeeping (slack_cache_*,
SURVEY §8(a) rows A0 and A5; "appended to a rolling KV cache for subsequent chunks", "preserves the
first few chunks as a global sink and keeps KV entries only for the most recent W chunks", P:251 paged pool behind a
logical page table).

Every state a serving loop produces and a one-snapshot test never sees is exercised on the CUDA path: page tables that
change between chunks, pages freed by one stream and handed to another WITHOUT being cleared (stale K/V bytes), a base /
hole that walks through a page as the window slides (both trim policies), re-append over the previous denoising step
followed by a commit, interleaved streams of different chunk lengths.

What it is compared with:
* every chunk's output, every denoising step: the oracle on the stream's WHOLE unpaged history (tests/replay.py
  TrueStream.reference_attention; it never sees a descriptor made by the pager), at the north-star tolerance
  (max-abs <= 2e-2, rel-Fro <= 1e-2 per chunk);
* the device pools after every append: bit-exact against a host pool image maintained with oracle.kv_append.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_15319_b200 import binding
from replay import TrueStream, check_cache_invariants

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
SENTINEL = 0x7FC1     # bf16 NaN: a read of a never-written slot poisons the output


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    c = binding.Context(0)
    yield c
    c.close()


def replay(ctx, policy, page_size, n_pages, specs, n_chunks, steps=2, H=2, D=128, batch=True, force_splits=0):
    """specs: [(q_len, window, sink)].  batch=True: all streams of a round are co-batched in one plan / append / attention;
    batch=False: one call per stream (the paper's one-stream-at-a-time dispatch)."""
    cache = binding.Cache(n_pages, page_size, policy)
    host_k = np.full((n_pages, H, page_size, D), SENTINEL, dtype=np.uint16)
    host_v = host_k.copy()
    dk = binding.to_torch(host_k, "bf16", DEV)
    dv = binding.to_torch(host_v, "bf16", DEV)
    pool = binding.Pool(dk, dv, n_pages, H, D, page_size, "bf16")
    true = [TrueStream(w, s, H, D, "bf16", seed=100 + i) for i, (_, w, s) in enumerate(specs)]
    ids = [cache.open(w, s) for (_, w, s) in specs]
    scale = 1.0 / np.sqrt(D)
    worst = 0.0
    for c in range(n_chunks):
        qls = [q if (i != 1 or c % 3) else max(1, q // 2) for i, (q, _, _) in enumerate(specs)]
        descs = [cache.begin_chunk(ids[i], qls[i]) for i in range(len(specs))]
        check_cache_invariants(cache, n_pages, descs)
        groups = [list(range(len(specs)))] if batch else [[i] for i in range(len(specs))]
        final = [None] * len(specs)
        for step in range(steps):
            drawn = [true[i].draw(qls[i]) for i in range(len(specs))]
            for g in groups:
                ds = [descs[i] for i in g]
                q = np.concatenate([drawn[i][0] for i in g])
                kn = np.concatenate([drawn[i][1] for i in g])
                vn = np.concatenate([drawn[i][2] for i in g])
                plan = ctx.slack_plan(pool, ds, force_splits=force_splits)
                qd, knd, vnd = (binding.to_torch(a, "bf16", DEV) for a in (q, kn, vn))
                ctx.slack_kv_append_planned(plan, pool, knd, vnd)
                oracle.kv_append(host_k, host_v, ds, kn, vn)
                out = torch.full_like(qd, float("nan"))
                ws = torch.empty(max(plan.workspace_bytes, 16), dtype=torch.uint8, device=DEV)
                ctx.slack_chunk_attention(plan, pool, qd, out, scale, workspace=ws)
                torch.cuda.synchronize()
                plan.close()                                              # plans come and go with every step
                assert np.array_equal(binding.to_numpy(dk, "bf16"), host_k), f"chunk {c} step {step}: K pool differs"
                assert np.array_equal(binding.to_numpy(dv, "bf16"), host_v), f"chunk {c} step {step}: V pool differs"
                got = out.float().cpu().numpy().astype(np.float64)
                r = 0
                for i in g:
                    want, _ = true[i].reference_attention(drawn[i][0], drawn[i][1], drawn[i][2], scale)
                    ma, rf = oracle.error_metrics(got[r:r + qls[i]], want)
                    assert ma <= 2e-2 and rf <= 1e-2, f"chunk {c} step {step} stream {i}: max_abs {ma:.3e} rel_fro {rf:.3e}"
                    worst = max(worst, rf)
                    r += qls[i]
            final = drawn
        for i in range(len(specs)):                                       # A5: the last denoising step's K/V is the chunk
            cache.commit(ids[i])
            true[i].commit(final[i][1], final[i][2])
    for sid in ids:
        cache.close_stream(sid)
    assert cache.free_pages == n_pages
    cache.close()
    return worst


@pytest.mark.parametrize("policy", [binding.TRIM_PAGES, binding.TRIM_TOKENS])
def test_replay_two_streams_window7_sink_p256(ctx, policy):
    """The verdict's case: >= 10 chunks, a 7-chunk window with a sink, two interleaved streams of different chunk lengths,
    S = 2 denoising steps per chunk, P = 256 with the window start walking through pages."""
    specs = [(150, 7 * 150, 72),      # sink ends mid-page; hole opens at chunk 7
             (90, 7 * 90, 0)]         # no sink: base walks (TRIM_TOKENS) or stays page-aligned (TRIM_PAGES)
    worst = replay(ctx, policy, 256, n_pages=14, specs=specs, n_chunks=12)
    print("replay P=256 worst rel_fro", worst)


@pytest.mark.parametrize("policy", [binding.TRIM_PAGES, binding.TRIM_TOKENS])
@pytest.mark.parametrize("batch", [True, False])
def test_replay_five_streams_recycling_pages_p128(ctx, policy, batch):
    """A pool with almost no slack: pages freed by one stream's sliding window are taken at once, uncleared, by the others."""
    specs = [(200, 3 * 200, 130),     # sink of more than a page, 3-chunk window
             (72, 5 * 72, 1),         # one-token sink; this stream's chunk length varies
             (257, 2 * 257, 0),       # short window, two query tiles + 1 row
             (129, 0, 0),             # unlimited window: only grows
             (64, 64, 16)]            # window = own chunk only, plus the sink
    worst = replay(ctx, policy, 128, n_pages=36, specs=specs, n_chunks=10, batch=batch)
    print("replay P=128 worst rel_fro", worst)


def test_replay_with_forced_splits(ctx):
    """The same replay with every row cut in three (split-KV partials + combine on a changing page table)."""
    specs = [(300, 900, 200), (140, 700, 0)]
    replay(ctx, binding.TRIM_TOKENS, 128, n_pages=30, specs=specs, n_chunks=8, steps=1, force_splits=3)
