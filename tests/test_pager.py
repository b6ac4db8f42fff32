"""CPU tests of the page bookkeeping (slack_cache_*).

Which physical page a stream gets is arbitrary (several results are correct), so what is checked is what is unique:
* every descriptor the pager hands out maps the stream's VISIBLE tokens to the slots that hold exactly those tokens.
  A shadow pool of int64 "true token index" values is written through the oracle's append with the pager's descriptors;
  reading the oracle's visible tokens back through the oracle's token->slot rule must give the sink plus the last W
  tokens of the TRUE stream (tests/replay.py, which never sees a descriptor) - for both trim policies, with and without a
  sink, for interleaved streams of different chunk lengths that recycle each other's pages;
* invariants: no page owned twice, free + owned = pool, the footprint of a windowed stream is bounded however long it
  runs, positions stay bounded (gap_slots / base re-numbering), pool exhaustion is reported and takes nothing;
* the planner accepts every descriptor the pager produces (host-only context) and its cover invariants hold.
"""
import numpy as np
import pytest

import oracle
from paper_2606_15319_b200 import binding, build
from replay import TrueStream, check_cache_invariants


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()


def shadow_replay(policy, page_size, n_pages, specs, n_chunks, steps=2, hctx=None):
    """specs: [(q_len, window, sink)] per stream; streams are interleaved round-robin.  Returns the max pages any stream held."""
    cache = binding.Cache(n_pages, page_size, policy)
    shadow = np.full((n_pages, 1, page_size, 1), -1, dtype=np.int64)      # [n_pages][H=1][P][D=1] of true indices
    shadow_v = shadow.copy()
    true = [TrueStream(w, s, 1, 1, "f32", seed=i) for i, (_, w, s) in enumerate(specs)]
    ids = [cache.open(w, s) for (_, w, s) in specs]
    held_max = [0] * len(specs)
    last = {}
    for c in range(n_chunks):
        for i, (q_len, window, sink) in enumerate(specs):
            # vary the chunk length a little on one stream: trimming must follow the chunk that is about to be generated
            ql = q_len if (i != 1 or c % 3) else max(1, q_len // 2)
            d = cache.begin_chunk(ids[i], ql)
            assert cache.begin_chunk(ids[i], ql).page_table.tolist() == d.page_table.tolist()   # idempotent until commit
            last[i] = d
            check_cache_invariants(cache, n_pages, list(last.values()))
            n_true = true[i].committed
            new_idx = (n_true + np.arange(ql)).astype(np.int64).reshape(ql, 1, 1)
            for _ in range(steps):                                       # re-append of a later denoising step overwrites
                oracle.kv_append(shadow, shadow_v, [d], new_idx, new_idx)
            vis = oracle.visible_tokens(d)
            page, slot = oracle.token_slots(d, vis, page_size)
            got = shadow[page, 0, slot, 0]
            want = true[i].visible_true(ql)
            assert np.array_equal(got, want), f"chunk {c} stream {i}: visible tokens through the page table differ"
            # positions stay bounded: sink + window + chunk + a few pages
            end_pos = d.base + d.gap_slots + d.n
            if window:
                assert end_pos <= sink + window + ql + 3 * page_size
                assert d.page_table.size <= -(-(sink + window + ql) // page_size) + 3
            held_max[i] = max(held_max[i], int(d.page_table.size))
            assert cache.stream_pages(ids[i]) == d.page_table.size
            if hctx is not None:                                         # the planner takes what the pager makes
                pool = binding.Pool.shape_only(n_pages, 2, 128, page_size, "bf16")
                plan = hctx.slack_plan(pool, [d])
                assert plan.num_items > 0
                plan.close()
            cache.commit(ids[i])
            true[i].commit(np.zeros((ql, 1, 1), np.float32), np.zeros((ql, 1, 1), np.float32))
    for sid in ids:
        cache.close_stream(sid)
    assert cache.free_pages == n_pages
    cache.close()
    return held_max


@pytest.mark.parametrize("policy", [binding.TRIM_PAGES, binding.TRIM_TOKENS])
@pytest.mark.parametrize("page_size", [4, 16])
def test_shadow_replay_window_sink_interleaved(policy, page_size):
    specs = [(10, 70, 0),      # 7-chunk window, no sink
             (6, 20, 7),       # sink ending mid-page, short window, chunk length varies
             (9, 27, 3 * page_size),   # sink ending on a page boundary
             (5, 0, 0),        # unlimited: never trims
             (7, 4, 2)]        # window shorter than the chunk
    held = shadow_replay(policy, page_size, n_pages=400, specs=specs, n_chunks=14)
    assert held[3] == -(-(14 * 5) // page_size)            # the unlimited stream keeps everything


def test_window_keeps_footprint_bounded_for_long_streams():
    held = shadow_replay(binding.TRIM_PAGES, 8, n_pages=64, specs=[(12, 36, 5), (12, 84, 0)], n_chunks=60, steps=1)
    assert held[0] <= -(-(5 + 36 + 12) // 8) + 3 and held[1] <= -(-(84 + 12) // 8) + 3


def test_planner_accepts_pager_descriptors():
    hctx = binding.Context(-1)
    shadow_replay(binding.TRIM_TOKENS, 128, n_pages=64, specs=[(300, 900, 130), (257, 700, 0)], n_chunks=6, steps=1, hctx=hctx)
    hctx.close()


def test_exhaustion_takes_nothing_and_errors():
    cache = binding.Cache(4, 8, binding.TRIM_PAGES)
    a = cache.open()
    cache.begin_chunk(a, 20)                       # 3 pages
    cache.commit(a)
    b = cache.open()
    with pytest.raises(binding.SlackError) as e:
        cache.begin_chunk(b, 20)                   # needs 3, 1 free
    assert e.value.status == binding.SLACK_ENOMEM and cache.free_pages == 1 and cache.stream_pages(b) == 0
    d = cache.begin_chunk(b, 8)
    assert d.page_table.size == 1 and cache.free_pages == 0
    with pytest.raises(binding.SlackError):
        cache.begin_chunk(b, 9)                    # another length while a chunk is begun
    with pytest.raises(binding.SlackError):
        cache.commit(a)                            # nothing begun on a
    cache.close_stream(a)
    assert cache.free_pages == 3
    # most recently freed page is handed out first (recycled pages are reused at once, stale bytes and all)
    c = cache.open()
    d2 = cache.begin_chunk(c, 1)
    assert d2.page_table.size == 1
    cache.close()


def test_bad_arguments():
    lib = binding.load()
    import ctypes as C
    h = C.c_void_p()
    assert lib.slack_cache_create(0, 16, 0, C.byref(h)) == binding.SLACK_EINVAL
    assert lib.slack_cache_create(8, 12, 0, C.byref(h)) == binding.SLACK_EINVAL      # page size not a power of two
    assert lib.slack_cache_create(8, 16, 7, C.byref(h)) == binding.SLACK_EINVAL
    cache = binding.Cache(8, 16)
    with pytest.raises(binding.SlackError):
        cache.begin_chunk(3, 4)                    # no such stream
    with pytest.raises(binding.SlackError):
        cache.open(-1, 0)
    assert cache.stream_pages(0) == -1
    cache.close()
