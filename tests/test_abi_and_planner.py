"""CPU-only tests of the boundary and the host logic: libslack.so loads and exports every symbol include/slack.h
declares; slack_plan on a host-only context validates descriptors (status codes of slack.h) and emits plans that
satisfy the cover invariants (the plan has many valid answers, so it is checked by invariants).
No compute call is made: data-path calls on a host-only context must fail with SLACK_ECUDA (no CPU fallback)."""
import os
import re
import subprocess

import numpy as np
import pytest

from paper_2606_15319_b200 import binding, build, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def hctx():
    build.build()
    c = binding.Context(-1)
    yield c
    c.close()


def declared_symbols(header="slack.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(slack_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound():
    build.build()
    names = declared_symbols()
    assert {"slack_kv_append", "slack_plan", "slack_chunk_attention"} <= set(names)
    out = subprocess.check_output(["nm", "-D", "--defined-only", binding.LIB_PATH], text=True)
    exported = set(l.split()[-1] for l in out.splitlines() if l.strip())
    for n in names:
        assert n in exported, f"{n} declared in slack.h but not exported"
        assert n in binding.SYMBOLS, f"{n} has no ctypes signature in the binding"
    lib = binding.load()
    assert lib.slack_abi_version() == 3
    # include/slack_diag.h is exported by -DSLACK_DIAGNOSTICS builds only; the default library carries none of it
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == ["slack.h", "slack_diag.h"]
    diag = declared_symbols("slack_diag.h")
    assert diag == ["slack_debug_set"] and set(diag) == set(binding.DIAG_SYMBOLS)
    if os.environ.get("SLACK_DIAGNOSTICS", "0") in ("", "0"):
        assert not (set(diag) & exported), "the default build must not export the diagnostics calls"
        ksyms = subprocess.check_output(["nm", "-C", "--defined-only", binding.LIB_PATH], text=True)
        assert "attn_tc_kernel<true" not in ksyms, "the traced kernel instantiation must not be in the default build"


def test_struct_sizes_match_header():
    import ctypes as C
    assert C.sizeof(binding.CPool) == 56 and C.sizeof(binding.CStream) == 40
    assert C.sizeof(binding.CPlanOpts) == 16 and C.sizeof(binding.CWorkItem) == 52


def test_host_only_context_has_no_data_path(hctx):
    w = W.small_ragged()
    pool = binding.Pool.shape_only(w.n_pages, w.n_heads, w.head_dim, w.page_size, w.dtype)
    plan = hctx.slack_plan(pool, w.streams)
    with pytest.raises(binding.SlackError) as e:
        hctx.slack_chunk_attention(plan, pool, 256, 256, 1.0)
    assert e.value.status == binding.SLACK_ECUDA
    with pytest.raises(binding.SlackError) as e:
        hctx.slack_kv_append(pool, w.streams, 256, 256)
    assert e.value.status == binding.SLACK_ECUDA


def _pool(w, **kw):
    args = dict(n_pages=w.n_pages, n_heads=w.n_heads, head_dim=w.head_dim, page_size=w.page_size, dtype=w.dtype)
    args.update(kw)
    return binding.Pool.shape_only(**args)


def check_cover(w, plan, n_cta):
    """Every (stream, head, query row) is covered by items whose key-tile ranges partition the stream's tile range;
    partial slots are used iff a range is cut, each exactly once; queues are contiguous per CTA."""
    items = plan.items()
    row0 = 0
    by_key = {}
    for it in items:
        by_key.setdefault((it["stream"], it["head"], it["q_row0"]), []).append(it)
        assert 0 <= it["cta"] < n_cta
        assert 1 <= it["q_rows"] <= 256
        assert it["kv_tile_begin"] < it["kv_tile_end"]
    ctas = [it["cta"] for it in items]
    assert ctas == sorted(ctas), "items must be stored queue by queue"
    for a, b in zip(items, items[1:] + [None]):     # dual items: the companion follows in the same queue, same key steps
        if a["dual"]:
            assert b is not None and b["cta"] == a["cta"] and not b["dual"]
            assert a["q_rows"] <= 128 and b["q_rows"] <= 128
            assert (a["kv_tile_end"] - a["kv_tile_begin"], a["sink_tiles"]) == (b["kv_tile_end"] - b["kv_tile_begin"], b["sink_tiles"])
    slots = [it["partial_slot"] for it in items if it["partial_slot"] >= 0]
    assert sorted(slots) == list(range(plan.num_partial_slots))
    for si, s in enumerate(w.streams):
        if s.q_len == 0:
            assert not any(k[0] == si for k in by_key)
            continue
        n = s.cache_len + s.q_len
        lo = max(0, n - s.window) if s.window > 0 else 0
        sink = min(getattr(s, "sink_len", 0), n)
        gap = getattr(s, "gap_slots", 0)
        if lo <= sink and gap == 0:         # the window still touches the sink and no slot is skipped: one visible range
            lo, sink = 0, 0
        lo = max(lo, sink)
        pos_lo, pos_hi = s.base + (gap if sink else 0) + lo, s.base + gap + n
        t0, t1 = pos_lo // 128, -(-pos_hi // 128)
        want_sink_tiles = (-(-(s.base + sink) // 128) - s.base // 128) if sink > 0 else 0
        for h in range(w.n_heads):
            covered = 0
            for qb in range(-(-s.q_len // 256)):
                parts = sorted(by_key[(si, h, row0 + qb * 256)], key=lambda x: x["kv_tile_begin"])
                assert parts[0]["kv_tile_begin"] == t0 and parts[-1]["kv_tile_end"] == t1
                for a, b in zip(parts, parts[1:]):
                    assert a["kv_tile_end"] == b["kv_tile_begin"]
                for pi, p in enumerate(parts):
                    assert (p["pos_lo"], p["pos_hi"]) == (pos_lo, pos_hi)
                    assert p["q_rows"] == min(256, s.q_len - qb * 256)
                    assert (p["partial_slot"] >= 0) == (len(parts) > 1)
                    # the sink rides with the first piece of the row only
                    assert p["sink_tiles"] == (want_sink_tiles if pi == 0 else 0)
                    assert p["sink_pos_hi"] == (s.base + sink if pi == 0 else s.base)
                covered += parts[0]["q_rows"]
            assert covered == s.q_len
        row0 += s.q_len
    return items


@pytest.mark.parametrize("pairs", [1, 2])
@pytest.mark.parametrize("splits", [0, 1, 2, 5])
@pytest.mark.parametrize("n_cta", [1, 7, 8, 148])
@pytest.mark.parametrize("make", [W.small_ragged, W.sink_ragged, W.gap_ragged])
def test_plan_cover_small(hctx, splits, n_cta, make, pairs):
    """cta_pairs = 2 (include/slack.h): the same items, dealt to sm_count / 2 queues, one per CTA pair."""
    w = make()
    plan = hctx.slack_plan(_pool(w), w.streams, sm_count=n_cta, force_splits=splits, cta_pairs=pairs)
    paired = pairs == 2 and n_cta % 2 == 0                      # an odd CTA count cannot pair up
    assert plan.kernel_kind == (2 if paired else 0)
    check_cover(w, plan, n_cta // 2 if paired else n_cta)
    if splits == 1:
        assert plan.num_partial_slots == 0 and plan.workspace_bytes == 0
    else:
        assert plan.workspace_bytes == plan.num_partial_slots * 256 * (128 + 1) * 4


def _descr_only(maker):
    """Config workloads without drawing the (large) tensors: only descriptors are needed for planning."""
    import unittest.mock as m
    with m.patch.object(W, "_draw", lambda rng, shape, amp, dtype: np.zeros((0,), dtype=np.uint16)):
        return maker()


@pytest.mark.parametrize("pairs", [1, 2])
@pytest.mark.parametrize("maker", [W.config2, W.config3, W.config4, lambda: W.config5(7), lambda: W.config5(1), W.config5b])
def test_plan_cover_and_balance_full_configs(hctx, maker, pairs):
    w = _descr_only(maker)
    plan = hctx.slack_plan(_pool(w), w.streams, sm_count=148, cta_pairs=pairs)
    nq = 148 // pairs
    items = check_cover(w, plan, nq)
    load = np.zeros(nq)
    companion = False
    for it in items:
        if companion:                # second member of a dual item: rides in the first one's key steps
            companion = False
            continue
        companion = bool(it["dual"])
        load[it["cta"]] += (2.0 if (pairs == 2 or it["q_rows"] > 128 or it["dual"]) else 1.70) * (it["kv_tile_end"] - it["kv_tile_begin"]) + 7.75
    assert load.max() <= 1.25 * load.mean() + 40, f"{w.name}: makespan {load.max():.0f} vs ideal {load.mean():.0f}"


def test_plan_is_deterministic_and_layer_invariant(hctx):
    w = _descr_only(W.config3)
    a = hctx.slack_plan(_pool(w), w.streams).items()
    b = hctx.slack_plan(_pool(w), w.streams).items()
    assert a == b


def test_static_workspace_entry_point_needs_a_device(hctx):
    """slack_chunk_attention_static / slack_static_workspace_init (no-allocation variant): like every data call, refused by
    a host-only context; the size check against SLACK_STATIC_WORKSPACE_BYTES comes first and needs no device."""
    w = W.small_ragged(page_size=256)
    plan = hctx.slack_plan(_pool(w), w.streams, force_splits=3)
    assert 0 < plan.workspace_bytes <= (32 << 20)
    with pytest.raises(binding.SlackError) as e:
        hctx.slack_static_workspace_init()
    assert e.value.status == binding.SLACK_ECUDA
    with pytest.raises(binding.SlackError) as e:
        hctx.slack_chunk_attention_static(plan, _pool(w), None, None, w.scale)
    assert e.value.status == binding.SLACK_ECUDA
    w = _descr_only(W.config3)
    big = hctx.slack_plan(_pool(w), w.streams, force_splits=3)
    assert big.workspace_bytes > (32 << 20)
    with pytest.raises(binding.SlackError) as e:
        hctx.slack_chunk_attention_static(big, _pool(w), None, None, w.scale)
    assert e.value.status == binding.SLACK_ENOMEM and "static workspace" in str(e.value)


def test_kernel_kind_selection(hctx):
    w = W.config1()
    assert hctx.slack_plan(_pool(w), w.streams).kernel_kind == 1            # f32 -> SIMT
    w = W.small_ragged(page_size=64)
    assert hctx.slack_plan(_pool(w), w.streams).kernel_kind == 1            # page < 128 -> SIMT
    w = W.small_ragged()
    assert hctx.slack_plan(_pool(w), w.streams, force_simt=1).kernel_kind == 1
    w = W.small_ragged(head_dim=64)                                         # bf16 head_dim 64: tensor-core kernel, never
    for pairs in (0, 1, 2):                                                 # CTA pairs, never dual items
        plan = hctx.slack_plan(_pool(w), w.streams, cta_pairs=pairs)
        assert plan.kernel_kind == 0 and not any(i["dual"] for i in plan.items())
    assert hctx.slack_plan(_pool(w), w.streams, force_simt=1).kernel_kind == 1


# ------------------------------------------------------------------------------------------------ error behaviour
def _expect(hctx, status, w, pool=None, mutate=None, **opts):
    streams = [W.StreamSpec(s.q_len, s.cache_len, s.base, s.window, s.sink_len, s.page_table.copy(), s.gap_slots) for s in w.streams]
    if mutate:
        mutate(streams)
    with pytest.raises(binding.SlackError) as e:
        hctx.slack_plan(pool or _pool(w), streams, **opts)
    assert e.value.status == status, str(e.value)


def test_plan_rejects_malformed_descriptors(hctx):
    w = W.small_ragged()
    E, U = binding.SLACK_EINVAL, binding.SLACK_EUNSUPPORTED
    _expect(hctx, E, w, mutate=lambda s: setattr(s[0], "q_len", -1))
    _expect(hctx, E, w, mutate=lambda s: setattr(s[0], "base", w.page_size))
    _expect(hctx, E, w, mutate=lambda s: setattr(s[0], "page_table", s[0].page_table[:-1]))
    _expect(hctx, E, w, mutate=lambda s: s[0].page_table.__setitem__(0, w.n_pages))
    _expect(hctx, E, w, mutate=lambda s: s[0].page_table.__setitem__(0, -1))
    _expect(hctx, E, w, mutate=lambda s: s[1].page_table.__setitem__(0, int(s[0].page_table[0])))   # page owned twice
    _expect(hctx, E, w, mutate=lambda s: setattr(s[0], "sink_len", -4))
    _expect(hctx, E, w, mutate=lambda s: setattr(s[0], "gap_slots", -1))
    _expect(hctx, E, w, mutate=lambda s: setattr(s[0], "gap_slots", 5))                      # a hole needs a sink in front of it
    def young(s):
        s[0].sink_len, s[0].gap_slots = s[0].cache_len + 1, 5                                # ... and a filled sink
    _expect(hctx, E, w, mutate=young)
    _expect(hctx, U, w, pool=_pool(w, head_dim=96))
    _expect(hctx, U, w, pool=_pool(w, page_size=48))
    _expect(hctx, U, w, pool=_pool(w, page_size=8))
    _expect(hctx, E, w, pool=_pool(w, n_pages=0))


def test_empty_batches_are_legal(hctx):
    w = W.small_ragged()
    plan = hctx.slack_plan(_pool(w), [])
    assert plan.num_items == 0 and plan.workspace_bytes == 0
    empty = [W.StreamSpec(0, s.cache_len, s.base, s.window, 0, s.page_table) for s in w.streams]
    plan = hctx.slack_plan(_pool(w), empty)
    assert plan.num_items == 0


def test_sparse_plan_geometry(hctx):
    """Mask geometry and workspace the block-sparse call needs (include/slack.h): rows = sum ceil(Lq/256); words cover the
    last key block of the longest stream; the sparse workspace holds the split-KV partials plus one uint16 per dense
    key-tile step and one int32 per item."""
    w = W.small_ragged(page_size=256)
    pool = binding.Pool(None, None, w.n_pages, w.n_heads, w.head_dim, w.page_size, w.dtype)
    plan = hctx.slack_plan(pool, w.streams, force_splits=2)
    assert plan.mask_rows == sum(-(-s.q_len // 256) for s in w.streams)
    assert plan.mask_min_words == -(-max(-(-(s.base + s.gap_slots + s.n) // 128) for s in w.streams) // 32)
    items = plan.items()
    steps = sum(it["sink_tiles"] + it["kv_tile_end"] - it["kv_tile_begin"] for it in items)
    assert plan.sparse_workspace_bytes >= plan.workspace_bytes + 2 * steps + 4 * len(items)
    packed = W.pack_block_masks(w, W.random_block_masks(w, 0.5, seed=1))
    assert packed.shape == (plan.mask_rows, w.n_heads, plan.mask_min_words)
