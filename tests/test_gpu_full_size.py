"""-m gpu parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default plan options).
The oracle computes SAMPLED query rows one by one (rows are independent, so a sampled row is exact):
per stream the tile-boundary rows {0, 127, 128, 255, 256, Lq-73, Lq-72, Lq-1} plus seeded random rows, every head,
every visible key.  Append is checked bit-exactly over the whole pool."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_15319_b200 import binding, workloads as W
import gpu_harness as G

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    c = binding.Context(0)
    yield c
    c.close()


def sample_rows(w, n_random=24, seed=123):
    rng = np.random.default_rng(seed)
    rows = []
    for s in w.streams:
        if s.q_len == 0:
            rows.append(np.zeros(0, dtype=np.int64))
            continue
        fixed = [0, 127, 128, 255, 256, s.q_len - 73, s.q_len - 72, s.q_len - 1]
        fixed = [r for r in fixed if 0 <= r < s.q_len]
        rnd = rng.integers(0, s.q_len, size=n_random).tolist()
        rows.append(np.unique(np.array(fixed + rnd, dtype=np.int64)))
    return rows


def full_case(ctx, w, check_append=True, **opts):
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    if check_append:
        assert G.pools_equal_oracle(w, pool), f"{w.name}: append not bit-exact"
    out, lse, plan, launches = G.gpu_attention(ctx, w, pool, **opts)
    assert np.isfinite(out).all(), f"{w.name}: unwritten / non-finite output rows"
    rows = sample_rows(w)
    want, want_lse = G.oracle_attention(w, rows=rows)
    res = G.check_attention(w, out, lse, want, want_lse)
    assert plan.kernel_kind == 0
    return res, plan


def test_cfg2_single_stream(ctx):
    res, plan = full_case(ctx, W.config2())
    print("cfg2", res, plan.num_items, plan.num_partial_slots)


def test_cfg3_ragged8(ctx):
    res, plan = full_case(ctx, W.config3())
    print("cfg3", res, plan.num_items, plan.num_partial_slots)


def test_cfg4_mixed16_window(ctx):
    w = W.config4()
    assert any(s.window and s.cache_len + s.q_len > s.window for s in w.streams), "config 4 must clip a window (A3)"
    res, plan = full_case(ctx, w)
    print("cfg4", res, plan.num_items, plan.num_partial_slots)


@pytest.mark.parametrize("kv_chunks,splits", [(1, 0), (7, 0), (7, 2), (4, 4)])
def test_cfg5_long_cache_points(ctx, kv_chunks, splits):
    res, plan = full_case(ctx, W.config5(kv_chunks=kv_chunks), check_append=(kv_chunks == 7 and splits == 0),
                          force_splits=splits)
    print("cfg5", kv_chunks, splits, res, plan.num_items, plan.num_partial_slots)


def test_cfg5b_decode_like(ctx):
    w = W.config5b(n_streams=16)
    res, plan = full_case(ctx, w)
    print("cfg5b", res, plan.num_items, plan.num_partial_slots)
