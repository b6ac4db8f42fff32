"""-m gpu parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the same
seeded inputs.  Bars (BASELINE.json north_star): append / page-table indexing bit-exact (whole-pool compare over a
NaN-sentinel-filled pool); attention max-abs <= 2e-2 and relative Frobenius <= 1e-2, whole output and per stream.
The fp32 SIMT path has the tighter self-imposed gate 1e-5 / 1e-5 (reading A10)."""
import copy

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


def run_case(ctx, w, tol=(2e-2, 1e-2), rows=None, **opts):
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    out, lse, plan, launches = G.gpu_attention(ctx, w, pool, **opts)
    want, want_lse = G.oracle_attention(w, rows=rows)
    res = G.check_attention(w, out, lse, want, want_lse, max_abs_tol=tol[0], rel_fro_tol=tol[1])
    # rows of `out` the plan must have written: none may keep the NaN pre-fill
    assert np.isfinite(out).all(), f"{w.name}: unwritten / non-finite output rows"
    res.update(kind=plan.kernel_kind, items=plan.num_items, slots=plan.num_partial_slots, launches=launches)
    return res, out, lse, pool


# ------------------------------------------------------------------------------------------------ append (A1)
@pytest.mark.parametrize("make", [W.config1, W.small_ragged, lambda: W.small_ragged(dtype="f32", head_dim=64, page_size=16)])
def test_append_bit_exact_small(ctx, make):
    w = make()
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    assert G.pools_equal_oracle(w, pool)


def test_append_planned_equals_unplanned_and_reappend_overwrites(ctx):
    w = W.small_ragged()
    pool = G.make_pool(w)
    plan = ctx.slack_plan(pool, w.streams)
    G.gpu_append_all(ctx, w, pool, planned_plan=plan)
    assert G.pools_equal_oracle(w, pool)
    # a later denoising step re-appends different values at the same position: only those slots change
    w2 = copy.copy(w)
    w2.k_new = w.v_new
    w2.v_new = w.k_new
    kn = binding.to_torch(w2.k_new, w.dtype, "cuda:0")
    vn = binding.to_torch(w2.v_new, w.dtype, "cuda:0")
    ctx.slack_kv_append_planned(plan, pool, kn, vn)
    torch.cuda.synchronize()
    assert G.pools_equal_oracle(w2, pool)


def test_append_bit_exact_cfg2_full_size(ctx):
    w = W.config2()
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    assert G.pools_equal_oracle(w, pool)


# ------------------------------------------------------------------------------------------------ attention, small
def test_cfg1_fp32_simt(ctx):
    res, *_ = run_case(ctx, W.config1(), tol=(1e-5, 1e-5))
    assert res["kind"] == 1 and res["launches"] == 1


@pytest.mark.parametrize("page_size", [128, 256, 512])
@pytest.mark.parametrize("splits", [0, 1, 2, 3])
def test_small_ragged_tensor_core(ctx, page_size, splits):
    res, *_ = run_case(ctx, W.small_ragged(page_size=page_size), force_splits=splits)
    assert res["kind"] == G.TC_KIND


# ------------------------------------------------------------------------------------------------ sink + local
@pytest.mark.parametrize("page_size", [128, 256])
@pytest.mark.parametrize("splits", [0, 1, 3])
def test_sink_plus_local_window_tensor_core(ctx, page_size, splits):
    """Visible keys = [0, sink) U [max(sink, lo), n): the sink tiles are visited before the window tiles of the first
    piece of every row; sink ends mid-tile, shares a tile with the window start, or is absorbed by the window."""
    res, *_ = run_case(ctx, W.sink_ragged(page_size=page_size), force_splits=splits)
    assert res["kind"] == G.TC_KIND


@pytest.mark.parametrize("page_size", [128, 256])
@pytest.mark.parametrize("splits", [0, 1, 3])
def test_bounded_sink_cache_with_hole(ctx, page_size, splits):
    """gap_slots (include/slack.h): a "sink + local" cache whose out-of-window tokens were dropped; append lands behind the
    hole bit-exactly and attention visits the sink tiles, skips the hole and visits the window tiles."""
    w = W.gap_ragged(page_size=page_size)
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    assert G.pools_equal_oracle(w, pool)
    res, *_ = run_case(ctx, w, force_splits=splits)
    assert res["kind"] == G.TC_KIND


def test_bounded_sink_cache_with_hole_simt(ctx):
    res, *_ = run_case(ctx, W.gap_ragged(dtype="f32", head_dim=64, page_size=16), tol=(1e-5, 1e-5))
    assert res["kind"] == 1
    res, *_ = run_case(ctx, W.gap_ragged(), force_simt=1)
    assert res["kind"] == 1


def test_sink_plus_local_window_simt(ctx):
    res, *_ = run_case(ctx, W.sink_ragged(dtype="f32", head_dim=64, page_size=16), tol=(1e-5, 1e-5))
    assert res["kind"] == 1
    res, *_ = run_case(ctx, W.sink_ragged(), force_simt=1)
    assert res["kind"] == 1


def test_small_ragged_simt_bf16_and_small_pages(ctx):
    res, *_ = run_case(ctx, W.small_ragged(page_size=32))
    assert res["kind"] == 1          # page_size < 128 is served by the SIMT path
    res, *_ = run_case(ctx, W.small_ragged(head_dim=64), force_simt=1)
    assert res["kind"] == 1          # bf16 head_dim 64 on request (by default the tensor-core kernel: test_gpu_d64.py)


def test_tensor_core_agrees_with_simt(ctx):
    w = W.small_ragged(seed=21)
    _, out_tc, lse_tc, _ = run_case(ctx, w)
    _, out_si, lse_si, _ = run_case(ctx, w, force_simt=1)
    ma, rf = oracle.error_metrics(out_tc, out_si)
    assert rf <= 1e-2 and ma <= 2e-2
    assert np.max(np.abs(lse_tc - lse_si)) <= 1e-3


def test_batched_equals_each_stream_alone(ctx):
    """With force_splits=1 every (stream, head, q-block) item runs the same key-tile sequence whatever else is in
    the batch, so the batched output is BIT-identical to each stream run alone (reading A13)."""
    w = W.small_ragged(seed=5)
    _, out_b, _, _ = run_case(ctx, w, force_splits=1)
    r = 0
    for si, s in enumerate(w.streams):
        if s.q_len:
            wa = W.make_workload("alone", dtype=w.dtype, n_heads=w.n_heads, head_dim=w.head_dim, page_size=w.page_size,
                                 q_lens=[s.q_len], cache_lens=[s.cache_len], windows=[s.window], bases=[s.base], seed=99)
            wa.q = w.q[r:r + s.q_len]
            wa.k_new, wa.v_new = w.k_new[r:r + s.q_len], w.v_new[r:r + s.q_len]
            wa.k_prior, wa.v_prior = [w.k_prior[si]], [w.v_prior[si]]
            _, out_a, _, _ = run_case(ctx, wa, force_splits=1)
            assert np.array_equal(out_a, out_b[r:r + s.q_len]), f"stream {si}"
        r += s.q_len


# ------------------------------------------------------------------------------------------------ adversarial inputs
def _scaled(w, q_mul=1.0, v_off=0.0):
    f = lambda a: W.bf16_bits_to_f32(a)
    if q_mul != 1.0:
        w.q = W.f32_to_bf16_bits(f(w.q) * np.float32(q_mul))
    if v_off:
        w.v_new = W.f32_to_bf16_bits(f(w.v_new) + np.float32(v_off))
        w.v_prior = [W.f32_to_bf16_bits(f(v) + np.float32(v_off)) for v in w.v_prior]
    return w


@pytest.mark.parametrize("q_mul", [4.0, 16.0])
def test_peaky_logits(ctx, q_mul):
    run_case(ctx, _scaled(W.small_ragged(seed=31), q_mul=q_mul))


def test_v_common_offset(ctx):
    run_case(ctx, _scaled(W.small_ragged(seed=32), v_off=100.0), tol=(1.0, 1e-2))  # |out| ~ 100: rel-Fro binds


def test_late_large_logits_force_rescale(ctx):
    """A few keys late in the order score far above the rest: the running max jumps after many tiles, which
    exercises the thresholded O rescale of the tensor-core kernel."""
    w = W.make_workload("late_max", dtype="bf16", n_heads=2, head_dim=128, page_size=128, q_lens=[260], cache_lens=[1500],
                        windows=[0], bases=[3], seed=33, amp=0.5)
    q = W.bf16_bits_to_f32(w.q)
    kn = W.bf16_bits_to_f32(w.k_new)
    for j in (40, 200, 259):                       # own-chunk keys = the last tiles visited
        kn[j] = 6.0 * q[j % 260] / np.maximum(np.linalg.norm(q[j % 260], axis=-1, keepdims=True), 1e-6) * 4.0
    w.k_new = W.f32_to_bf16_bits(kn)
    run_case(ctx, w, force_splits=1)
    run_case(ctx, w, force_splits=3)


def test_huge_logit_jumps_inside_a_tile(ctx):
    """Keys whose logit exceeds everything seen before by 100-300 nats (>> 64 in log2 units), sitting in the first and
    in the second 64 columns of late key tiles, once and twice on the same query row, rising and falling: the lazy-rescale
    logic must take its exact path (true maximum, rescale, recompute) instead of overflowing.  The oracle is fp64."""
    w = W.make_workload("huge_jumps", dtype="bf16", n_heads=2, head_dim=128, page_size=128, q_lens=[260], cache_lens=[1500],
                        windows=[0], bases=[3], seed=35, amp=0.5)
    q = W.bf16_bits_to_f32(w.q)
    unit = q / np.maximum(np.linalg.norm(q, axis=-1, keepdims=True), 1e-6)         # [260, H, D]
    kn = W.bf16_bits_to_f32(w.k_new)
    kp = W.bf16_bits_to_f32(w.k_prior[0])
    # own-chunk token j sits at position 3 + 1500 + j: column (1503 + j) % 128 of its tile
    cols = {j: (1503 + j) % 128 for j in (40, 100, 200, 230, 259)}
    assert cols[40] < 64 and cols[200] < 64 and cols[100] >= 64 and cols[259] >= 64
    kn[40] = 250.0 * unit[40]          # first half of a tile, row 40
    kn[100] = 300.0 * unit[100]        # second half, row 100
    kn[200] = 200.0 * unit[7]          # row 7: first jump ...
    kn[259] = 420.0 * unit[7]          # ... and a larger one later, second half
    kn[230] = 150.0 * unit[40]         # row 40 again, smaller than its first jump (must not disturb it)
    kp[700] = 180.0 * unit[100]        # an early big key for row 100 (mid-cache), overtaken later by kn[100]
    w.k_new = W.f32_to_bf16_bits(kn)
    w.k_prior = [W.f32_to_bf16_bits(kp)]
    for splits in (1, 3):
        res, out, lse, _ = run_case(ctx, w, force_splits=splits)
        assert np.isfinite(lse).all()


def test_all_equal_logits_and_zero_q(ctx):
    w = W.small_ragged(seed=34)
    w.q = np.zeros_like(w.q)
    res, out, lse, _ = run_case(ctx, w)
    # closed form: lse = ln(Lk)
    r = 0
    for s in w.streams:
        if s.q_len:
            lk = len(oracle.visible_tokens(s))
            assert np.allclose(lse[:, r:r + s.q_len], np.log(lk), atol=1e-4)
        r += s.q_len


# ------------------------------------------------------------------------------------------------ unusual shapes / sizes
@pytest.mark.parametrize("n_heads,page_size,lq,lc,window,base", [
    (5, 1024, 300, 70000, 0, 1023),        # long cache (550 key tiles), odd head count, base at the last slot of a page
    (1, 128, 257, 40000, 33000, 127),      # one head, window cutting mid-tile far into the cache
    (40, 256, 129, 515, 0, 0),             # many heads, short cache
])
def test_unusual_shapes_sampled_rows(ctx, n_heads, page_size, lq, lc, window, base):
    w = W.make_workload("odd_shape", dtype="bf16", n_heads=n_heads, head_dim=128, page_size=page_size, q_lens=[lq],
                        cache_lens=[lc], windows=[window], bases=[base], seed=77, amp=0.5, spare_pages=2)
    rows = [np.unique(np.concatenate([[0, 127, 128, lq - 1], np.random.default_rng(5).integers(0, lq, size=24)]))]
    for splits in (0, 1):
        res, out, *_ = run_case(ctx, w, rows=rows, force_splits=splits)
        assert res["kind"] == G.TC_KIND


# ------------------------------------------------------------------------------------------------ plan / staging lifetime
def test_plans_created_and_destroyed_while_kernels_are_in_flight(ctx):
    """slack_plan takes its tables from the ctx arena and slack_plan_destroy hands them back through events: hundreds of
    plans are made, used once on one of two streams and destroyed at once (no synchronisation in between); every output
    must equal the one computed with a long-lived plan, bit for bit."""
    w = W.small_ragged(page_size=256)
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    ref, _, plan0, _ = G.gpu_attention(ctx, w, pool, force_splits=2)
    q = binding.to_torch(w.q, w.dtype, "cuda:0")
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = [torch.full_like(q, float("nan")) for _ in range(2)]
    wss = [torch.empty(max(plan0.workspace_bytes, 16), dtype=torch.uint8, device="cuda:0") for _ in range(2)]
    torch.cuda.synchronize()
    for it in range(300):
        st = streams[it & 1]
        plan = ctx.slack_plan(pool, w.streams, force_splits=2, cta_pairs=plan0.kernel_kind)   # 0 (automatic) or 2
        ctx.slack_chunk_attention(plan, pool, q, outs[it & 1], w.scale, workspace=wss[it & 1], stream=st)
        plan.close()
    torch.cuda.synchronize()
    for o in outs:
        assert np.array_equal(o.float().cpu().numpy().astype(np.float64), ref)


def test_unplanned_appends_on_two_streams_do_not_share_staging(ctx):
    """two slack_kv_append calls back to back on different streams used to share one staging table."""
    wa, wb = W.small_ragged(seed=41, page_size=256), W.small_ragged(seed=42, page_size=256)
    pa, pb = G.make_pool(wa), G.make_pool(wb)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    ka, va = binding.to_torch(wa.k_new, wa.dtype, "cuda:0"), binding.to_torch(wa.v_new, wa.dtype, "cuda:0")
    kb, vb = binding.to_torch(wb.k_new, wb.dtype, "cuda:0"), binding.to_torch(wb.v_new, wb.dtype, "cuda:0")
    torch.cuda.synchronize()
    for _ in range(20):
        ctx.slack_kv_append(pa, wa.streams, ka, va, stream=sa)
        ctx.slack_kv_append(pb, wb.streams, kb, vb, stream=sb)
    torch.cuda.synchronize()
    import helpers
    for w, pool in ((wa, pa), (wb, pb)):
        ko, vo = helpers.empty_pools(w, G.host_fill(w))
        oracle.kv_append(ko, vo, w.streams, w.k_new, w.v_new)
        assert np.array_equal(binding.to_numpy(pool.k_pool, w.dtype), ko) and np.array_equal(binding.to_numpy(pool.v_pool, w.dtype), vo)
