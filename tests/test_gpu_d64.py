"""-m gpu parity tests of bf16 with head_dim 64 on the tensor-core kernel (include/slack.h: head_dim in {64, 128}; the
kD = 64 instantiations of csrc/attn_tc.cu: half-sized Q / K / V tiles, N = 64 for P V, 64 TMEM columns of O, and the
head_dim 64 instantiation of the combine kernel).  Same oracle and bars as tests/test_gpu_parity.py: append bit-exact,
attention max-abs <= 2e-2 and relative Frobenius <= 1e-2 against the fp64 definition, whole output and per stream."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_15319_b200 import binding, workloads as W
import gpu_harness as G
from test_gpu_sparse import run_sparse

pytestmark = pytest.mark.gpu

D = 64


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    c = binding.Context(0)
    yield c
    c.close()


def run(ctx, w, tol=(2e-2, 1e-2), **opts):
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    assert G.pools_equal_oracle(w, pool)
    out, lse, plan, launches = G.gpu_attention(ctx, w, pool, **opts)
    want, want_lse = G.oracle_attention(w)
    res = G.check_attention(w, out, lse, want, want_lse, max_abs_tol=tol[0], rel_fro_tol=tol[1])
    assert np.isfinite(out).all(), f"{w.name}: unwritten / non-finite output rows"
    return plan, out, lse, launches


@pytest.mark.parametrize("page_size", [128, 256, 1024])
@pytest.mark.parametrize("splits", [0, 1, 3])
def test_small_ragged_d64_tensor_core(ctx, page_size, splits):
    plan, _, _, launches = run(ctx, W.small_ragged(head_dim=D, page_size=page_size), force_splits=splits)
    assert plan.kernel_kind == 0                       # not the SIMT kernel (1); pairs (2) are head_dim 128 only
    if splits > 1:
        assert plan.num_partial_slots > 0 and launches == 2     # attention + the head_dim 64 combine


@pytest.mark.parametrize("make", [W.sink_ragged, W.gap_ragged])
@pytest.mark.parametrize("splits", [0, 2])
def test_sink_and_gap_d64(ctx, make, splits):
    plan, *_ = run(ctx, make(head_dim=D, page_size=256), force_splits=splits)
    assert plan.kernel_kind == 0


@pytest.mark.parametrize("sm_count", [1, 3, 0])
def test_d64_queue_counts_and_more_heads(ctx, sm_count):
    plan, *_ = run(ctx, W.small_ragged(head_dim=D, n_heads=5, seed=31), sm_count=sm_count)
    assert plan.kernel_kind == 0


def test_d64_pair_request_falls_back_to_one_cta_per_item(ctx):
    plan, *_ = run(ctx, W.small_ragged(head_dim=D, seed=33), cta_pairs=2)
    assert plan.kernel_kind == 0


def test_d64_agrees_with_simt(ctx):
    w = W.small_ragged(head_dim=D, seed=21)
    _, out_tc, lse_tc, _ = run(ctx, w)
    plan, out_si, lse_si, _ = run(ctx, w, force_simt=1)
    assert plan.kernel_kind == 1
    ma, rf = oracle.error_metrics(out_tc, out_si)
    assert rf <= 1e-2 and ma <= 2e-2
    assert np.max(np.abs(lse_tc - lse_si)) <= 1e-3


@pytest.mark.parametrize("q_mul", [4.0, 16.0])
def test_d64_peaky_logits(ctx, q_mul):
    w = W.small_ragged(head_dim=D, seed=41)
    w.q = W.f32_to_bf16_bits(W.bf16_bits_to_f32(w.q) * np.float32(q_mul))
    run(ctx, w)


def test_d64_late_large_logits_force_rescale(ctx):
    """A few keys late in the order score far above everything before them: the running max jumps after many tiles (the
    thresholded rescale of O, here in its 64 TMEM columns), unsplit and across split pieces."""
    w = W.make_workload("late_max_d64", dtype="bf16", n_heads=2, head_dim=D, page_size=128, q_lens=[260], cache_lens=[1500],
                        windows=[0], bases=[3], seed=33, amp=0.5)
    q = W.bf16_bits_to_f32(w.q)
    kn = W.bf16_bits_to_f32(w.k_new)
    for j in (40, 200, 259):                       # own-chunk keys = the last tiles visited
        kn[j] = 24.0 * q[j] / np.maximum(np.linalg.norm(q[j], axis=-1, keepdims=True), 1e-6)
    w.k_new = W.f32_to_bf16_bits(kn)
    run(ctx, w, force_splits=1)
    run(ctx, w, force_splits=3)


def test_d64_deterministic(ctx):
    w = W.small_ragged(head_dim=D, seed=43, page_size=256)
    _, a, la, _ = run(ctx, w, force_splits=2)
    _, b, lb, _ = run(ctx, w, force_splits=2)
    assert np.array_equal(a, b) and np.array_equal(la, lb)


@pytest.mark.parametrize("rho", [0.0, 0.5, 0.9])
@pytest.mark.parametrize("splits", [0, 3])
def test_d64_block_sparse(ctx, rho, splits):
    w = W.small_ragged(head_dim=D, page_size=256)
    res = run_sparse(ctx, w, W.random_block_masks(w, rho, seed=5), force_splits=splits)
    assert res["kind"] == 0


def test_d64_decode_like_short_chunks(ctx):
    """Many single-tile items (no dual items at head_dim 64: the plan must not mark any)."""
    rng = np.random.default_rng(7)
    n = 12
    w = W.make_workload("decode_like_d64", dtype="bf16", n_heads=4, head_dim=D, page_size=128,
                        q_lens=[int(x) for x in rng.integers(1, 129, size=n)],
                        cache_lens=[int(x) for x in rng.integers(0, 1500, size=n)], windows=[0] * n,
                        bases=[int(x) for x in rng.integers(0, 128, size=n)], seed=7, amp=0.5, spare_pages=2)
    plan, *_ = run(ctx, w, sm_count=8)
    assert plan.kernel_kind == 0 and not any(i["dual"] for i in plan.items())


def test_d64_full_size_single_stream_full_output(ctx):
    """BASELINE.json configs[1]'s shape with head_dim 64 (4680 queries x 23400 keys x 12 heads, P = 256), default launch
    configuration: every output row against the oracle."""
    w = W.make_workload("cfg2_shape_d64", dtype="bf16", n_heads=12, head_dim=D, page_size=256, q_lens=[4680],
                        cache_lens=[4 * 4680], windows=[0], seed=2064, amp=0.5, n_pages=128)
    plan, *_ = run(ctx, w)
    assert plan.kernel_kind == 0
