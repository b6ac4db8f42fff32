"""-m gpu parity tests of the CTA-pair attention kernel (csrc/attn_tc2.cu: tcgen05 cta_group::2, slack_plan_opts.cta_pairs
= 2): the same oracle, the same tolerances as tests/test_gpu_parity.py.  (SLACK_TEST_CTA_PAIRS=2 reruns every other GPU
suite on this kernel; the cases here are the ones the default run always covers.)"""
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


def run_pairs(ctx, w, rows=None, **opts):
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    out, lse, plan, launches = G.gpu_attention(ctx, w, pool, cta_pairs=2, **opts)
    assert plan.kernel_kind == 2
    want, want_lse = G.oracle_attention(w, rows=rows)
    res = G.check_attention(w, out, lse, want, want_lse)
    if rows is None:
        assert np.isfinite(out).all()
    return res, out, lse, pool


@pytest.mark.parametrize("page_size", [128, 256, 512])
@pytest.mark.parametrize("splits", [0, 1, 2, 3])
def test_small_ragged_pairs(ctx, page_size, splits):
    run_pairs(ctx, W.small_ragged(page_size=page_size), force_splits=splits)


@pytest.mark.parametrize("make", [W.sink_ragged, W.gap_ragged])
@pytest.mark.parametrize("splits", [0, 2])
def test_sink_and_gap_pairs(ctx, make, splits):
    run_pairs(ctx, make(), force_splits=splits)


def test_few_ctas_and_odd_count_falls_back(ctx):
    w = W.small_ragged()
    run_pairs(ctx, w, sm_count=4)
    pool = G.make_pool(w)
    assert ctx.slack_plan(pool, w.streams, sm_count=7, cta_pairs=2).kernel_kind == 0      # an odd CTA count cannot pair up


def test_huge_logit_jumps_pairs(ctx):
    """Logits jumping by 100-400 nats late in the key order, in both column halves: the pair kernel's rescale waits for the
    previous P V (PV_DONE) and both halves of a row must agree on the new maximum."""
    w = W.make_workload("huge_jumps", dtype="bf16", n_heads=2, head_dim=128, page_size=128, q_lens=[260], cache_lens=[1500],
                        windows=[0], bases=[3], seed=35, amp=0.5)
    q = W.bf16_bits_to_f32(w.q)
    unit = q / np.maximum(np.linalg.norm(q, axis=-1, keepdims=True), 1e-6)
    kn = W.bf16_bits_to_f32(w.k_new)
    kn[40] = 250.0 * unit[40]
    kn[100] = 300.0 * unit[100]
    kn[200] = 200.0 * unit[7]
    kn[259] = 420.0 * unit[7]
    w.k_new = W.f32_to_bf16_bits(kn)
    for splits in (1, 3):
        res, out, lse, _ = run_pairs(ctx, w, force_splits=splits)
        assert np.isfinite(lse).all()


def test_cfg2_full_size_full_output_pairs(ctx):
    run_pairs(ctx, W.config2())


def test_repeated_launches_are_bit_identical(ctx):
    w = W.small_ragged(page_size=256)
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    ref, _, plan, _ = G.gpu_attention(ctx, w, pool, cta_pairs=2, force_splits=2)
    q = binding.to_torch(w.q, w.dtype, "cuda:0")
    ws = torch.full((max(plan.workspace_bytes, 16),), 0xFF, dtype=torch.uint8, device="cuda:0")
    for _ in range(25):
        out = torch.full_like(q, float("nan"))
        ws.fill_(0xFF)
        ctx.slack_chunk_attention(plan, pool, q, out, w.scale, workspace=ws)
        torch.cuda.synchronize()
        assert np.array_equal(out.float().cpu().numpy().astype(np.float64), ref)
