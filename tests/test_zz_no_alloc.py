"""-m gpu test of slack_chunk_attention_static (include/slack.h "A3 + A4 without a caller workspace"): attention whose
split-KV workspace is a static device array inside libslack.so, for callers that cannot allocate (CUDA graph capture,
serving loops).  Collected last on purpose (file name): the suite runs with pytest -x.

The new entry point runs the same kernels as slack_chunk_attention, so its output must equal the existing path's bit for
bit; the comparison is still written with the tolerances of tests/test_gpu_parity.py (max-abs <= 2e-2, rel-Fro <= 1e-2),
on two calls in a row (the second finds the first call's partials in the shared array), and both are checked against
the oracle as well."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_15319_b200 import binding, workloads as W
import gpu_harness as G

pytestmark = pytest.mark.gpu

LIMIT = 32 << 20


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    c = binding.Context(0)
    yield c
    c.close()


def _static_call(ctx, plan, pool, w, dev="cuda:0"):
    q = binding.to_torch(w.q, w.dtype, dev)
    out = torch.full_like(q, float("nan"))
    lse = torch.full((w.n_heads, max(w.total_q, 1)), float("nan"), dtype=torch.float32, device=dev)
    ctx.slack_chunk_attention_static(plan, pool, q, out, w.scale, lse=lse)
    torch.cuda.synchronize()
    return out.float().cpu().numpy().astype(np.float64), lse.cpu().numpy().astype(np.float64)[:, :w.total_q], ctx.last_launch_count


@pytest.mark.parametrize("make, opts", [
    (lambda: W.small_ragged(page_size=256), {"force_splits": 3}),            # split rows: partial slots + combine
    (lambda: W.sink_ragged(page_size=256), {"force_splits": 2}),
    (lambda: W.small_ragged(head_dim=64, page_size=256), {"force_splits": 2}),
    (lambda: W.small_ragged(), {}),                                          # automatic plan
])
def test_static_workspace_matches_existing_path_twice(ctx, make, opts):
    assert ctx.slack_static_workspace_init() == LIMIT
    w = make()
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    ref, ref_lse, plan, ref_launches = G.gpu_attention(ctx, w, pool, cta_pairs=1, **opts)      # existing path, own workspace
    assert plan.workspace_bytes <= LIMIT
    if opts.get("force_splits", 0) > 1:
        assert plan.num_partial_slots > 0, "the case must use the scratch memory"
    want, want_lse = G.oracle_attention(w)
    for call in range(2):
        out, lse, launches = _static_call(ctx, plan, pool, w)
        assert np.isfinite(out).all(), f"call {call}: unwritten / non-finite output rows"
        assert launches == ref_launches
        ma, rf = oracle.error_metrics(out, ref)
        assert ma <= 2e-2 and rf <= 1e-2, f"call {call}: differs from slack_chunk_attention: max_abs {ma:.3e} rel_fro {rf:.3e}"
        assert np.max(np.abs(lse - ref_lse)) <= 2e-2
        assert np.array_equal(out, ref) and np.array_equal(lse, ref_lse), f"call {call}: same kernels, same plan: same bits"
        G.check_attention(w, out, lse, want, want_lse)


def test_static_workspace_fp8_pool_twice(ctx):
    """FP8 pools keep the quantised Q in the workspace too."""
    w = W.small_ragged(page_size=256)
    pool = G.make_pool_fp8(w)
    G.gpu_append_all(ctx, w, pool)
    ref, ref_lse, plan, _ = G.gpu_attention(ctx, w, pool, force_splits=2)
    assert 0 < plan.workspace_bytes <= LIMIT
    for call in range(2):
        out, lse, _ = _static_call(ctx, plan, pool, w)
        ma, rf = oracle.error_metrics(out, ref)
        assert ma <= 2e-2 and rf <= 1e-2 and np.array_equal(out, ref) and np.array_equal(lse, ref_lse), f"call {call}"


def test_static_workspace_rejects_plans_beyond_the_limit(ctx):
    """A plan whose partials need more than the 32 MiB is refused with SLACK_ENOMEM and a message; nothing is launched and
    `out` is not touched; the same plan runs through slack_chunk_attention with a caller workspace."""
    n = 8
    w = W.make_workload("many_partials", dtype="bf16", n_heads=16, head_dim=128, page_size=256, q_lens=[512] * n,
                        cache_lens=[2000] * n, windows=[0] * n, seed=5, amp=0.5)
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    plan = ctx.slack_plan(pool, w.streams, force_splits=8, cta_pairs=1)
    assert plan.workspace_bytes > LIMIT
    q = binding.to_torch(w.q, w.dtype, "cuda:0")
    out = torch.full_like(q, float("nan"))
    with pytest.raises(binding.SlackError) as e:
        ctx.slack_chunk_attention_static(plan, pool, q, out, w.scale)
    assert e.value.status == binding.SLACK_ENOMEM and "static workspace" in str(e.value)
    torch.cuda.synchronize()
    assert ctx.last_launch_count == 0 and bool(torch.isnan(out.float()).all())
    ws = torch.empty(plan.workspace_bytes, dtype=torch.uint8, device="cuda:0")
    ctx.slack_chunk_attention(plan, pool, q, out, w.scale, workspace=ws)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out.float()).all())
