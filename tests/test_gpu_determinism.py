"""-m gpu stress tests standing in for racecheck (compute-sanitizer is not available on the GPU pool): the hot path has
no atomics and a fixed reduction order, so every launch of the same plan on the same inputs must produce the SAME BITS;
a barrier-protocol or shared-memory race shows up as a run that differs.  The split-KV workspace is poisoned with NaN
before every launch, so a partial that is read before it is written (or never written) also shows."""
import numpy as np
import pytest
import torch

from paper_2606_15319_b200 import binding, workloads as W
import gpu_harness as G

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    c = binding.Context(0)
    yield c
    c.close()


def repeat_bits(ctx, w, reps, sparse_rho=None, **opts):
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    plan = ctx.slack_plan(pool, w.streams, **opts)
    q = binding.to_torch(w.q, w.dtype, DEV)
    nbytes = max(plan.sparse_workspace_bytes if sparse_rho is not None else plan.workspace_bytes, 16)
    ws = torch.empty((nbytes + 3) // 4, dtype=torch.float32, device=DEV)
    md = None
    if sparse_rho is not None:
        md = torch.from_numpy(W.pack_block_masks(w, W.random_block_masks(w, sparse_rho, seed=3)).view(np.int32)).to(DEV)
    ref = None
    for r in range(reps):
        ws.fill_(float("nan"))
        out = torch.full_like(q, float("nan"))
        lse = torch.full((w.n_heads, max(w.total_q, 1)), float("nan"), dtype=torch.float32, device=DEV)
        if md is None:
            ctx.slack_chunk_attention(plan, pool, q, out, w.scale, lse=lse, workspace=ws)
        else:
            ctx.slack_chunk_attention_sparse(plan, pool, q, out, w.scale, md, lse=lse, workspace=ws)
        torch.cuda.synchronize()
        bits = (out.view(torch.int16).clone(), lse.view(torch.int32).clone())
        assert torch.isfinite(out.float()).all(), f"run {r}: non-finite output"
        if ref is None:
            ref = bits
        else:
            assert torch.equal(bits[0], ref[0]) and torch.equal(bits[1], ref[1]), f"run {r} differs from run 0"


@pytest.mark.parametrize("splits", [0, 3])
def test_small_batch_is_bitwise_repeatable(ctx, splits):
    repeat_bits(ctx, W.small_ragged(page_size=256), reps=40, force_splits=splits)


def test_sink_and_sparse_are_bitwise_repeatable(ctx):
    repeat_bits(ctx, W.sink_ragged(page_size=256), reps=25, force_splits=2)
    repeat_bits(ctx, W.small_ragged(page_size=256, seed=5), reps=25, sparse_rho=0.6, force_splits=2)


def test_cfg3_full_size_is_bitwise_repeatable(ctx):
    """All 148 queues busy, 1883 items, ragged lengths: six launches, identical bits (values not drawn: the oracle checks
    of test_gpu_full_size.py cover correctness; this one is about run-to-run stability at full occupancy)."""
    import unittest.mock as m
    with m.patch.object(W, "_draw", lambda rng, shape, amp, dtype: np.zeros((0,), dtype=np.uint16)):
        w = W.config3()
    H, D, P = w.n_heads, w.head_dim, w.page_size
    gen = torch.Generator(device=DEV)
    gen.manual_seed(11)
    kp = torch.empty(w.n_pages, H, P, D, device=DEV, dtype=torch.bfloat16)
    vp = torch.empty_like(kp)
    for t in (kp, vp):
        for a in range(0, w.n_pages, 64):
            n = min(64, w.n_pages - a)
            t[a:a + n] = (torch.randn(n, H, P, D, device=DEV, generator=gen) * 0.5).to(torch.bfloat16)
    pool = binding.Pool(kp, vp, w.n_pages, H, D, P, "bf16")
    q = (torch.randn(w.total_q, H, D, device=DEV, generator=gen) * 0.5).to(torch.bfloat16)
    plan = ctx.slack_plan(pool, w.streams)
    ws = torch.empty((max(plan.workspace_bytes, 16) + 3) // 4, dtype=torch.float32, device=DEV)
    ref = None
    for r in range(6):
        ws.fill_(float("nan"))
        out = torch.full_like(q, float("nan"))
        ctx.slack_chunk_attention(plan, pool, q, out, w.scale, workspace=ws)
        torch.cuda.synchronize()
        assert torch.isfinite(out.float()).all()
        bits = out.view(torch.int16).clone()
        if ref is None:
            ref = bits
        else:
            assert torch.equal(bits, ref), f"run {r} differs from run 0"
