"""-m gpu parity tests of the block-sparse variant (slack_chunk_attention_sparse, PAPER.md P:88 knob
(2)) against the oracle's block-sparse definition, element by element, through the C ABI.  Same bars as the dense path:
max-abs <= 2e-2 and relative Frobenius <= 1e-2 (bf16), 1e-5 / 1e-5 on the fp32 SIMT path; rows left without a key must be
exactly 0 with lse = -inf."""
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


def run_sparse(ctx, w, masks, tol=(2e-2, 1e-2), rows=None, extra_words=0, **opts):
    dev = "cuda:0"
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    plan = ctx.slack_plan(pool, w.streams, **opts)
    packed = W.pack_block_masks(w, masks)
    if extra_words:
        packed = np.concatenate([packed, np.full(packed.shape[:2] + (extra_words,), 0xFFFFFFFF, dtype=np.uint32)], axis=2)
    assert packed.shape[0] == plan.mask_rows and packed.shape[2] >= plan.mask_min_words
    mask_d = torch.from_numpy(np.ascontiguousarray(packed).view(np.int32)).to(dev)
    q = binding.to_torch(w.q, w.dtype, dev)
    out = torch.full_like(q, float("nan"))
    lse = torch.full((w.n_heads, max(w.total_q, 1)), float("nan"), dtype=torch.float32, device=dev)
    ws = torch.empty(max(plan.sparse_workspace_bytes, 16), dtype=torch.uint8, device=dev)
    ctx.slack_chunk_attention_sparse(plan, pool, q, out, w.scale, mask_d, lse=lse, workspace=ws)
    torch.cuda.synchronize()
    out_np = out.float().cpu().numpy().astype(np.float64)
    lse_np = lse.cpu().numpy().astype(np.float64)[:, :w.total_q]
    ko, vo = oracle_pools(w, fill=G.host_fill(w))
    want, want_lse = oracle.chunk_attention(ko, vo, w.streams, w.q, w.scale, w.dtype, rows=rows, block_masks=masks)
    empty = np.isneginf(want_lse)                       # [H, rows]
    if empty.any():
        assert np.all(np.isneginf(lse_np[empty])), "rows without a key must report lse = -inf"
        assert np.all(out_np[empty.T] == 0.0), "rows without a key must be exactly 0"
        want_lse = np.where(empty, np.nan, want_lse)    # compared above; exclude from the abs-difference check
        lse_np = np.where(empty, np.nan, lse_np)
    res = G.check_attention(w, out_np, lse_np, want, want_lse, max_abs_tol=tol[0], rel_fro_tol=tol[1])
    if rows is None:
        assert np.isfinite(out_np).all(), f"{w.name}: unwritten / non-finite output rows"
    res.update(kind=plan.kernel_kind, slots=plan.num_partial_slots, empty_rows=int(empty.sum()))
    return res


@pytest.mark.parametrize("rho", [0.0, 0.5, 0.9])
@pytest.mark.parametrize("splits", [0, 1, 3])
def test_small_ragged_sparse(ctx, rho, splits):
    w = W.small_ragged(page_size=256)
    res = run_sparse(ctx, w, W.random_block_masks(w, rho, seed=5), force_splits=splits)
    assert res["kind"] == 0


@pytest.mark.parametrize("page_size", [128, 512])
def test_sink_ragged_sparse(ctx, page_size):
    w = W.sink_ragged(page_size=page_size)
    res = run_sparse(ctx, w, W.random_block_masks(w, 0.6, seed=6), force_splits=2)
    assert res["kind"] == 0


def test_unstructured_masks_with_empty_rows_and_empty_pieces(ctx):
    """Masks drawn without any guarantee: some (query block, head) rows have no selected visible block (-> zeros), and
    with forced splits some pieces of a row have none (-> their partial must weigh nothing in the combine)."""
    w = W.small_ragged(page_size=128, seed=17)
    rng = np.random.default_rng(3)
    masks = []
    for s in w.streams:
        n_qb, n_kb = -(-s.q_len // 256), -(-(s.base + s.n) // 128)
        masks.append(rng.random((w.n_heads, max(n_qb, 1), n_kb)) < 0.25 if s.q_len else None)
    masks[0][:, 0, :] = False                           # a whole query block of stream 0 without keys
    for splits in (1, 4):
        res = run_sparse(ctx, w, masks, force_splits=splits)
        assert res["empty_rows"] >= 256 * w.n_heads


def test_wider_mask_rows_and_invisible_bits(ctx):
    w = W.sink_ragged(page_size=256, seed=19)
    masks = W.random_block_masks(w, 0.5, seed=8)
    for s, m in zip(w.streams, masks):
        inv = np.setdiff1d(np.arange(m.shape[2]), W.visible_key_blocks(s))
        m[:, :, inv] = True                             # bits of blocks without a visible key are ignored
    run_sparse(ctx, w, masks, extra_words=2)


def test_all_ones_mask_equals_dense_call(ctx):
    dev = "cuda:0"
    w = W.small_ragged(page_size=256, seed=23)
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    dense, dense_lse, plan, _ = G.gpu_attention(ctx, w, pool)
    packed = W.pack_block_masks(w, [None] * len(w.streams))
    mask_d = torch.from_numpy(packed.view(np.int32)).to(dev)
    q = binding.to_torch(w.q, w.dtype, dev)
    out = torch.full_like(q, float("nan"))
    ws = torch.empty(max(plan.sparse_workspace_bytes, 16), dtype=torch.uint8, device=dev)
    ctx.slack_chunk_attention_sparse(plan, pool, q, out, w.scale, mask_d, workspace=ws)
    torch.cuda.synchronize()
    assert np.array_equal(out.float().cpu().numpy().astype(np.float64), dense)   # same steps, same order: bit-identical


def test_fp32_simt_sparse(ctx):
    w = W.small_ragged(dtype="f32", head_dim=64, page_size=16, amp=1.0)
    res = run_sparse(ctx, w, W.random_block_masks(w, 0.5, seed=9), tol=(1e-5, 1e-5))
    assert res["kind"] == 1


def test_cfg2_full_size_sparse_full_output(ctx):
    """BASELINE.json configs[1] shape at rho = 0.8, in the launch configuration bench.py --sparsity times: EVERY
    output row against the oracle (every planned item, every partial slot)."""
    w = W.config2()
    masks = W.random_block_masks(w, 0.8, seed=2)
    res = run_sparse(ctx, w, masks)
    assert res["kind"] == 0


def test_sparse_argument_errors(ctx):
    w = W.small_ragged(page_size=256)
    pool = G.make_pool(w)
    plan = ctx.slack_plan(pool, w.streams)
    q = binding.to_torch(w.q, w.dtype, "cuda:0")
    out = torch.empty_like(q)
    packed = W.pack_block_masks(w, [None] * len(w.streams))
    mask_d = torch.from_numpy(packed.view(np.int32)).to("cuda:0")
    with pytest.raises(binding.SlackError):             # workspace too small for the step lists
        ctx.slack_chunk_attention_sparse(plan, pool, q, out, w.scale, mask_d,
                                         workspace=torch.empty(16, dtype=torch.uint8, device="cuda:0"))
    if plan.mask_min_words > 1:
        narrow = mask_d[:, :, :plan.mask_min_words - 1].contiguous()
        ws = torch.empty(plan.sparse_workspace_bytes, dtype=torch.uint8, device="cuda:0")
        with pytest.raises(binding.SlackError):
            ctx.slack_chunk_attention_sparse(plan, pool, q, out, w.scale, narrow, workspace=ws)
