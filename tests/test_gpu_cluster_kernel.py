"""-m gpu parity tests of the experimental 2-CTA-cluster attention kernel (csrc/attn_tc2.cu: one query tile per SM,
double-buffered S in TMEM, K/V tiles shared by TMA multicast), selected with slack_debug_set key 2 for plans made for half
the SMs.  Same oracle, same bars as the production kernel."""
import numpy as np
import pytest
import torch

from paper_2606_15319_b200 import binding, workloads as W
import gpu_harness as G

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    c = binding.Context(0)
    c.debug_use_cluster_kernel(True)
    yield c
    c.close()


def run(ctx, w, rows=None, **opts):
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    out, lse, plan, launches = G.gpu_attention(ctx, w, pool, sm_count=74, **opts)
    want, want_lse = G.oracle_attention(w, rows=rows)
    res = G.check_attention(w, out, lse, want, want_lse)
    assert np.isfinite(out).all() and plan.kernel_kind == 0
    return res


@pytest.mark.parametrize("page_size", [128, 256])
@pytest.mark.parametrize("splits", [0, 1, 3])
def test_cluster_kernel_small_ragged(ctx, page_size, splits):
    run(ctx, W.small_ragged(page_size=page_size), force_splits=splits)


def test_cluster_kernel_sink_and_windows(ctx):
    run(ctx, W.sink_ragged(page_size=256), force_splits=2)


def test_cluster_kernel_late_large_logits(ctx):
    w = W.make_workload("late_max", dtype="bf16", n_heads=2, head_dim=128, page_size=128, q_lens=[260], cache_lens=[1500],
                        windows=[0], bases=[3], seed=33, amp=0.5)
    q = W.bf16_bits_to_f32(w.q)
    kn = W.bf16_bits_to_f32(w.k_new)
    for j in (40, 200, 259):
        kn[j] = 24.0 * q[j % 260] / np.maximum(np.linalg.norm(q[j % 260], axis=-1, keepdims=True), 1e-6)
    kn[100] = 300.0 * q[100] / np.maximum(np.linalg.norm(q[100], axis=-1, keepdims=True), 1e-6)
    w.k_new = W.f32_to_bf16_bits(kn)
    run(ctx, w, force_splits=1)


def test_cluster_kernel_cfg2_sampled_rows(ctx):
    w = W.config2()
    rows = [np.unique(np.concatenate([[0, 127, 128, 255, 256, 4607, 4608, 4679], np.random.default_rng(1).integers(0, 4680, size=40)]))]
    run(ctx, w, rows=rows)
