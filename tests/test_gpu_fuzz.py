"""-m gpu randomized parity: seeded random batches (ragged chunk and cache lengths incl. empty ones, windows, sinks, bases
anywhere in the first page, 1-5 heads, head_dim 64 / 128, page sizes 128-512, forced split counts, queue counts) through
the C ABI against the fp64 oracle: append bit-exact, attention at the bars of tests/test_gpu_parity.py.  The hand-built
suites pin the known edge cases; this one guards the combinations nobody thought of.  Every case is reproducible from its
seed (printed in the test id)."""
import numpy as np
import pytest
import torch

from paper_2606_15319_b200 import binding, workloads as W
import gpu_harness as G
from test_gpu_sparse import run_sparse

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    c = binding.Context(0)
    yield c
    c.close()


def random_batch(seed, dtype="bf16"):
    rng = np.random.default_rng(1000 + seed)
    n = int(rng.integers(1, 9))
    page_size = int(rng.choice([128, 256, 512]))
    q_lens, cache_lens, windows, sinks, bases = [], [], [], [], []
    for _ in range(n):
        kind = rng.integers(0, 6)
        q = 0 if kind == 0 else int(rng.choice([1, 72, 127, 128, 129, 255, 256, 257, int(rng.integers(1, 700))]))
        c = 0 if kind == 1 else int(rng.integers(0, 3000))
        total = q + c
        if rng.random() < 0.5 or total == 0:
            wdw, sink = 0, 0
        else:
            wdw = int(rng.integers(max(q, 1), total + 2))              # covers the own chunk, may exceed what is held
            sink = int(rng.choice([0, 0, 1, 16, int(rng.integers(1, 400))]))
        q_lens.append(q); cache_lens.append(c); windows.append(wdw); sinks.append(sink)
        bases.append(int(rng.integers(0, page_size)))
    if sum(q_lens) == 0:
        q_lens[0] = 5
    opts = {"force_splits": int(rng.choice([0, 0, 1, 2, 5])), "sm_count": int(rng.choice([0, 0, 1, 7, 20]))}
    n_heads, head_dim, amp = int(rng.integers(1, 6)), int(rng.choice([64, 128])), float(rng.choice([0.5, 1.0, 2.0]))
    w = W.make_workload(f"fuzz_{seed}", dtype=dtype, n_heads=n_heads, head_dim=head_dim, page_size=page_size, q_lens=q_lens,
                        cache_lens=cache_lens, windows=windows, bases=bases, sink_lens=sinks, seed=seed, amp=amp, spare_pages=2)
    # The 2e-2 max-abs bar is stated for BASELINE's value distribution (amp 0.5: |out| < 2).  With amp 2 the logits have
    # sigma 4, rows rest on a few keys and |out| reaches 6-8, where half an ulp of the bf16 OUTPUT alone is 1.6e-2: the
    # absolute bar scales with the data, the relative one (1e-2) does not.
    return w, opts, 2e-2 * max(1.0, amp)


@pytest.mark.parametrize("seed", range(16))
def test_random_batches_dense(ctx, seed):
    w, opts, max_abs = random_batch(seed)
    pool = G.make_pool(w)
    G.gpu_append_all(ctx, w, pool)
    assert G.pools_equal_oracle(w, pool)
    out, lse, plan, _ = G.gpu_attention(ctx, w, pool, **opts)
    want, want_lse = G.oracle_attention(w)
    G.check_attention(w, out, lse, want, want_lse, max_abs_tol=max_abs)
    assert np.isfinite(out).all(), f"{w.name}: unwritten / non-finite output rows"
    assert plan.kernel_kind in (0, 2)


@pytest.mark.parametrize("seed", range(16, 22))
def test_random_batches_block_sparse(ctx, seed):
    w, opts, max_abs = random_batch(seed)
    rho = [0.3, 0.6, 0.9][seed % 3]
    run_sparse(ctx, w, W.random_block_masks(w, rho, seed=seed), tol=(max_abs, 1e-2), **opts)


@pytest.mark.parametrize("seed", range(22, 28))
def test_random_batches_fp8(ctx, seed):
    from oracle import fp8_attention as F
    from helpers import oracle_pools_fp8
    w, opts, _ = random_batch(seed)
    for retry in range(1, 8):                           # FP8 pools are head_dim 128 only: take the next seed that has it
        if w.head_dim == 128:
            break
        w, opts, _ = random_batch(seed + 100 * retry)
    assert w.head_dim == 128
    pool = G.make_pool_fp8(w)
    G.gpu_append_all(ctx, w, pool)
    img = oracle_pools_fp8(w)
    assert all(np.array_equal(a, b, equal_nan=True) for a, b in zip(G.fp8_pool_images(pool), img)), "FP8 append is not bit-exact"
    out, lse, plan, _ = G.gpu_attention(ctx, w, pool, **opts)
    want, want_lse = F.chunk_attention_fp8(*img, w.streams, w.q, w.scale, w.dtype)
    # amp 2 makes rows that rest on 2-3 keys: the peaky-row bar of tests/test_gpu_fp8.py
    G.check_attention(w, out, lse, want, want_lse, max_abs_tol=8e-2 * max(1.0, float(np.abs(want[np.isfinite(want)]).max())),
                      rel_fro_tol=4e-2, lse_tol=2e-2)
    assert np.isfinite(out).all()
