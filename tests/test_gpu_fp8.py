"""-m gpu parity tests of the FP8 path (PAPER.md P:88 knob (4); rule: include/slack.h slack_dtype,
DESIGN.md A19), through the C ABI against oracle/fp8_attention.py on the same seeded inputs.

* the quantising append is BIT-EXACT: every code and every scale of the whole pool image, untouched bytes included;
* attention is compared with the oracle's definition on the DEQUANTISED Q, K, V (exact P).  The kernel additionally rounds
  P to e4m3 (3 mantissa bits: relative error up to 2^-4, ~2.6 % rms); with the i.i.d. zero-mean V of the synthetic
  workloads that error does not average out RELATIVE to the output (signal and noise both shrink like 1/sqrt(keys)), so the
  gate is rel-Fro <= 4e-2 and max-abs <= 2e-2 (A19 derives it); inputs whose V has a common component are held
  to 5e-3, which is what catches a wrong scale, exponent offset or normalisation."""
import copy

import numpy as np
import pytest
import torch

import oracle
from oracle import fp8_attention as F
from paper_2606_15319_b200 import binding, workloads as W
import gpu_harness as G
from helpers import oracle_pools_fp8

pytestmark = pytest.mark.gpu
TOL = dict(max_abs_tol=2e-2, rel_fro_tol=4e-2, lse_tol=2e-2)


@pytest.fixture(scope="module")
def ctx():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device; the product has no CPU fallback"
    c = binding.Context(0)
    yield c
    c.close()


def assert_pool_equals_oracle(w, pool):
    kc, vc, ks, vs = oracle_pools_fp8(w)
    gk, gv, gks, gvs = G.fp8_pool_images(pool)
    assert np.array_equal(gks, ks, equal_nan=True) and np.array_equal(gvs, vs, equal_nan=True), "scales differ"
    assert np.array_equal(gk, kc) and np.array_equal(gv, vc), "codes differ"


@pytest.mark.parametrize("make", [W.small_ragged, lambda: W.small_ragged(page_size=256), W.sink_ragged, W.gap_ragged,
                                  lambda: W.small_ragged(page_size=512, seed=5)])
def test_quantising_append_bit_exact(ctx, make):
    w = make()
    pool = G.make_pool_fp8(w)
    G.gpu_append_all(ctx, w, pool)
    assert_pool_equals_oracle(w, pool)


def test_append_planned_reappend_and_large_values(ctx):
    """The planned variant writes the same bytes; a later denoising step re-appends other values at the same positions
    (blocks the chunk started get new scales, a block it continues keeps the old one and saturates: 30 x larger values)."""
    w = W.small_ragged()
    pool = G.make_pool_fp8(w)
    plan = ctx.slack_plan(pool, w.streams)
    G.gpu_append_all(ctx, w, pool, planned_plan=plan)
    assert_pool_equals_oracle(w, pool)
    w2 = copy.copy(w)
    big = oracle.to_f64(w.v_new, "bf16").astype(np.float32) * np.float32(30)
    w2.k_new, w2.v_new = W.f32_to_bf16_bits(big), w.k_new
    ctx.slack_kv_append_planned(plan, pool, binding.to_torch(w2.k_new, "bf16", "cuda:0"), binding.to_torch(w2.v_new, "bf16", "cuda:0"))
    torch.cuda.synchronize()
    assert_pool_equals_oracle(w2, pool)
    assert np.isin(G.fp8_pool_images(pool)[0], (0x7E, 0xFE)).any(), "the case must exercise saturation"


def test_append_division_bit_exact_over_extreme_scales(ctx):
    """code = e4m3(fp32(x) / scale) with the IEEE division of the rule, whatever the magnitudes: every fresh 128-token block
    (and head) is scaled by its own power of two from 2^-140 (bf16 denormals: a denormal scale) to 2^120, one block holds
    an infinity, zeros of both signs are sprinkled in, and the 64 tokens that CONTINUE the block started by the earlier
    chunk are spread over 2^-100 .. 2^100 against its stored scale (quotients far above 448, far below the smallest code,
    and everything between).  The kernel shares one reciprocal per thread (quant.cu Divider); the oracle divides."""
    n_blocks = 24
    w = W.make_workload("fp8_scales", dtype="bf16", n_heads=4, head_dim=128, page_size=256, q_lens=[64 + 128 * n_blocks + 40],
                        cache_lens=[64], windows=[0], bases=[0], seed=71, amp=0.5, spare_pages=1)
    rng = np.random.default_rng(72)
    for name in ("k_new", "v_new"):
        x = W.bf16_bits_to_f32(getattr(w, name)).astype(np.float64)                  # [Lq, H, D]
        e_tok = rng.integers(-100, 101, size=(64, w.n_heads, 1))
        x[:64] *= np.exp2(e_tok)
        for b in range(n_blocks + 1):
            e_blk = rng.integers(-140, 121, size=(1, w.n_heads, 1))
            x[64 + 128 * b: 64 + 128 * (b + 1)] *= np.exp2(e_blk)
        z = rng.random(x.shape) < 0.01
        x[z] = np.where(rng.random(int(z.sum())) < 0.5, 0.0, -0.0)
        x[64 + 128 * 3 + 5, 1, 17] = np.inf                                          # amax = inf -> scale = inf -> codes +-0
        x[64 + 128 * 3 + 9, 1, 18] = -np.inf                                         # inf / inf -> the NaN code
        with np.errstate(over="ignore", under="ignore"):
            setattr(w, name, W.f32_to_bf16_bits(x.astype(np.float32)))
    pool = G.make_pool_fp8(w)
    G.gpu_append_all(ctx, w, pool)
    assert_pool_equals_oracle(w, pool)
    codes = G.fp8_pool_images(pool)[0]
    assert np.isin(codes, (0x7E, 0xFE)).any() and np.isin(codes, (0x7F, 0xFF)).any() and (codes == 0x80).any()


def test_append_cfg2_full_size_bit_exact(ctx):
    w = W.config2()
    pool = G.make_pool_fp8(w)
    G.gpu_append_all(ctx, w, pool)
    assert_pool_equals_oracle(w, pool)


def run_fp8(ctx, w, tol=TOL, rows=None, **opts):
    pool = G.make_pool_fp8(w)
    G.gpu_append_all(ctx, w, pool)
    out, lse, plan, launches = G.gpu_attention(ctx, w, pool, **opts)
    kc, vc, ks, vs = oracle_pools_fp8(w)
    want, want_lse = F.chunk_attention_fp8(kc, vc, ks, vs, w.streams, w.q, w.scale, w.dtype, rows=rows)
    res = G.check_attention(w, out, lse, want, want_lse, **tol)
    if rows is None:
        assert np.isfinite(out).all(), f"{w.name}: unwritten / non-finite output rows"
    res.update(kind=plan.kernel_kind, slots=plan.num_partial_slots, launches=launches)
    return res, out, want


@pytest.mark.parametrize("page_size", [128, 256])
@pytest.mark.parametrize("splits", [0, 1, 3])
def test_small_ragged_fp8(ctx, page_size, splits):
    res, *_ = run_fp8(ctx, W.small_ragged(page_size=page_size), force_splits=splits)
    assert res["kind"] == 0 and res["launches"] >= 2          # Q quantiser + attention (+ combine)


@pytest.mark.parametrize("make", [W.sink_ragged, W.gap_ragged])
def test_sink_and_gap_fp8(ctx, make):
    run_fp8(ctx, make(), force_splits=2)


def test_common_component_in_v_is_held_to_half_a_percent(ctx):
    """V = 100 + noise: P's rounding errors average out against the common component, so a wrong V scale, exponent offset
    (the 2^7 shift, log2 sv) or normalisation (1 / (128 l)) shows at the 1e-3 level."""
    w = W.small_ragged(seed=21)
    shift = lambda a: W.f32_to_bf16_bits(oracle.to_f64(a, "bf16").astype(np.float32) + np.float32(100))
    w.v_new = shift(w.v_new)
    w.v_prior = [shift(v) for v in w.v_prior]
    res, out, want = run_fp8(ctx, w, tol=dict(max_abs_tol=1.0, rel_fro_tol=5e-3, lse_tol=2e-2))
    assert abs(np.nanmean(out) - np.nanmean(want)) < 0.2


def test_tile_scales_differ_by_orders_of_magnitude(ctx):
    """Chunks whose K and V magnitudes differ 64 x between key tiles: the per-tile K scale enters the logits, the per-tile V
    scale rides in P's exponent and the row sum is corrected per tile (attn_tc.cu header): any slip shows immediately."""
    w = W.small_ragged(seed=22)
    for arrs in (w.k_prior, w.v_prior):
        for i, a in enumerate(arrs):
            x = oracle.to_f64(a, "bf16").astype(np.float32)
            blk = (np.arange(x.shape[0]) // 128) % 3
            x *= np.where(blk == 0, 1.0, np.where(blk == 1, 8.0, 0.125)).astype(np.float32)[:, None, None]
            arrs[i] = W.f32_to_bf16_bits(x)
    big = dict(TOL, max_abs_tol=0.3)              # outputs reach +-3 here (V x 8): the absolute gate scales with them
    run_fp8(ctx, w, tol=big)
    run_fp8(ctx, w, tol=big, force_splits=3)


def test_adversarial_logits_fp8(ctx):
    """Q x 8 (peaky rows) and a late +30 logit jump: the lazy rescale (threshold 2^1 here) and P's saturation bound."""
    w = W.small_ragged(seed=23)
    w.q = W.f32_to_bf16_bits(oracle.to_f64(w.q, "bf16").astype(np.float32) * np.float32(8))
    # a row that rests on two or three keys is off by up to 2^-4 of a single p * v (|v| up to ~2 here): the absolute gate
    # is widened to 8e-2 for the peaky cases, rel-Fro stays (measured 4.5e-3)
    peaky = dict(TOL, max_abs_tol=8e-2)
    run_fp8(ctx, w, tol=peaky)
    w = W.small_ragged(seed=24)
    kp = oracle.to_f64(w.k_prior[0], "bf16").astype(np.float32)
    qd = oracle.to_f64(w.q, "bf16").astype(np.float32)
    kp[-3:] = qd[0:3] * np.float32(40.0)          # three late keys aligned with three queries: logits far above the rest
    w.k_prior[0] = W.f32_to_bf16_bits(kp)
    run_fp8(ctx, w, tol=peaky)


def test_cfg2_full_size_fp8_sampled_rows(ctx):
    w = W.config2()
    rng = np.random.default_rng(7)
    rows = [np.sort(np.unique(np.concatenate([[0, 127, 128, 4607, 4608, 4679], rng.choice(s.q_len, 90, replace=False)]))) for s in w.streams]
    res, out, want = run_fp8(ctx, w, rows=rows)
    assert np.isfinite(out).all()


def test_cfg5b_shape_fp8_dual_items_full_output(ctx):
    """The decode-like supplementary config's shape (72-query chunks over 8190 keys, 12 heads, P = 256) with 12 streams (the
    oracle dequantises the whole pool image in fp64: 64 streams would need 13 GB), default launch configuration: the plan
    pairs the heads of a stream into dual items; every output row against the FP8 oracle."""
    w = W.config5b(n_streams=12)
    res, out, want = run_fp8(ctx, w)
    pool = G.make_pool_fp8(w)
    items = ctx.slack_plan(pool, w.streams).items()
    assert sum(i["dual"] for i in items) >= len(items) // 4


def test_unsupported_combinations(ctx):
    w = W.small_ragged()
    pool = G.make_pool_fp8(w)
    with pytest.raises(binding.SlackError) as e:
        ctx.slack_plan(pool, w.streams, force_simt=1)
    assert e.value.status == binding.SLACK_EUNSUPPORTED
    w64 = W.small_ragged(page_size=64)
    with pytest.raises(binding.SlackError) as e:
        ctx.slack_plan(binding.Pool.shape_only(w64.n_pages, w64.n_heads, w64.head_dim, 64, "fp8"), w64.streams)
    assert e.value.status == binding.SLACK_EUNSUPPORTED
    bad = binding.Pool(pool.k_pool, pool.v_pool, w.n_pages, w.n_heads, w.head_dim, w.page_size, "fp8")      # no scales
    with pytest.raises(binding.SlackError) as e:
        ctx.slack_kv_append(bad, w.streams, binding.to_torch(w.k_new, "bf16", "cuda:0"), binding.to_torch(w.v_new, "bf16", "cuda:0"))
    assert e.value.status == binding.SLACK_EINVAL


def test_page_transfer_moves_codes_and_scales(ctx):
    """NEXT-4 on an FP8 pool: the listed pages' head slices arrive bit for bit, codes AND block scales, nothing else
    changes; attention through the new page ids gives the same bits as before the move."""
    w = W.small_ragged(page_size=256)
    pool = G.make_pool_fp8(w)
    G.gpu_append_all(ctx, w, pool)
    out0, lse0, plan0, _ = G.gpu_attention(ctx, w, pool, force_splits=1)
    s0 = w.streams[0]
    sp = np.asarray(s0.page_table, dtype=np.int32)
    dst = G.make_pool_fp8(w)                                     # a second pool of the same shape, NaN-filled
    dp = np.random.default_rng(3).permutation(w.n_pages)[:sp.size].astype(np.int32)
    h0, h1 = 0, w.n_heads
    ctx.slack_kv_transfer([pool], [dst], sp, dp, h0, h1)
    torch.cuda.synchronize()
    src_img, dst_img = G.fp8_pool_images(pool), G.fp8_pool_images(dst)
    want = [np.full_like(a, 0x7F) if a.dtype == np.uint8 else np.full_like(a, np.nan) for a in src_img]
    oracle.kv_transfer(src_img[0], src_img[1], want[0], want[1], sp, dp, h0, h1)          # codes
    oracle.kv_transfer(src_img[2], src_img[3], want[2], want[3], sp, dp, h0, h1)          # scales: same slicing rule
    for g, x in zip(dst_img, want):
        assert np.array_equal(g, x, equal_nan=True)
    # a head sub-range moves only that partition
    dst2 = G.make_pool_fp8(w)
    ctx.slack_kv_transfer([pool], [dst2], sp, dp, 1, 2)
    torch.cuda.synchronize()
    want2 = [np.full_like(a, 0x7F) if a.dtype == np.uint8 else np.full_like(a, np.nan) for a in src_img]
    oracle.kv_transfer(src_img[0], src_img[1], want2[0], want2[1], sp, dp, 1, 2)
    oracle.kv_transfer(src_img[2], src_img[3], want2[2], want2[3], sp, dp, 1, 2)
    for g, x in zip(G.fp8_pool_images(dst2), want2):
        assert np.array_equal(g, x, equal_nan=True)
    # stream 0 re-homed alone into `dst`: same attention bits as inside the original batch (force_splits = 1)
    import copy
    s_new = copy.copy(s0)
    s_new.page_table = dp.copy()
    w1 = copy.copy(w)
    w1.streams = [s_new]
    w1.q = w.q[:s0.q_len]
    out1, _, _, _ = G.gpu_attention(ctx, w1, dst, force_splits=1)
    assert np.array_equal(out1, out0[:s0.q_len])


# ------------------------------------------------------------------------------------------------ dual items on FP8 pools
def _decode_like(seed, n=10, heads=4, page_size=128):
    """Many short chunks (1..128 queries) over ragged caches, some windowed, bases anywhere in the first page."""
    rng = np.random.default_rng(seed)
    q = [int(x) for x in rng.integers(1, 129, size=n)]
    c = [int(x) for x in rng.integers(0, 1500, size=n)]
    wdw = [0 if i % 3 else 700 for i in range(n)]
    b = [int(x) for x in rng.integers(0, page_size, size=n)]
    return W.make_workload("decode_like_fp8", dtype="bf16", n_heads=heads, head_dim=128, page_size=page_size, q_lens=q,
                           cache_lens=c, windows=wdw, bases=b, seed=seed, amp=0.5, spare_pages=2)


@pytest.mark.parametrize("seed", [1, 2])
@pytest.mark.parametrize("sm_count", [0, 8, 3])
def test_decode_like_batches_use_dual_items_fp8(ctx, seed, sm_count):
    """Two single-tile items share a CTA on FP8 pools too (each tile slot with its own K/V codes AND its own tile scales)."""
    w = _decode_like(seed)
    res, *_ = run_fp8(ctx, w, sm_count=sm_count)
    pool = G.make_pool_fp8(w)
    items = ctx.slack_plan(pool, w.streams, sm_count=sm_count).items()
    assert sum(i["dual"] for i in items) >= len(items) // 4, "short chunks should pair up"


def test_dual_items_fp8_split_rows_sinks_and_unequal_scales(ctx):
    """Few queues, long caches: dual rows are cut into pieces; the two members' key tiles carry scales 64 x apart."""
    w = W.make_workload("decode_long_fp8", dtype="bf16", n_heads=4, head_dim=128, page_size=256, q_lens=[72, 100, 1, 128],
                        cache_lens=[5000, 5000, 3000, 2500], windows=[0, 4000, 0, 0], bases=[3, 0, 255, 17],
                        sink_lens=[0, 200, 0, 0], seed=9, amp=0.5, spare_pages=1)
    for h in range(w.n_heads):                           # heads pair up inside a stream: give each head its own magnitude
        f = np.float32(8.0 ** (h - 1))
        for arr in [w.k_new, w.v_new] + list(w.k_prior) + list(w.v_prior):
            arr[:, h] = W.f32_to_bf16_bits(W.bf16_bits_to_f32(arr[:, h]) * f)
    w.q = W.f32_to_bf16_bits(W.bf16_bits_to_f32(w.q) * np.float32(0.25))     # keep the logits moderate under the larger K
    # |out| scales with V (x 64 on the last head, whose 16 x larger logits rest on a few keys: the peaky-row bar 8e-2 x 64);
    # rel-Fro binds, and a tile scale taken from the wrong member would be off by 8 x or more
    tol = dict(TOL, max_abs_tol=5.0)
    res, *_ = run_fp8(ctx, w, tol=tol, sm_count=12)
    pool = G.make_pool_fp8(w)
    items = ctx.slack_plan(pool, w.streams, sm_count=12).items()
    assert any(i["dual"] and i["partial_slot"] >= 0 for i in items)


def test_dual_fp8_repeated_launches_are_bit_identical(ctx):
    w = _decode_like(6)
    pool = G.make_pool_fp8(w)
    G.gpu_append_all(ctx, w, pool)
    plan = ctx.slack_plan(pool, w.streams)
    assert any(i["dual"] for i in plan.items())
    q = binding.to_torch(w.q, w.dtype, "cuda:0")
    ws = torch.full((max(plan.workspace_bytes, 16),), 0xFF, dtype=torch.uint8, device="cuda:0")
    ref = None
    for _ in range(20):
        out = torch.full_like(q, float("nan"))
        ws.fill_(0xFF)
        ctx.slack_chunk_attention(plan, pool, q, out, w.scale, workspace=ws)
        torch.cuda.synchronize()
        o = out.view(torch.int16).cpu().numpy()
        ref = o if ref is None else ref
        assert np.array_equal(o, ref)
