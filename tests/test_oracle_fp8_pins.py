"""Pins of the FP8 oracle (oracle/fp8_attention.py, PAPER.md P:88 knob (4)), CPU only.
Every pin compares against something other than the oracle's own code: the format's definition written with ldexp, an
independent pure-Python bit-level encoder (frexp arithmetic), torch's float8_e4m3fn cast, hand-built appends."""
import copy
import math

import numpy as np
import pytest
import torch

import oracle
from oracle import fp8_attention as F
from paper_2606_15319_b200 import workloads as W
from helpers import oracle_pools_fp8


# ------------------------------------------------------------------------------------------------ the format
def value_by_definition(code: int) -> float:
    """OCP FP8 E4M3 ("fn" variant): bias 7, subnormals at exponent field 0, no infinity, S.1111.111 = NaN, max 448."""
    s, e, m = code >> 7, (code >> 3) & 0xF, code & 7
    if e == 15 and m == 7:
        return math.nan
    v = math.ldexp(m, -9) if e == 0 else math.ldexp(8 + m, e - 10)
    return -v if s else v


def test_decode_matches_the_format_definition():
    got = F.e4m3_decode(np.arange(256, dtype=np.uint8))
    for c in range(256):
        want = value_by_definition(c)
        assert (math.isnan(want) and math.isnan(got[c])) or got[c] == want, c
    assert got[0x7E] == 448.0 and got[0x01] == 2.0 ** -9 and got[0x08] == 2.0 ** -6 and got[0x38] == 1.0


def test_every_finite_code_round_trips():
    codes = np.array([c for c in range(256) if c not in (0x7F, 0xFF)], dtype=np.uint8)
    back = F.e4m3_encode(F.e4m3_decode(codes))
    # -0 keeps its sign bit
    assert np.array_equal(back, codes)


def encode_bit_level(x: float) -> int:
    """Independent encoder: exponent / mantissa arithmetic with math.frexp and exact integer rounding (ties to even)."""
    if math.isnan(x):
        return 0x7F
    sign = 0x80 if math.copysign(1.0, x) < 0 else 0
    a = abs(x)
    if a == 0:
        return sign
    mant, exp = math.frexp(a)                 # a = mant * 2^exp, mant in [0.5, 1)
    e = exp - 1                               # a = (2 mant) * 2^e, 2 mant in [1, 2)
    q_exp = max(e, -6) - 3                    # spacing of representable values around a: 2^(e-3), or 2^-9 below 2^-6
    n = a / math.ldexp(1.0, q_exp)            # exact (power of two)
    lo = math.floor(n)
    frac = n - lo
    k = lo + (1 if frac > 0.5 or (frac == 0.5 and lo % 2 == 1) else 0)     # integer multiples of the spacing
    val = k * math.ldexp(1.0, q_exp)
    if val > 448.0:
        val = 448.0
    # val -> fields
    if val < 2.0 ** -6:
        return sign | int(round(val / 2.0 ** -9))
    m2, e2 = math.frexp(val)
    ee = e2 - 1
    return sign | ((ee + 7) << 3) | int(round((m2 * 2 - 1) * 8))


def test_encoder_against_bit_level_encoder_and_ties():
    rng = np.random.default_rng(0)
    xs = np.concatenate([rng.standard_normal(4000) * 3, rng.standard_normal(2000) * 300, rng.standard_normal(2000) * 1e-2,
                         rng.standard_normal(500) * 1e-4, np.array([0.0, -0.0, 448.0, 449.0, 464.0, 465.0, 1e9, -1e9, 2.0 ** -10, 2.0 ** -10 * 1.0001])])
    grid = F.e4m3_decode(np.arange(0, 127, dtype=np.uint8))
    mids = (grid[:-1] + grid[1:]) / 2                       # exact ties between neighbours
    xs = np.concatenate([xs, mids, -mids, np.nextafter(mids, 0), np.nextafter(mids, 1e9)])
    got = F.e4m3_encode(xs)
    want = np.array([encode_bit_level(float(v)) for v in xs], dtype=np.uint8)
    assert np.array_equal(got, want)
    # ties go to the even code: the midpoint of codes c and c+1 encodes to whichever is even
    tie = F.e4m3_encode(mids)
    assert np.all(tie % 2 == 0)
    assert F.e4m3_encode(np.array([np.nan]))[0] == 0x7F


def test_encoder_against_torch_cast_in_range():
    rng = np.random.default_rng(1)
    x = (rng.standard_normal(20000) * np.exp(rng.uniform(-8, 5, 20000))).astype(np.float32)
    x = x[np.abs(x) <= 448]
    want = torch.from_numpy(x).to(torch.float8_e4m3fn).view(torch.uint8).numpy()
    assert np.array_equal(F.e4m3_encode(x), want)


def test_saturation():
    assert list(F.e4m3_encode(np.array([448.0, 460.0, 1e6, np.inf, -1e6, -np.inf]))) == [0x7E, 0x7E, 0x7E, 0x7E, 0xFE, 0xFE]


# ------------------------------------------------------------------------------------------------ scales
def test_q_scale_is_amax_over_448_and_amax_maps_to_448():
    rng = np.random.default_rng(2)
    q = rng.standard_normal((5, 3, 16)).astype(np.float32)
    q[2, 1] = 0.0                                                 # an all-zero row: scale 1, codes 0
    codes, sq = F.quantize_q(q, "f32")
    amax = np.abs(q).max(axis=2)
    assert np.array_equal(sq, np.where(amax > 0, amax / np.float32(448), np.float32(1)).astype(np.float32))
    vals = F.e4m3_decode(codes)
    assert np.all(np.abs(vals).max(axis=2)[amax > 0] == 448.0)
    assert np.all(codes[2, 1] == 0) and sq[2, 1] == 1.0
    # dequantised error of every element is within half a grid step at its magnitude (relative 2^-4 for normal values)
    deq = vals * sq[:, :, None]
    assert np.all(np.abs(deq - q) <= np.maximum(np.abs(q) * 2.0 ** -4, sq[:, :, None] * 2.0 ** -10) * 1.0001)


def _one_stream(q_len, cache_len, base=0, pages=4, page_size=256, seed=0, sink=0, gap=0):
    w = W.make_workload("t", dtype="bf16", n_heads=2, head_dim=16, page_size=page_size, q_lens=[q_len], cache_lens=[cache_len],
                        windows=[0], bases=[base], sink_lens=[sink], gap_slots=[gap], seed=seed, amp=1.0, n_pages=pages)
    return w


def test_append_sets_or_keeps_block_scales():
    """Hand-checked ownership rule: a first chunk of 200 tokens at base 40 starts blocks 0 and 1 (positions 40..239); the
    next chunk of 100 tokens (positions 240..339) CONTINUES block 1 (keeps its scale, saturating) and starts block 2."""
    w1 = _one_stream(300, 0, base=40, seed=3)                                # the table covers both chunks (2 pages)
    s = copy.copy(w1.streams[0]); s.q_len = 200
    w1.streams, w1.k_new, w1.v_new = [s], w1.k_new[:200], w1.v_new[:200]
    shape = (w1.n_pages, 2, 256, 16)
    kc = np.full(shape, 0x7F, np.uint8); vc = kc.copy()
    ks = np.full((w1.n_pages, 2, 2), np.nan, np.float32); vs = ks.copy()
    F.kv_append_fp8(kc, vc, ks, vs, w1.streams, w1.k_new, w1.v_new, "bf16")
    x = oracle.to_f64(w1.k_new, "bf16").astype(np.float32)
    page0 = int(s.page_table[0])
    # block 0 holds tokens 0..87 (positions 40..127), block 1 tokens 88..199
    for h in range(2):
        assert ks[page0, h, 0] == np.abs(x[:88, h]).max() / np.float32(448)
        assert ks[page0, h, 1] == np.abs(x[88:, h]).max() / np.float32(448)
    assert np.isnan(ks[int(s.page_table[1]), 0, 0])                        # untouched block: untouched scale
    # slot of token 0 is 40; its code is e4m3(x / scale of block 0)
    want = F.e4m3_encode(x[0, 1] / ks[page0, 1, 0])
    assert np.array_equal(kc[page0, 1, 40], want)
    assert np.all(kc[page0, :, :40] == 0x7F) and np.all(kc[page0, :, 240:] == 0x7F)   # nothing else written
    # second chunk, 10 x larger values: block 1 keeps its scale (codes saturate), block 2 (page 1, block 0) gets its own
    s2 = copy.copy(s); s2.cache_len, s2.q_len = 200, 100
    big = W.f32_to_bf16_bits((np.random.default_rng(4).standard_normal((100, 2, 16)) * 10).astype(np.float32))
    keep = ks.copy()
    F.kv_append_fp8(kc, vc, ks, vs, [s2], big, big, "bf16")
    assert np.array_equal(ks[page0], keep[page0])
    xb = oracle.to_f64(big, "bf16").astype(np.float32)
    page1 = int(s.page_table[1])
    assert ks[page1, 0, 0] == np.abs(xb[16:, 0]).max() / np.float32(448)   # tokens 216.. of the stream = rows 16.. of the chunk
    assert np.any(np.isin(kc[page0, :, 240:256], (0x7E, 0xFE)))            # saturated against the older, smaller scale
    # re-append of the same chunk with other values (a later denoising step) rewrites scales and codes from the new values
    again = W.f32_to_bf16_bits((np.random.default_rng(5).standard_normal((100, 2, 16))).astype(np.float32))
    F.kv_append_fp8(kc, vc, ks, vs, [s2], again, again, "bf16")
    xa = oracle.to_f64(again, "bf16").astype(np.float32)
    assert ks[page1, 1, 0] == np.abs(xa[16:, 1]).max() / np.float32(448)
    assert np.array_equal(ks[page0], keep[page0])


def test_recycled_page_gets_a_new_scale():
    w = _one_stream(128, 0, seed=6)
    kc = np.full((w.n_pages, 2, 256, 16), 0x11, np.uint8); vc = kc.copy()
    ks = np.full((w.n_pages, 2, 2), 123.0, np.float32); vs = ks.copy()       # stale scales of a previous owner
    F.kv_append_fp8(kc, vc, ks, vs, w.streams, w.k_new, w.v_new, "bf16")
    p0 = int(w.streams[0].page_table[0])
    x = oracle.to_f64(w.k_new, "bf16").astype(np.float32)
    assert ks[p0, 0, 0] == np.abs(x[:, 0]).max() / np.float32(448) and ks[p0, 0, 1] == 123.0


def test_halves_equal_whole_when_blocks_are_not_split():
    """Appending a chunk in two calls cut at a block boundary gives the same pool as one call (blocks are independent);
    cut inside a block the second part inherits the first part's scale (so the pools may differ: that is the rule)."""
    w = _one_stream(384, 0, seed=7)
    s = w.streams[0]
    one = oracle_pools_fp8(w)
    kc = np.full_like(one[0], 0x7F); vc = kc.copy()
    ks = np.full_like(one[2], np.nan); vs = ks.copy()
    a = copy.copy(s); a.q_len = 256
    b = copy.copy(s); b.cache_len, b.q_len = 256, 128
    F.kv_append_fp8(kc, vc, ks, vs, [a], w.k_new[:256], w.v_new[:256], "bf16")
    F.kv_append_fp8(kc, vc, ks, vs, [b], w.k_new[256:], w.v_new[256:], "bf16")
    for x, y in zip(one, (kc, vc, ks, vs)):
        assert np.array_equal(x, y, equal_nan=True)


# ------------------------------------------------------------------------------------------------ attention
def test_attention_is_the_definition_on_dequantised_operands():
    w = W.small_ragged(head_dim=16, n_heads=2, page_size=128)
    kc, vc, ks, vs = oracle_pools_fp8(w)
    out, lse = F.chunk_attention_fp8(kc, vc, ks, vs, w.streams, w.q, w.scale, w.dtype)
    # the same through independent steps: dequantise by hand, call the bf16-path oracle with fp64 operands
    qc, sq = F.quantize_q(w.q, w.dtype)
    qd = np.array([[value_by_definition(int(c)) for c in row] for row in qc.reshape(-1, 16)]).reshape(qc.shape) * sq[:, :, None]
    kd = F.dequantize_pool(kc, ks); vd = F.dequantize_pool(vc, vs)
    want, want_lse = oracle.chunk_attention(kd, vd, w.streams, qd, w.scale, "f64")
    assert np.array_equal(out, want) and np.array_equal(lse, want_lse)
    # quantisation error against the unquantised oracle stays at the few-percent level e4m3 allows (3 mantissa bits)
    from helpers import oracle_pools
    ko, vo = oracle_pools(w)
    ref, _ = oracle.chunk_attention(ko, vo, w.streams, w.q, w.scale, w.dtype)
    _, rf = oracle.error_metrics(out, ref)
    assert 1e-3 < rf < 6e-2
    # rounding P to e4m3 as the kernel does moves the result by less than the tolerance of the GPU parity test
    outp, _ = F.chunk_attention_fp8(kc, vc, ks, vs, w.streams, w.q, w.scale, w.dtype, quantize_p=True)
    _, rfp = oracle.error_metrics(outp, out)
    assert 0 < rfp < 3e-2


def test_dequantised_pool_reads_back_within_half_a_step():
    w = W.small_ragged(head_dim=16, n_heads=2, page_size=128)
    kc, vc, ks, vs = oracle_pools_fp8(w)
    kd = F.dequantize_pool(kc, ks)
    r = 0
    for s in w.streams:
        if s.q_len:
            got = oracle.gather_kv(kd, s, np.arange(s.cache_len, s.cache_len + s.q_len))
            want = oracle.to_f64(w.k_new[r:r + s.q_len], w.dtype)
            assert np.all(np.isfinite(got))
            # new-chunk tokens in blocks the chunk started are within 2^-4 relative / half a subnormal step; tokens that
            # continue an older block may saturate, so only a loose bound holds for them
            assert np.median(np.abs(got - want) / np.maximum(np.abs(want), 1e-3)) < 2.0 ** -4
        r += s.q_len
