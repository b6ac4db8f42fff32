"""ORACLE (test infrastructure, not product code) — FP8 attention, SURVEY.md 8(f) NEXT-3.

PAPER.md P:88 knob (4) "quantization mode Q", Q in {FP16, FP8}; "SageAttention2 for online FP8 attention
quantization ... dynamically quantizes and dequantizes activations online without quantizing model weights".  The paper
fixes neither the format nor the scale granularity; reading A19 does (and says why):

  format     OCP FP8 E4M3 ("e4m3fn": 1 sign, 4 exponent bits of bias 7, 3 mantissa bits, subnormals m/8 * 2^-6, no infinity,
             0x7f / 0xff = NaN, largest finite value 448), conversion = round to nearest, ties to even, values beyond the
             range saturate to +-448
  K, V       quantised ONCE, when a chunk is appended to the pool (the pool then holds codes + scales: half the bytes of
             bf16).  One fp32 scale per (physical page, head, 128-slot key block), K and V separately:
                 scale = amax / 448,  amax = max |x| over the tokens THIS append writes into the block, all of head_dim
                 (amax = 0 -> scale = 1),  code = e4m3(fp32(x) / scale)            [both divisions in IEEE fp32]
             An append SETS a block's scale iff none of the stream's earlier tokens [0, cache_len) lies in that block;
             otherwise the block already has a scale (from the append that started it) and the new tokens are quantised
             with the stored one, saturating.  Re-appending the same chunk (a later denoising step) therefore rewrites
             the same scales and codes from the new values; a recycled page's stale scale is replaced by its new owner.
  Q          quantised online inside the attention call, one scale per (query row, head): sq = amax_d |q| / 448 (0 -> 1)
  P          quantised online by the kernel to e4m3 (fp32 accumulation of P V); the row sum uses the unrounded fp32 P

Parity target of the CUDA path = `chunk_attention_fp8`: the DEFINITION (oracle.chunk_attention, fp64) applied to the
DEQUANTISED Q, K, V, with exact P.  The kernel's own rounding of P is then the only modelling difference; its size is
bounded in DESIGN.md and measured by `chunk_attention_fp8(..., quantize_p=True)`, which rounds P the way the algorithm
does in the absence of lazy rescaling (each row's sv-weighted probabilities, largest = 1, times 128, to e4m3).

Pins (tests/test_oracle_fp8_pins.py): all 254 finite codes round-trip; the decoder against the format's definition written
with ldexp; the encoder against an independent pure-Python bit-level encoder (frexp arithmetic), against torch's
float8_e4m3fn cast on in-range values, on every midpoint between neighbouring codes (ties to even) and beyond the range
(saturation); scale = amax/448 and amax -> code 448; the scale-ownership rule on hand-built appends (fresh block, block
continued by a later chunk, re-append, recycled page); dequantised attention == chunk_attention on the dequantised arrays.
"""
from __future__ import annotations

from typing import Optional, Sequence

import numpy as np

from .chunk_attention import chunk_attention, token_positions, to_f64

E4M3_MAX = 448.0
KEY_BLOCK = 128          # slots per scale block = the kernel's key tile (include/slack.h)
P_SHIFT = 128.0          # P is scaled by 2^7 before its e4m3 rounding (largest entry 128 <= 448)


# ----------------------------------------------------------------------------------------------
# the format
# ----------------------------------------------------------------------------------------------

def e4m3_decode(codes: np.ndarray) -> np.ndarray:
    """uint8 e4m3fn codes -> fp64 values (NaN for 0x7f / 0xff), from the bit fields."""
    c = np.asarray(codes, dtype=np.uint8).astype(np.int64)
    sign = np.where(c & 0x80, -1.0, 1.0)
    e = (c >> 3) & 0xF
    m = (c & 0x7).astype(np.float64)
    val = np.where(e == 0, m / 8.0 * 2.0 ** -6, (1.0 + m / 8.0) * np.exp2((e - 7).astype(np.float64)))
    val = np.where((e == 15) & ((c & 0x7) == 7), np.nan, val)
    return sign * val


_GRID = e4m3_decode(np.arange(0, 127, dtype=np.uint8))      # the 127 non-negative finite values, ascending; index = code


def e4m3_encode(x: np.ndarray) -> np.ndarray:
    """Round to the nearest representable value, ties to the even code, |x| beyond 448 (after rounding) -> +-448; NaN ->
    0x7f.  Written as that definition: nearest neighbour on the grid of finite values."""
    x = np.asarray(x, dtype=np.float64)
    a = np.minimum(np.abs(x), E4M3_MAX)
    hi = np.clip(np.searchsorted(_GRID, a, side="left"), 0, 126)         # first grid value >= a
    lo = np.clip(hi - 1, 0, 126)
    d_hi, d_lo = _GRID[hi] - a, a - _GRID[lo]
    pick_hi = (d_hi < d_lo) | ((d_hi == d_lo) & (hi % 2 == 0))
    code = np.where(pick_hi, hi, lo).astype(np.uint8)
    code = np.where(np.signbit(x), code | np.uint8(0x80), code).astype(np.uint8)
    return np.where(np.isnan(x), np.uint8(0x7F), code).astype(np.uint8)


def _f32(x: np.ndarray, dtype: str) -> np.ndarray:
    return to_f64(x, dtype).astype(np.float32)       # bf16 / f32 storage widens exactly


def _scale_of(amax: np.ndarray) -> np.ndarray:
    """amax / 448 in fp32, 1 where amax == 0."""
    amax = np.asarray(amax, dtype=np.float32)
    return np.where(amax > 0, amax / np.float32(E4M3_MAX), np.float32(1.0)).astype(np.float32)


def quantize_with_scale(x_f32: np.ndarray, scale_f32: np.ndarray) -> np.ndarray:
    """e4m3(fp32(x) / scale), the division in IEEE fp32 (what the append kernel must reproduce bit for bit)."""
    return e4m3_encode((np.asarray(x_f32, dtype=np.float32) / np.asarray(scale_f32, dtype=np.float32)).astype(np.float32))


# ----------------------------------------------------------------------------------------------
# Q: per (row, head)
# ----------------------------------------------------------------------------------------------

def quantize_q(q: np.ndarray, dtype: str):
    """q [R, H, D] storage dtype -> (codes uint8 [R, H, D], sq fp32 [R, H])."""
    qf = _f32(q, dtype)
    sq = _scale_of(np.abs(qf).max(axis=2))
    return quantize_with_scale(qf, sq[:, :, None]), sq


# ----------------------------------------------------------------------------------------------
# K, V: quantising append
# ----------------------------------------------------------------------------------------------

def kv_append_fp8(k_codes: np.ndarray, v_codes: np.ndarray, k_scale: np.ndarray, v_scale: np.ndarray,
                  streams: Sequence, k_new: np.ndarray, v_new: np.ndarray, dtype: str) -> None:
    """In place on the pool image: codes uint8 [n_pages, H, P, D], scales fp32 [n_pages, H, P // 128].  k_new / v_new:
    ragged concat [sum Lq, H, D] of `dtype` (bf16 bit patterns or f32).  Follows the header's rule token block by block."""
    page_size = k_codes.shape[2]
    assert page_size % KEY_BLOCK == 0
    row = 0
    for s in streams:
        if s.q_len == 0:
            continue
        table = np.asarray(s.page_table, dtype=np.int64)
        new_pos = token_positions(s, np.arange(s.cache_len, s.cache_len + s.q_len))
        old_blocks = set((token_positions(s, np.arange(0, s.cache_len)) // KEY_BLOCK).tolist())
        for codes, scales, src in ((k_codes, k_scale, k_new), (v_codes, v_scale, v_new)):
            x = _f32(src[row:row + s.q_len], dtype)                       # [Lq, H, D]
            for kb in np.unique(new_pos // KEY_BLOCK):
                sel = np.nonzero(new_pos // KEY_BLOCK == kb)[0]           # tokens of this append in block kb
                page = table[(kb * KEY_BLOCK) // page_size]
                blk = ((kb * KEY_BLOCK) % page_size) // KEY_BLOCK
                if int(kb) not in old_blocks:                             # this append starts the block: it sets the scale
                    scales[page, :, blk] = _scale_of(np.abs(x[sel]).max(axis=(0, 2)))
                sc = scales[page, :, blk]                                 # [H]
                slot = new_pos[sel] % page_size
                codes[page, :, slot, :] = quantize_with_scale(x[sel], sc[None, :, None])
        row += s.q_len


def dequantize_pool(codes: np.ndarray, scales: np.ndarray) -> np.ndarray:
    """[n_pages, H, P, D] fp64 = decode(code) * scale of the slot's 128-slot block (NaN where the code is NaN)."""
    n_pages, H, P, D = codes.shape
    val = e4m3_decode(codes).reshape(n_pages, H, P // KEY_BLOCK, KEY_BLOCK, D)
    return (val * scales.astype(np.float64)[:, :, :, None, None]).reshape(n_pages, H, P, D)


# ----------------------------------------------------------------------------------------------
# attention over the quantised operands
# ----------------------------------------------------------------------------------------------

def chunk_attention_fp8(k_codes, v_codes, k_scale, v_scale, streams: Sequence, q: np.ndarray, scale: float, dtype: str,
                        rows: Optional[Sequence[Optional[np.ndarray]]] = None, quantize_p: bool = False):
    """(out fp64 [sum Lq, H, D], lse fp64 [H, sum Lq]): oracle.chunk_attention on the dequantised Q, K, V (exact P).
    quantize_p: additionally round P as the header says (error-budget variant, small inputs only: per-row Python)."""
    q_codes, sq = quantize_q(q, dtype)
    qd = e4m3_decode(q_codes) * sq.astype(np.float64)[:, :, None]
    kd = dequantize_pool(k_codes, k_scale)
    vd = dequantize_pool(v_codes, v_scale)
    if not quantize_p:
        return chunk_attention(kd, vd, streams, qd, scale, "f64", rows=rows)
    return _attention_p8(k_codes, v_codes, k_scale, v_scale, kd, streams, qd, scale, rows)


def _attention_p8(k_codes, v_codes, k_scale, v_scale, kd, streams, qd, scale, rows):
    """out_i = sum_t P8_t sv_t V8_t / sum_t p_t with P8 = e4m3(128 w_t / max_t w_t) / 128 * max_t w_t / sv_t... written out:
    w_t = p_t * sv_t is what multiplies the V codes; the algorithm rounds w_t / max(w) * 128 to e4m3."""
    from .chunk_attention import gather_kv, visible_tokens
    total_q, H, D = qd.shape
    P = k_codes.shape[2]
    out = np.full((total_q, H, D), np.nan)
    lse = np.full((H, total_q), np.nan)
    v_val = e4m3_decode(v_codes)
    row0 = 0
    for si, s in enumerate(streams):
        if s.q_len == 0:
            continue
        toks = visible_tokens(s)
        pos = token_positions(s, toks)
        table = np.asarray(s.page_table, dtype=np.int64)
        page, blk = table[pos // P], (pos % P) // KEY_BLOCK
        sel = np.arange(s.q_len) if rows is None or rows[si] is None else np.asarray(rows[si], dtype=np.int64)
        k_all = gather_kv(kd, s, toks)
        v_all = gather_kv(v_val, s, toks)
        for h in range(H):
            sv = v_scale[page, h, blk].astype(np.float64)
            for r in sel:
                sc = scale * (k_all[:, h, :] @ qd[row0 + r, h, :])
                m = sc.max()
                p = np.exp(sc - m)
                w = p * sv
                wq = e4m3_decode(e4m3_encode(w / w.max() * P_SHIFT)) / P_SHIFT * w.max()
                out[row0 + r, h, :] = (wq @ v_all[:, h, :]) / p.sum()
                lse[h, row0 + r] = m + np.log(p.sum())
        row0 += s.q_len
    return out, lse
