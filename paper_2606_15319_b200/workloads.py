"""Seeded synthetic workload generators (shared by the oracle tests, the GPU tests and bench.py).

This module holds NONE of the method's arithmetic: it draws random numbers, rounds them to the
storage dtype, picks chunk/cache lengths and hands out physical page ids.  The token->slot rule,
the append and the attention live in `oracle/` (CPU, fp64) and in `csrc/` (CUDA) separately.

Shapes follow BASELINE.json configs 1-5 (B:cfgN) and SURVEY.md §8(d); the paper itself fixes only
"three latent frames per chunk, 480p" (§7.1, App. B) and the rolling window of
W in {1,3,7} chunks (§2.1, App. A).  Everything is i.i.d. Gaussian and stands in for
real AR-DiT activations (the paper's VBench prompts / weights are not available and not needed:
the path's cost and its correctness depend on shapes only).

Storage dtypes: "f32" arrays are numpy float32; "bf16" arrays are numpy uint16 holding the
bfloat16 bit pattern (numpy has no bf16), produced by round-to-nearest-even from float32.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np

# geometry the configs are built from (B:cfg1, B:cfg2, B:cfg4; "three latent frames")
FRAMES_PER_CHUNK = 3
FULL_RES_FRAME_TOKENS = 30 * 52      # 480p latent frame, Wan-1.3B-like (B:cfg2)
LOW_RES_FRAME_TOKENS = 15 * 26       # low-fidelity stream (B:cfg4)
TINY_FRAME_TOKENS = 4 * 6            # B:cfg1
WINDOW_FRAMES = 21                   # B:cfg4 "rolling window capped at 21 latent frames" = 7 chunks (P:568 W=7)
FULL_RES_CHUNK = FRAMES_PER_CHUNK * FULL_RES_FRAME_TOKENS   # 4680
LOW_RES_CHUNK = FRAMES_PER_CHUNK * LOW_RES_FRAME_TOKENS     # 1170
TINY_CHUNK = FRAMES_PER_CHUNK * TINY_FRAME_TOKENS           # 72
N_LAYERS = 30                        # B:cfg5 "30-layer loop"


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """Round float32 -> bfloat16 (round-to-nearest-even), returned as uint16 bit patterns."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    rounded = u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))
    return (rounded >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    """Exact widening of bfloat16 bit patterns to float32 (for handing data to torch / printing)."""
    return (np.ascontiguousarray(b, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


@dataclass
class StreamSpec:
    """One stream of the batch, in the vocabulary of include/slack.h (slack_stream)."""
    q_len: int                 # Lq: tokens of the new chunk
    cache_len: int             # Lc: tokens of earlier chunks held for this stream
    base: int                  # slot of logical token 0 inside page_table[0]
    window: int                # Wt: max visible keys including the own chunk; 0 = unlimited
    sink_len: int              # leading tokens always visible ("sink + local"); 0 in all configs
    page_table: np.ndarray     # int32 [n_table_pages], logical page -> physical page
    gap_slots: int = 0         # unused slots between the sink and the first held token behind it (include/slack.h)

    @property
    def n(self) -> int:
        return self.cache_len + self.q_len


@dataclass
class Workload:
    name: str
    dtype: str                 # "bf16" | "f32"
    n_heads: int
    head_dim: int
    page_size: int
    n_pages: int
    scale: float
    streams: List[StreamSpec]
    q: np.ndarray              # [sum Lq, H, D] storage dtype
    k_new: np.ndarray          # [sum Lq, H, D]
    v_new: np.ndarray          # [sum Lq, H, D]
    k_prior: List[np.ndarray] = field(default_factory=list)   # per stream [Lc, H, D]
    v_prior: List[np.ndarray] = field(default_factory=list)
    seed: int = 0

    @property
    def storage(self):
        return np.uint16 if self.dtype == "bf16" else np.float32

    @property
    def total_q(self) -> int:
        return int(sum(s.q_len for s in self.streams))


def _draw(rng: np.random.Generator, shape, amp: float, dtype: str) -> np.ndarray:
    x = rng.standard_normal(shape, dtype=np.float32)
    if amp != 1.0:
        x *= np.float32(amp)
    return f32_to_bf16_bits(x) if dtype == "bf16" else x


def make_workload(name: str, *, dtype: str, n_heads: int, head_dim: int, page_size: int,
                  q_lens: Sequence[int], cache_lens: Sequence[int], windows: Sequence[int],
                  bases: Optional[Sequence[int]] = None, sink_lens: Optional[Sequence[int]] = None,
                  gap_slots: Optional[Sequence[int]] = None,
                  seed: int = 0, amp: float = 1.0, shuffle_pages: bool = True,
                  spare_pages: int = 0, scale: Optional[float] = None,
                  n_pages: Optional[int] = None) -> Workload:
    """General generator: draws Q/K/V and hands every stream disjoint physical pages.

    Pages come from one global random permutation of the pool (rng seed+7) unless
    shuffle_pages is False (identity order, B:cfg1).  The pool gets `spare_pages` extra pages that
    no stream owns (tests fill them with sentinels / NaNs).
    """
    n_streams = len(q_lens)
    bases = list(bases) if bases is not None else [0] * n_streams
    sink_lens = list(sink_lens) if sink_lens is not None else [0] * n_streams
    gaps = list(gap_slots) if gap_slots is not None else [0] * n_streams
    need = [-(-(bases[i] + gaps[i] + cache_lens[i] + q_lens[i]) // page_size) for i in range(n_streams)]
    total = int(sum(need)) + int(spare_pages)
    if n_pages is None:
        n_pages = max(total, 1)
    assert n_pages >= total, "pool too small for the requested streams"
    prng = np.random.default_rng(seed + 7)
    order = prng.permutation(n_pages) if shuffle_pages else np.arange(n_pages)
    rng = np.random.default_rng(seed)
    streams, k_prior, v_prior = [], [], []
    at = 0
    for i in range(n_streams):
        table = np.ascontiguousarray(order[at:at + need[i]], dtype=np.int32)
        at += need[i]
        streams.append(StreamSpec(int(q_lens[i]), int(cache_lens[i]), int(bases[i]), int(windows[i]),
                                  int(sink_lens[i]), table, int(gaps[i])))
    tq = int(sum(q_lens))
    q = _draw(rng, (tq, n_heads, head_dim), amp, dtype)
    k_new = _draw(rng, (tq, n_heads, head_dim), amp, dtype)
    v_new = _draw(rng, (tq, n_heads, head_dim), amp, dtype)
    for i in range(n_streams):
        k_prior.append(_draw(rng, (int(cache_lens[i]), n_heads, head_dim), amp, dtype))
        v_prior.append(_draw(rng, (int(cache_lens[i]), n_heads, head_dim), amp, dtype))
    if scale is None:
        scale = 1.0 / float(np.sqrt(head_dim))
    return Workload(name, dtype, n_heads, head_dim, page_size, int(n_pages), float(scale), streams,
                    q, k_new, v_new, k_prior, v_prior, seed)


# ----------------------------------------------------------------------------------------------
# BASELINE.json configs
# ----------------------------------------------------------------------------------------------

def config1(seed: int = 0) -> Workload:
    """B:cfg1 tiny reference: 1 stream, H=2, D=64, fp32, 72 queries, 144 cached, P=16, identity table."""
    return make_workload("cfg1_tiny_fp32", dtype="f32", n_heads=2, head_dim=64, page_size=16,
                         q_lens=[TINY_CHUNK], cache_lens=[2 * TINY_CHUNK], windows=[0], seed=seed,
                         amp=1.0, shuffle_pages=False)


def config2(seed: int = 2000, layer: int = 0) -> Workload:
    """B:cfg2 single Wan-1.3B-like stream: H=12, D=128, bf16, 4680 queries, 4 prior chunks, P=256,
    92 pages drawn from a shuffled 128-page pool."""
    return make_workload(f"cfg2_single_stream_L{layer}", dtype="bf16", n_heads=12, head_dim=128,
                         page_size=256, q_lens=[FULL_RES_CHUNK], cache_lens=[4 * FULL_RES_CHUNK],
                         windows=[0], seed=seed + layer, amp=0.5, n_pages=128)


def config3(seed: int = 3000, layer: int = 0) -> Workload:
    """B:cfg3 ragged batch of 8 streams, prior chunks ~ U{0..6}."""
    priors = np.random.default_rng(seed + 7).integers(0, 7, size=8)
    return make_workload(f"cfg3_ragged8_L{layer}", dtype="bf16", n_heads=12, head_dim=128, page_size=256,
                         q_lens=[FULL_RES_CHUNK] * 8, cache_lens=[int(p) * FULL_RES_CHUNK for p in priors],
                         windows=[0] * 8, seed=seed + layer, amp=0.5, spare_pages=16)


def config4(seed: int = 4000, layer: int = 0) -> Workload:
    """B:cfg4 mixed fidelity: 8 full-res + 8 low-res streams, 21-frame rolling window, priors ~ U{0..7}
    (reading A3: 7 priors leaves the oldest chunk resident but outside the window)."""
    priors = np.random.default_rng(seed + 7).integers(0, 8, size=16)
    q_lens = [FULL_RES_CHUNK] * 8 + [LOW_RES_CHUNK] * 8
    windows = [WINDOW_FRAMES * FULL_RES_FRAME_TOKENS] * 8 + [WINDOW_FRAMES * LOW_RES_FRAME_TOKENS] * 8
    return make_workload(f"cfg4_mixed16_L{layer}", dtype="bf16", n_heads=12, head_dim=128, page_size=256,
                         q_lens=q_lens, cache_lens=[int(p) * q for p, q in zip(priors, q_lens)],
                         windows=windows, seed=seed + layer, amp=0.5, spare_pages=16)


def config5(kv_chunks: int = 7, seed: int = 5000, layer: int = 0) -> Workload:
    """B:cfg5 long-cache point: 4 streams, Lk = kv_chunks*4680 (1..7), full 21-frame window."""
    assert 1 <= kv_chunks <= 7
    return make_workload(f"cfg5_long4_k{kv_chunks}_L{layer}", dtype="bf16", n_heads=12, head_dim=128,
                         page_size=256, q_lens=[FULL_RES_CHUNK] * 4,
                         cache_lens=[(kv_chunks - 1) * FULL_RES_CHUNK] * 4,
                         windows=[WINDOW_FRAMES * FULL_RES_FRAME_TOKENS] * 4, seed=seed + layer, amp=0.5)


def config5b(seed: int = 5500, n_streams: int = 64) -> Workload:
    """Supplementary decode-like case: 64 streams, 72-query chunks, 8190 keys."""
    return make_workload("cfg5b_decode_like", dtype="bf16", n_heads=12, head_dim=128, page_size=256,
                         q_lens=[TINY_CHUNK] * n_streams, cache_lens=[8190 - TINY_CHUNK] * n_streams,
                         windows=[0] * n_streams, seed=seed, amp=0.5)


def small_ragged(seed: int = 11, dtype: str = "bf16", n_heads: int = 2, head_dim: int = 128,
                 page_size: int = 128, amp: float = 0.5) -> Workload:
    """Parity-test sized ragged batch the oracle finishes in seconds: spans several 128-row tiles with
    ragged tails, a Lq=1 stream, a Lq=129 stream, an empty cache, a mid-page base and a clipped window."""
    q_lens = [300, 1, 129, 72, 257, 0, 128]
    cache_lens = [517, 700, 0, 1000, 255, 64, 384]
    windows = [0, 0, 0, 600, 400, 0, 0]
    bases = [0, 5, 127 % page_size, 77 % page_size, 1, 0, 0]
    return make_workload(f"small_ragged_{dtype}", dtype=dtype, n_heads=n_heads, head_dim=head_dim,
                         page_size=page_size, q_lens=q_lens, cache_lens=cache_lens, windows=windows,
                         bases=bases, seed=seed, amp=amp, spare_pages=3)


def sink_ragged(seed: int = 13, dtype: str = "bf16", n_heads: int = 2, head_dim: int = 128,
                page_size: int = 128, amp: float = 0.5) -> Workload:
    """"Sink + local" cases: windows that have moved past the sink (two visible ranges, the
    sink ending mid-tile and sharing / not sharing a tile with the window start), a sink the window still touches
    (one range), a sink longer than the stream, and a stream without sink in the same batch."""
    q_lens = [300, 129, 72, 257, 128, 64]
    cache_lens = [1517, 900, 1000, 255, 2000, 300]
    windows = [600, 400, 300, 400, 512, 0]
    sink_lens = [72, 200, 1, 300, 4096, 16]
    bases = [0, 5, 77 % page_size, 1, 0, 3]
    return make_workload(f"sink_ragged_{dtype}", dtype=dtype, n_heads=n_heads, head_dim=head_dim,
                         page_size=page_size, q_lens=q_lens, cache_lens=cache_lens, windows=windows,
                         bases=bases, sink_lens=sink_lens, seed=seed, amp=amp, spare_pages=3)


def gap_ragged(seed: int = 17, dtype: str = "bf16", n_heads: int = 2, head_dim: int = 128,
               page_size: int = 128, amp: float = 0.5) -> Workload:
    """Bounded "sink + local" caches whose out-of-window tokens were dropped (gap_slots, include/slack.h): a hole that
    ends mid-tile, a hole of less than a tile with sink and window in the same 128-position tile, a hole in a one-page
    sink, a window that still covers everything held, plus a stream without sink in the same batch."""
    q_lens = [300, 129, 72, 257, 64]
    cache_lens = [900, 700, 500, 1300, 300]          # held tokens (sink included)
    windows = [700, 0, 400, 1557, 0]
    sink_lens = [72, 200, 1, 300, 0]
    gaps = [312, 17, 127, 84, 0]
    bases = [0, 5, 77 % page_size, 1, 3]
    return make_workload(f"gap_ragged_{dtype}", dtype=dtype, n_heads=n_heads, head_dim=head_dim,
                         page_size=page_size, q_lens=q_lens, cache_lens=cache_lens, windows=windows,
                         bases=bases, sink_lens=sink_lens, gap_slots=gaps, seed=seed, amp=amp, spare_pages=3)


# ----------------------------------------------------------------------------------------------
# block-sparse masks (P:88 knob (2), rho in {0,.6,.7,.8,.9} P:568)
# ----------------------------------------------------------------------------------------------
# Geometry of the mask INPUT as include/slack.h publishes it: one bit per (head, 256-row query block, 128-position key
# block); key block kb covers positions [128 kb, 128 kb + 128) of the stream's page-table space (position = base + token).
MASK_BLOCK_Q = 256
MASK_BLOCK_K = 128


def visible_positions(s) -> np.ndarray:
    """Positions (page-table space, include/slack.h) of the keys a stream's chunk may use: bookkeeping for placing mask
    bits and counting flops only; the attention itself is defined in oracle/ and csrc/ separately."""
    n = s.cache_len + s.q_len
    lo = max(0, n - s.window) if s.window > 0 else 0
    sink = min(s.sink_len, n)
    lo = max(lo, sink)
    gap = getattr(s, "gap_slots", 0)
    return np.concatenate([s.base + np.arange(0, sink, dtype=np.int64), s.base + gap + np.arange(lo, n, dtype=np.int64)])


def visible_key_blocks(s: StreamSpec, block_k: int = MASK_BLOCK_K) -> np.ndarray:
    """Indices of the key blocks that hold at least one visible position of the stream (sink range, then window range)."""
    return np.unique(visible_positions(s) // block_k)


def random_block_masks(w: Workload, sparsity: float, seed: int = 0, block_q: int = MASK_BLOCK_Q,
                       block_k: int = MASK_BLOCK_K, keep_last: bool = True) -> List[Optional[np.ndarray]]:
    """Seeded stand-in for a block-selection rule (the paper's is Light Forcing's [39], not available): per
    stream a boolean array [H, ceil(Lq/block_q), ceil((base+n)/block_k)]; for every (head, query block) a fraction
    `sparsity` (rounded) of the VISIBLE key blocks is dropped uniformly at random.  With keep_last the last visible block
    (it holds the end of the own chunk) is always kept, so no row is left without a key."""
    rng = np.random.default_rng(seed + 31)
    masks: List[Optional[np.ndarray]] = []
    for s in w.streams:
        if s.q_len == 0:
            masks.append(None)
            continue
        n_qb = -(-s.q_len // block_q)
        n_kb = -(-(s.base + getattr(s, "gap_slots", 0) + s.cache_len + s.q_len) // block_k)
        vis = visible_key_blocks(s, block_k)
        m = np.zeros((w.n_heads, n_qb, n_kb), dtype=bool)
        n_drop = int(round(sparsity * vis.size))
        if keep_last:
            n_drop = min(n_drop, vis.size - 1)
        for h in range(w.n_heads):
            for qb in range(n_qb):
                cand = vis[:-1] if keep_last else vis
                drop = rng.choice(cand, size=min(n_drop, cand.size), replace=False) if n_drop > 0 else np.array([], dtype=np.int64)
                m[h, qb, vis] = True
                m[h, qb, drop] = False
        masks.append(m)
    return masks


def pack_block_masks(w: Workload, masks: Sequence[Optional[np.ndarray]], block_q: int = MASK_BLOCK_Q,
                     block_k: int = MASK_BLOCK_K) -> np.ndarray:
    """The mask in the layout include/slack.h asks for: uint32 [sum_s ceil(Lq_s/block_q)][H][words], bit (kb % 32) of
    word kb // 32 = key block kb; rows of a stream follow each other in stream order; a None mask packs as all ones."""
    n_kb_max = max([-(-(s.base + getattr(s, "gap_slots", 0) + s.cache_len + s.q_len) // block_k) for s in w.streams] + [1])
    words = -(-n_kb_max // 32)
    rows = []
    for s, m in zip(w.streams, masks):
        n_qb = -(-s.q_len // block_q)
        if n_qb == 0:
            continue
        bits = np.ones((n_qb, w.n_heads, words * 32), dtype=bool)
        if m is not None:
            bits[:] = False
            bits[:, :, :m.shape[2]] = np.transpose(m[:, :n_qb, :], (1, 0, 2))
        packed = np.packbits(bits.reshape(n_qb, w.n_heads, words, 32), axis=-1, bitorder="little")
        rows.append(packed.reshape(n_qb, w.n_heads, words, 4).view("<u4")[..., 0])
    if not rows:
        return np.zeros((0, w.n_heads, words), dtype=np.uint32)
    return np.ascontiguousarray(np.concatenate(rows, axis=0), dtype=np.uint32)
