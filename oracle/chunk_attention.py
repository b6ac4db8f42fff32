"""ORACLE — test infrastructure, not product code.

Plain, slow, fp64 CPU statement of what the hot path computes: paged KV append (exact copy) and
ragged chunk attention over per-stream paged KV caches.  Only `tests/`, `__graft_entry__.smoke()`
and `bench.py`'s cpu_baseline / `--impl reference` leg may import this package; it shares no code
with `paper_2606_15319_b200/csrc` (the CUDA path) or its Python binding and imports neither.

What it follows
---------------
* A chunk's tokens attend to the cached K/V of the stream's earlier chunks, and the finished chunk
  is appended to the rolling KV cache: PAPER.md P:21 (§1), P:84 (§2.1 "AR-DiT").
* Bounded cache: "preserves the first few chunks as a global sink and keeps KV entries only for the
  most recent W chunks": P:86 (§2.1), knob (3) P:88, W in {1,3,7} chunks P:568 (App. A).
* Paged KV pool with a logical->physical page table per worker: P:152 (§3.2), P:251 (§4.4).
* Everything the paper leaves open (mask inside the chunk, window counting the own chunk, pool
  layout, scale, append-then-attend) is taken from BASELINE.json north_star/configs as read in
  SURVEY.md §8(c) A1-A16 and listed in DESIGN.md "Readings".

Definition; for stream s, head h, with n = Lc + Lq:
    lo      = max(0, n - Wt) if Wt > 0 else 0
    visible = [0, sink) U [max(sink, lo), n)             (sink = min(sink_len, n); 0 in all configs)
    s_t     = scale * <q_i, k_t>      for t in visible   (every query row sees every visible key:
                                                          bidirectional inside the own chunk, A1)
    out_i   = sum_t softmax_t(s)_t * v_t ,   lse_i = ln sum_t exp(s_t)
Held token t of a stream sits at POSITION pos(t) = base + t, plus gap_slots when t >= sink_len (the hole
left behind the sink by tokens that were dropped from a bounded "sink + local" cache), i.e. at
physical page page_table[pos // P], slot pos % P of a pool laid out [n_pages][H][P][D] (the
token->slot rule of include/slack.h).  cache_len counts held tokens only.

Block-sparse variant (PAPER.md P:88 knob (2) "skips nonselected attention blocks
with sparse masks ... controlled by attention sparsity rho", rho in {0,.6,.7,.8,.9} P:568, selection
rule from Light Forcing [39] P:319 - the rule is NOT in the paper, so the mask is an INPUT here):
    query block  qb = i // block_q            (i = chunk-local query row)
    key block    kb = pos(t) // block_k       (position of key token t in the stream's page-table space)
    t is used iff it is visible (above) AND mask[h, qb, kb]
    out_i = softmax over the used keys; a row with no used key has out_i = 0 and lse_i = -inf.

State-plane page transfer ("transfer(stream, src, dst, page_range)"
layer-major asynchronous streaming, "migrates only the KV pages corresponding to the head partition"):
an exact copy, for every layer, of the head slices [h0, h1) of the listed source pages into the listed destination
pages of another pool; nothing else in the destination changes (`kv_transfer`).

Since attention is a *defined* function the oracle is that definition written out: gather, one
matmul, a max-subtracted exp, one matmul, a division - in fp64, no tiling over keys, no online
softmax, no splits.  Query rows are processed in blocks of <= `row_block` rows only to bound
memory (rows are independent, so this changes no row's arithmetic).

Pins (tests/test_oracle_pins.py): pure-Python brute force, closed forms (V=1, K=0 mean, single key,
one-hot V, logit shift), torch SDPA fp64, dense block-causal masked attention over the whole
sequence, page permutation invariance, NaN poisoning of unowned slots, scipy logsumexp, LSE merge.
Block-sparse pins (tests/test_oracle_sparse_pins.py): all-ones mask == dense, pure-Python brute force
with tiny blocks, torch SDPA fp64 with an element-wise boolean mask, K=0 closed form (mean of V over the
used keys, base/window swept), disjoint-mask LSE merge == union mask, bits of invisible blocks ignored,
empty rows.
The paper prints no numeric example for this path, so no paper-valued fixture exists.
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import numpy as np


# ----------------------------------------------------------------------------------------------
# storage decoding (exact)
# ----------------------------------------------------------------------------------------------

def to_f64(x: np.ndarray, dtype: str) -> np.ndarray:
    """Exact conversion of stored values to fp64. dtype 'bf16': uint16 bit patterns; 'f32': float32."""
    if dtype == "bf16":
        assert x.dtype == np.uint16
        return (x.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)
    if dtype == "f32":
        assert x.dtype == np.float32
        return x.astype(np.float64)
    if dtype == "f64":          # already-widened operands (oracle/fp8_attention.py hands dequantised values in)
        assert x.dtype == np.float64
        return x
    raise ValueError(dtype)


# ----------------------------------------------------------------------------------------------
# token -> slot rule and visible range
# ----------------------------------------------------------------------------------------------

def token_positions(stream, tokens: np.ndarray) -> np.ndarray:
    """pos(t) = base + t for the sink tokens t < sink_len, base + gap_slots + t behind them (include/slack.h)."""
    t = np.asarray(tokens, dtype=np.int64)
    gap = getattr(stream, "gap_slots", 0)
    return stream.base + t + np.where(t >= getattr(stream, "sink_len", 0), gap, 0)


def token_slots(stream, tokens: np.ndarray, page_size: int) -> Tuple[np.ndarray, np.ndarray]:
    """(physical page, slot) of held tokens of one stream: page_table[pos // P], pos % P."""
    pos = token_positions(stream, tokens)
    table = np.asarray(stream.page_table, dtype=np.int64)
    return table[pos // page_size], pos % page_size


def visible_tokens(stream) -> np.ndarray:
    """Logical key positions a stream's new chunk attends to, ascending (A2, A9)."""
    n = stream.cache_len + stream.q_len
    lo = max(0, n - stream.window) if stream.window > 0 else 0
    sink = min(getattr(stream, "sink_len", 0), n)
    lo = max(lo, sink)
    return np.concatenate([np.arange(0, sink, dtype=np.int64), np.arange(lo, n, dtype=np.int64)])


# ----------------------------------------------------------------------------------------------
# A1: KV append (exact copy)
# ----------------------------------------------------------------------------------------------

def kv_append(k_pool: np.ndarray, v_pool: np.ndarray, streams: Sequence, k_new: np.ndarray,
              v_new: np.ndarray) -> None:
    """Write logical tokens [Lc, Lc+Lq) of every stream into the pool image, in place.

    k_pool/v_pool: [n_pages, H, P, D] storage dtype; k_new/v_new: ragged concat [sum Lq, H, D] in
    stream order.  Pure copy: no byte outside the named slots changes.
    """
    page_size = k_pool.shape[2]
    row = 0
    for s in streams:
        if s.q_len:
            page, slot = token_slots(s, np.arange(s.cache_len, s.cache_len + s.q_len), page_size)
            k_pool[page, :, slot, :] = k_new[row:row + s.q_len]     # token i -> (page[i], all heads, slot[i])
            v_pool[page, :, slot, :] = v_new[row:row + s.q_len]
        row += s.q_len


def gather_kv(pool: np.ndarray, stream, tokens: np.ndarray) -> np.ndarray:
    """Rows of one pool for the given logical tokens of one stream -> [len(tokens), H, D] (storage dtype)."""
    page, slot = token_slots(stream, tokens, pool.shape[2])
    return pool[page, :, slot, :]


# ----------------------------------------------------------------------------------------------
# NEXT-4: state-plane page transfer (exact copy)
# ----------------------------------------------------------------------------------------------

def kv_transfer(src_k: np.ndarray, src_v: np.ndarray, dst_k: np.ndarray, dst_v: np.ndarray,
                src_pages: Sequence[int], dst_pages: Sequence[int], head_begin: int, head_end: int) -> None:
    """One layer of transfer(stream, src, dst, page_range): page src_pages[i] of the source pool image becomes page
    dst_pages[i] of the destination pool image, heads [head_begin, head_end) only (the head partition of P:660-662);
    in place on dst_*; pools are [n_pages, H, P, D] of the same H, P, D and storage dtype."""
    assert len(src_pages) == len(dst_pages)
    for sp, dp in zip(src_pages, dst_pages):
        dst_k[dp, head_begin:head_end] = src_k[sp, head_begin:head_end]
        dst_v[dp, head_begin:head_end] = src_v[sp, head_begin:head_end]


# ----------------------------------------------------------------------------------------------
# A3: chunk attention (definition)
# ----------------------------------------------------------------------------------------------

def attend_rows(q_rows: np.ndarray, k: np.ndarray, v: np.ndarray, scale: float):
    """softmax(scale * q k^T) v for fp64 q_rows [R, D], k/v [Lk, D]. Returns (out [R, D], lse [R])."""
    s = scale * (q_rows @ k.T)
    m = s.max(axis=1, keepdims=True)
    p = np.exp(s - m)
    l = p.sum(axis=1, keepdims=True)
    out = (p @ v) / l
    lse = (m + np.log(l))[:, 0]
    return out, lse


def _sparse_stream(k_pool, v_pool, s, toks, sel, q, row0, scale, dtype, mask, block_q, block_k, out, lse) -> None:
    """Block-sparse rows of one stream: for every head and query block, softmax over the visible keys whose
    key block is selected (header; P:88 knob (2)).  Rows of one query block share their key set."""
    n_heads = q.shape[1]
    key_block = token_positions(s, toks) // block_k        # key block of every visible token
    assert mask.shape[0] == n_heads and mask.shape[1] >= -(-s.q_len // block_q) and mask.shape[2] > int(key_block.max())
    for h in range(n_heads):
        for qb in np.unique(sel // block_q):
            r = sel[sel // block_q == qb]
            used = toks[mask[h, qb, key_block]]            # visible AND selected
            if used.size == 0:
                out[row0 + r, h, :] = 0.0
                lse[h, row0 + r] = -np.inf
                continue
            kh = to_f64(np.ascontiguousarray(gather_kv(k_pool, s, used)[:, h, :]), dtype)
            vh = to_f64(np.ascontiguousarray(gather_kv(v_pool, s, used)[:, h, :]), dtype)
            qh = to_f64(np.ascontiguousarray(q[row0 + r, h, :]), dtype)
            o, l = attend_rows(qh, kh, vh, scale)
            out[row0 + r, h, :] = o
            lse[h, row0 + r] = l


def chunk_attention(k_pool: np.ndarray, v_pool: np.ndarray, streams: Sequence, q: np.ndarray,
                    scale: float, dtype: str, row_block: int = 512,
                    rows: Optional[Sequence[Optional[np.ndarray]]] = None,
                    block_masks: Optional[Sequence[Optional[np.ndarray]]] = None,
                    block_q: int = 256, block_k: int = 128):
    """Ragged chunk attention for a batch of streams; precondition: own chunk already appended.

    q: [sum Lq, H, D] storage dtype.  Returns (out fp64 [sum Lq, H, D], lse fp64 [H, sum Lq]).
    `rows`: optional per-stream arrays of chunk-local query rows to compute (others stay NaN) - rows
    are independent, so a sampled row is exact (used at full size).
    `block_masks`: optional per-stream boolean arrays [H, ceil(Lq/block_q), >= ceil((base+n)/block_k)]
    (None = dense for that stream): the block-sparse variant of the header (P:88 knob (2)).
    """
    total_q, n_heads, head_dim = q.shape
    out = np.full((total_q, n_heads, head_dim), np.nan, dtype=np.float64)
    lse = np.full((n_heads, total_q), np.nan, dtype=np.float64)
    row0 = 0
    for si, s in enumerate(streams):
        if s.q_len == 0:
            continue
        toks = visible_tokens(s)
        sel = np.arange(s.q_len) if rows is None or rows[si] is None else np.asarray(rows[si], dtype=np.int64)
        if sel.size and block_masks is not None and block_masks[si] is not None:
            _sparse_stream(k_pool, v_pool, s, toks, sel, q, row0, scale, dtype, np.asarray(block_masks[si], dtype=bool),
                           block_q, block_k, out, lse)
        elif sel.size:
            k_all = gather_kv(k_pool, s, toks)          # [Lk, H, D] storage
            v_all = gather_kv(v_pool, s, toks)
            for h in range(n_heads):
                kh = to_f64(np.ascontiguousarray(k_all[:, h, :]), dtype)
                vh = to_f64(np.ascontiguousarray(v_all[:, h, :]), dtype)
                for b in range(0, sel.size, row_block):
                    r = sel[b:b + row_block]
                    qh = to_f64(np.ascontiguousarray(q[row0 + r, h, :]), dtype)
                    o, l = attend_rows(qh, kh, vh, scale)
                    out[row0 + r, h, :] = o
                    lse[h, row0 + r] = l
        row0 += s.q_len
    return out, lse


# ----------------------------------------------------------------------------------------------
# A4: split-KV combine formula (stated here only so its pin can live in the oracle's test-suite)
# ----------------------------------------------------------------------------------------------

def lse_merge(outs: List[np.ndarray], lses: List[np.ndarray]):
    """Merge per-part normalised outputs O_p [R, D] and lse_p [R] over disjoint key sets:
    m = max_p lse_p ; out = sum_p e^{lse_p-m} O_p / sum_p e^{lse_p-m} ; lse = m + ln sum_p e^{lse_p-m}."""
    L = np.stack(lses, axis=0)
    m = L.max(axis=0)
    w = np.exp(L - m)
    den = w.sum(axis=0)
    out = sum(w[p][:, None] * outs[p] for p in range(len(outs))) / den[:, None]
    return out, m + np.log(den)


# ----------------------------------------------------------------------------------------------
# error metrics
# ----------------------------------------------------------------------------------------------

def error_metrics(got: np.ndarray, want: np.ndarray):
    """max-abs and relative Frobenius error of `got` (any float dtype, widened exactly) vs fp64 `want`,
    over the entries where `want` is not NaN (row-sampled oracles leave the rest NaN)."""
    g = np.asarray(got, dtype=np.float64)
    mask = ~np.isnan(want)
    d = g[mask] - want[mask]
    if d.size == 0:
        return 0.0, 0.0
    if not np.all(np.isfinite(g[mask])):
        return float("inf"), float("inf")
    den = float(np.sqrt(np.sum(want[mask] ** 2)))
    return float(np.max(np.abs(d))), float(np.sqrt(np.sum(d * d)) / den) if den > 0 else float(np.sqrt(np.sum(d * d)))
