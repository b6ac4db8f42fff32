"""Test-side helpers: build the ORACLE's pool image for a workload (uses only oracle/ + numpy)."""
import copy

import numpy as np

import oracle


def empty_pools(w, fill=0):
    shape = (w.n_pages, w.n_heads, w.page_size, w.head_dim)
    k = np.full(shape, fill, dtype=w.storage)
    return k, k.copy()


def prior_streams(streams):
    """Descriptors that append each stream's prior tokens [0, Lc) as if they were one chunk (streams without a hole)."""
    out = []
    for s in streams:
        assert getattr(s, "gap_slots", 0) == 0, "use prior_batches() for streams with gap_slots"
        p = copy.copy(s)
        p.q_len, p.cache_len = s.cache_len, 0
        out.append(p)
    return out


def prior_batches(w):
    """[(descriptors, k, v)] append batches that write every stream's prior tokens [0, Lc).  An append writes one
    contiguous run of positions, so a stream with a hole behind its sink (gap_slots) takes two: its sink tokens first
    (no hole yet), then the held tokens behind the hole."""
    first, second = [], []
    k1, v1, k2, v2 = [], [], [], []
    for s, kp, vp in zip(w.streams, w.k_prior, w.v_prior):
        a = copy.copy(s)
        b = copy.copy(s)
        if getattr(s, "gap_slots", 0) > 0:
            a.q_len, a.cache_len, a.gap_slots = s.sink_len, 0, 0
            b.q_len, b.cache_len = s.cache_len - s.sink_len, s.sink_len
            k1.append(kp[:s.sink_len]); v1.append(vp[:s.sink_len])
            k2.append(kp[s.sink_len:]); v2.append(vp[s.sink_len:])
        else:
            a.q_len, a.cache_len = s.cache_len, 0
            b.q_len = 0
            k1.append(kp); v1.append(vp)
            k2.append(kp[:0]); v2.append(vp[:0])
        first.append(a)
        second.append(b)
    out = []
    for descs, ks, vs in ((first, k1, v1), (second, k2, v2)):
        if any(d.q_len for d in descs):
            out.append((descs, np.concatenate(ks), np.concatenate(vs)))
    return out


def oracle_pools(w, fill=0, with_new=True):
    """Pool image after appending the prior chunks (and, if with_new, the new chunk) with the oracle."""
    k, v = empty_pools(w, fill)
    for descs, kk, vv in prior_batches(w):
        oracle.kv_append(k, v, descs, kk, vv)
    if with_new:
        oracle.kv_append(k, v, w.streams, w.k_new, w.v_new)
    return k, v


def stream_rows(w):
    """[(row0, row1)] of each stream inside the ragged concat."""
    out, r = [], 0
    for s in w.streams:
        out.append((r, r + s.q_len))
        r += s.q_len
    return out


def oracle_pools_fp8(w, code_fill=0x7F, scale_fill=np.nan, with_new=True):
    """FP8 pool image (codes uint8 [n_pages, H, P, D] + fp32 scales [n_pages, H, P // 128], K and V) after the oracle's
    quantising append of the prior chunks (and, if with_new, the new chunk).  Unwritten slots keep `code_fill` (0x7f =
    NaN) and untouched scales `scale_fill`."""
    F = oracle.fp8_attention
    shape = (w.n_pages, w.n_heads, w.page_size, w.head_dim)
    kc = np.full(shape, code_fill, dtype=np.uint8)
    vc = kc.copy()
    ks = np.full((w.n_pages, w.n_heads, w.page_size // F.KEY_BLOCK), scale_fill, dtype=np.float32)
    vs = ks.copy()
    for descs, kk, vv in prior_batches(w):
        F.kv_append_fp8(kc, vc, ks, vs, descs, kk, vv, w.dtype)
    if with_new:
        F.kv_append_fp8(kc, vc, ks, vs, w.streams, w.k_new, w.v_new, w.dtype)
    return kc, vc, ks, vs
