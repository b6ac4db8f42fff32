"""Test-side helpers: build the ORACLE's pool image for a workload (uses only oracle/ + numpy)."""
import copy

import numpy as np

import oracle


def empty_pools(w, fill=0):
    shape = (w.n_pages, w.n_heads, w.page_size, w.head_dim)
    k = np.full(shape, fill, dtype=w.storage)
    return k, k.copy()


def prior_streams(streams):
    """Descriptors that append each stream's prior tokens [0, Lc) as if they were one chunk."""
    out = []
    for s in streams:
        p = copy.copy(s)
        p.q_len, p.cache_len = s.cache_len, 0
        out.append(p)
    return out


def oracle_pools(w, fill=0, with_new=True):
    """Pool image after appending the prior chunks (and, if with_new, the new chunk) with the oracle."""
    k, v = empty_pools(w, fill)
    if any(s.cache_len for s in w.streams):
        oracle.kv_append(k, v, prior_streams(w.streams), np.concatenate(w.k_prior), np.concatenate(w.v_prior))
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
