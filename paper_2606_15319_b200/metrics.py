"""Measurement bookkeeping (flop / byte counts) for bench.py and the tests; SURVEY.md §8(d).

Not part of the data path: nothing here touches K/V/Q values.
"""
from __future__ import annotations

from typing import List


def visible_keys(streams) -> List[int]:
    """Lk per stream: keys in [lo, n) plus the sink prefix, lo = max(0, n - Wt) when Wt > 0."""
    from .workloads import visible_positions   # the one bookkeeping copy of the window formula outside oracle/ and csrc/
    return [int(visible_positions(s).size) for s in streams]


def attention_flops(streams, n_heads: int, head_dim: int) -> float:
    """4*H*D*sum_s Lq_s*Lk_s: QK^T and PV over VISIBLE keys only; padding/masked columns and the
    combine pass count zero."""
    return 4.0 * n_heads * head_dim * sum(s.q_len * lk for s, lk in zip(streams, visible_keys(streams)))


def append_bytes(streams, n_heads: int, head_dim: int, elem_bytes: int) -> float:
    """Bytes moved by one append call: read + write of K_new and V_new."""
    return 2.0 * 2.0 * sum(s.q_len for s in streams) * n_heads * head_dim * elem_bytes


def attention_min_bytes(streams, n_heads: int, head_dim: int, elem_bytes: int) -> float:
    """Minimal HBM traffic of one attention call: Q read + Out written + K and V read once."""
    vk = visible_keys(streams)
    return float(sum((2 * s.q_len + 2 * lk) * n_heads * head_dim * elem_bytes for s, lk in zip(streams, vk)))
