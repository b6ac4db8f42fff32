"""Pins for the oracle's state-plane page transfer (PAPER.md P:255 transfer(stream, src, dst,
page_range), P:660-662 head-partition-aware transfer).  A transfer is an exact copy, so the pins are the properties that
fix it: every named (page, head) slice arrives bit for bit, no other byte of the destination changes, complementary
head partitions compose to the full transfer, there-and-back is the identity, and a migrated stream attends identically
through its new page table (attention is invariant to where pages live: the same invariance that pins the gather)."""
import copy

import numpy as np
import pytest

import oracle
from paper_2606_15319_b200 import workloads as W
from helpers import oracle_pools


def migrate_setup(seed=3, dtype="bf16"):
    w = W.small_ragged(seed=seed, dtype=dtype, head_dim=16, n_heads=4)
    src_k, src_v = oracle_pools(w)
    rng = np.random.default_rng(seed)
    n_dst = w.n_pages + 5
    sent = np.uint16(0x7FC1) if dtype == "bf16" else np.float32(np.nan)
    dst_k = np.full((n_dst,) + src_k.shape[1:], sent, dtype=src_k.dtype)
    dst_v = dst_k.copy()
    s = w.streams[0]
    src_pages = np.asarray(s.page_table, dtype=np.int64)
    dst_pages = rng.permutation(n_dst)[:src_pages.size]
    return w, (src_k, src_v), (dst_k, dst_v), src_pages, dst_pages


@pytest.mark.parametrize("dtype", ["bf16", "f32"])
def test_named_slices_arrive_and_nothing_else_changes(dtype):
    w, (sk, sv), (dk, dv), sp, dp = migrate_setup(dtype=dtype)
    before_k, before_v = dk.copy(), dv.copy()
    oracle.kv_transfer(sk, sv, dk, dv, sp, dp, 1, 3)
    bits = (lambda a: a.view(np.uint32)) if dtype == "f32" else (lambda a: a)
    for a, b in zip(sp, dp):                               # written out independently of the routine's slicing
        for h in (1, 2):
            assert np.array_equal(bits(dk[b, h]), bits(sk[a, h])) and np.array_equal(bits(dv[b, h]), bits(sv[a, h]))
    touched = np.zeros(dk.shape[:2], dtype=bool)
    touched[np.asarray(dp)[:, None], np.array([1, 2])[None, :]] = True
    assert np.array_equal(bits(dk[~touched]), bits(before_k[~touched]))
    assert np.array_equal(bits(dv[~touched]), bits(before_v[~touched]))


def test_head_partitions_compose_and_round_trip_is_identity():
    w, (sk, sv), (dk, dv), sp, dp = migrate_setup()
    full_k, full_v = dk.copy(), dv.copy()
    oracle.kv_transfer(sk, sv, full_k, full_v, sp, dp, 0, w.n_heads)
    oracle.kv_transfer(sk, sv, dk, dv, sp, dp, 0, 2)       # SP2-style halves (heads partitioned across workers)
    oracle.kv_transfer(sk, sv, dk, dv, sp, dp, 2, w.n_heads)
    assert np.array_equal(dk, full_k) and np.array_equal(dv, full_v)
    back_k, back_v = np.zeros_like(sk), np.zeros_like(sv)
    oracle.kv_transfer(dk, dv, back_k, back_v, dp, sp, 0, w.n_heads)
    assert np.array_equal(back_k[sp], sk[sp]) and np.array_equal(back_v[sp], sv[sp])


def test_migrated_stream_attends_identically():
    w, (sk, sv), (dk, dv), sp, dp = migrate_setup()
    oracle.kv_transfer(sk, sv, dk, dv, sp, dp, 0, w.n_heads)
    s0 = w.streams[0]
    want, want_lse = oracle.chunk_attention(sk, sv, [s0], w.q[:s0.q_len], w.scale, w.dtype)
    moved = copy.copy(s0)
    moved.page_table = np.asarray(dp, dtype=np.int32)
    got, got_lse = oracle.chunk_attention(dk, dv, [moved], w.q[:s0.q_len], w.scale, w.dtype)
    assert np.array_equal(got, want) and np.array_equal(got_lse, want_lse)
