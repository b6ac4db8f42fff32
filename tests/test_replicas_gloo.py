"""N > 1 path of bench.py on CPU: world_size-2 `gloo` ranks.  The path does not shard (replicas
only, no data-path collective): each rank plans its OWN seeded batch of the same shape; torch.distributed provides the
barrier and the max over ranks of the per-rank device time; the whole-job value is the sum of the ranks' work over
that time.  This test runs exactly that host logic (descriptors, plan, reduction) with a host-only context."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, out_q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import argparse
    import bench
    from paper_2606_15319_b200 import binding, metrics
    args = argparse.Namespace(workload="cfg3", kv_chunks=7)
    w = bench.make_descriptors(args, seed_shift=rank)            # replicas: own batch per rank
    ctx = binding.Context(-1)                                     # host-only: planning needs no GPU
    pool = binding.Pool.shape_only(w.n_pages, w.n_heads, w.head_dim, w.page_size, w.dtype)
    plan = ctx.slack_plan(pool, w.streams, sm_count=148)
    flops = metrics.attention_flops(w.streams, w.n_heads, w.head_dim)
    fake_ms = 10.0 + 5.0 * rank                                   # stands in for the rank's CUDA-event time
    dist.barrier()
    t, f = bench.reduce_job(dist, fake_ms, flops)               # the very reduction bench.py's `value` is built from
    out_q.put((rank, plan.num_items, [s.cache_len for s in w.streams], flops, t, f))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_two_replicas_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_rank_main, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=150) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, items0, lc0, fl0, t0, f0), (r1, items1, lc1, fl1, t1, f1) = res
    assert (r0, r1) == (0, 1)
    assert lc0 != lc1, "each replica draws its own ragged batch (seed shifted by rank)"
    assert items0 > 0 and items1 > 0
    assert t0 == t1 == 15.0, "device time is the max over ranks"
    assert np.isclose(f0, fl0 + fl1) and f0 == f1, "whole-job work is the sum over replicas"
