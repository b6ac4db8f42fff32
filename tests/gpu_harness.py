"""GPU-side test harness: runs a Workload through the C ABI (via the binding) and compares with the oracle.

Used by the -m gpu tests and by __graft_entry__.smoke().  The GPU path never sees oracle data: both sides start
from the same seeded Workload arrays (paper_2606_15319_b200.workloads).
"""
from __future__ import annotations

import os

import numpy as np
import torch

import oracle
from paper_2606_15319_b200 import binding
from helpers import oracle_pools, prior_batches

# kernel kind the tensor-core cases report: 0, or 2 when SLACK_TEST_CTA_PAIRS=2 reruns the suites on CTA pairs
TC_KIND = 2 if os.environ.get("SLACK_TEST_CTA_PAIRS", "0") == "2" else 0

SENTINEL_BF16 = 0x7FC1   # a NaN bit pattern: any leak of an unowned / masked slot into the output shows up as NaN
SENTINEL_F32 = np.float32(np.nan)


def device_pools(w, device="cuda:0", sentinel=True):
    shape = (w.n_pages, w.n_heads, w.page_size, w.head_dim)
    if w.dtype == "bf16":
        fill = SENTINEL_BF16 if sentinel else 0
        k = torch.full(shape, fill, dtype=torch.int32, device=device).to(torch.int16).view(torch.bfloat16) if False else \
            torch.from_numpy(np.full(shape, fill, dtype=np.uint16).view(np.int16)).to(device).view(torch.bfloat16)
    else:
        k = torch.full(shape, float("nan") if sentinel else 0.0, dtype=torch.float32, device=device)
    return k, k.clone()


def host_fill(w, sentinel=True):
    if w.dtype == "bf16":
        return SENTINEL_BF16 if sentinel else 0
    return SENTINEL_F32 if sentinel else np.float32(0)


def gpu_append_all(ctx, w, pool, device="cuda:0", planned_plan=None):
    """Appends the prior chunks, then the new chunk, through slack_kv_append (or the planned variant for the new chunk)."""
    for descs, kk, vv in prior_batches(w):
        ctx.slack_kv_append(pool, descs, binding.to_torch(kk, w.dtype, device), binding.to_torch(vv, w.dtype, device))
    kn = binding.to_torch(w.k_new, w.dtype, device)
    vn = binding.to_torch(w.v_new, w.dtype, device)
    if planned_plan is not None:
        ctx.slack_kv_append_planned(planned_plan, pool, kn, vn)
    else:
        ctx.slack_kv_append(pool, w.streams, kn, vn)
    torch.cuda.synchronize()


def make_pool(w, device="cuda:0", sentinel=True):
    k, v = device_pools(w, device, sentinel)
    return binding.Pool(k, v, w.n_pages, w.n_heads, w.head_dim, w.page_size, w.dtype)


def gpu_attention(ctx, w, pool, device="cuda:0", want_lse=True, **plan_opts):
    # SLACK_TEST_CTA_PAIRS=1|2 reruns every case that does not choose itself on one CTA per item / on CTA pairs
    plan_opts.setdefault("cta_pairs", int(os.environ.get("SLACK_TEST_CTA_PAIRS", "0")))
    plan = ctx.slack_plan(pool, w.streams, **plan_opts)
    q = binding.to_torch(w.q, w.dtype, device)
    out = torch.full_like(q, float("nan"))
    lse = torch.full((w.n_heads, max(w.total_q, 1)), float("nan"), dtype=torch.float32, device=device) if want_lse else None
    ws = torch.empty(max(plan.workspace_bytes, 16), dtype=torch.uint8, device=device)
    ctx.slack_chunk_attention(plan, pool, q, out, w.scale, lse=lse, workspace=ws)
    torch.cuda.synchronize()
    launches = ctx.last_launch_count
    out_np = out.float().cpu().numpy().astype(np.float64)
    lse_np = lse.cpu().numpy().astype(np.float64)[:, :w.total_q] if want_lse else None
    return out_np, lse_np, plan, launches


def pools_equal_oracle(w, pool):
    """Whole-pool bit compare of the device pools with the oracle's pool image (same sentinel fill)."""
    ko, vo = oracle_pools(w, fill=host_fill(w))
    kg = binding.to_numpy(pool.k_pool, w.dtype)
    vg = binding.to_numpy(pool.v_pool, w.dtype)
    if w.dtype == "bf16":
        return bool(np.array_equal(kg, ko) and np.array_equal(vg, vo))
    return bool(np.array_equal(kg.view(np.uint32), ko.view(np.uint32)) and np.array_equal(vg.view(np.uint32), vo.view(np.uint32)))


def oracle_attention(w, rows=None):
    ko, vo = oracle_pools(w, fill=host_fill(w))
    return oracle.chunk_attention(ko, vo, w.streams, w.q, w.scale, w.dtype, rows=rows)


def check_attention(w, out_np, lse_np, want, want_lse, max_abs_tol=2e-2, rel_fro_tol=1e-2, lse_tol=2e-2, per_stream=True):
    """Returns a dict of error figures; raises AssertionError beyond tolerance (BASELINE.json north_star: max-abs <= 2e-2
    and relative Frobenius <= 1e-2, applied to the whole output and per stream)."""
    res = {}
    ma, rf = oracle.error_metrics(out_np, want)
    res["max_abs"], res["rel_fro"] = ma, rf
    assert ma <= max_abs_tol and rf <= rel_fro_tol, f"{w.name}: max_abs {ma:.3e} rel_fro {rf:.3e}"
    if per_stream:
        r = 0
        for si, s in enumerate(w.streams):
            if s.q_len:
                ma_s, rf_s = oracle.error_metrics(out_np[r:r + s.q_len], want[r:r + s.q_len])
                assert ma_s <= max_abs_tol and rf_s <= rel_fro_tol, f"{w.name} stream {si}: max_abs {ma_s:.3e} rel_fro {rf_s:.3e}"
            r += s.q_len
    if lse_np is not None and want_lse is not None:
        mask = ~np.isnan(want_lse)
        if mask.any():
            le = float(np.max(np.abs(lse_np[mask] - want_lse[mask])))
            res["lse_max_abs"] = le
            assert le <= lse_tol, f"{w.name}: lse max_abs {le:.3e}"
    return res


# ---------------------------------------------------------------------------------------------------- FP8 pools (NEXT-3)
def make_pool_fp8(w, device="cuda:0", code_fill=0x7F, scale_fill=float("nan")):
    """e4m3 code pools filled with the NaN code and scales filled with NaN: whatever the append does not write stays put."""
    shape = (w.n_pages, w.n_heads, w.page_size, w.head_dim)
    k = torch.full(shape, code_fill, dtype=torch.uint8, device=device)
    ks = torch.full((w.n_pages, w.n_heads, w.page_size // 128), scale_fill, dtype=torch.float32, device=device)
    return binding.Pool(k, k.clone(), w.n_pages, w.n_heads, w.head_dim, w.page_size, "fp8", k_scale=ks, v_scale=ks.clone())


def fp8_pool_images(pool):
    return (pool.k_pool.cpu().numpy(), pool.v_pool.cpu().numpy(), pool.k_scale.cpu().numpy(), pool.v_scale.cpu().numpy())
