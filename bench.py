"""bench.py — one JSON line: chunk-attention TFLOP/s of the hot path on B200 (BASELINE.json metric).

A STEP is one denoising step of one chunk batch, i.e. one pass of the whole hot path:
    slack_plan (host, once per step)  ->  for each of the 30 layers:  slack_kv_append  ->  slack_chunk_attention
                                                                       (attention kernel + split-KV combine)
Every layer has its own pools and its own seeded Q / K_new / V_new, so each launch reads K/V that is not in L2
(cfg2: 201 MB of pools per layer, 6 GB per step >> 126 MB L2) — no explicit L2 flush is needed.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg3|cfg4|cfg5|cfg5b] [--impl reference]
                    [--sparsity RHO]   block-sparse variant (P:88 knob (2), rho in {.6,.7,.8,.9} P:568): every layer gets
                                       its own seeded block mask; flops count the SELECTED (query, key) pairs only
                    [--no-others]      skip the short supplementary blocks (config.others)

The headline workload is BASELINE.json configs[4] at the full 21-frame window (4 streams, Lk = 32760): the long-cache
configuration `north_star` states its target on and the largest one of the roofline sweep that fits one GPU (24 GB of
pools for 30 layers).  configs[1]-[3] and the decode-like case are parity-test cases; at N = 1 short blocks of configs[3]
(mixed streams: chunks/s), configs[2] (the 460 MB append) and the decode-like case (HBM GB/s) are added under
`config.others`, never as the headline.

value   = attention FLOPs (4*H*D*sum Lq*Lk, visible keys only) of all ranks / device time of the K steps (max over ranks)
e2e     = the same with Q/K_new/V_new copied from pinned host memory and Out copied back inside the timed region
roofline= the attention kernel alone (CUDA events recorded by the library around that kernel on its stream);
          frac = achieved / MEASURED_PEAKS.json bf16_tflops (the burst figure: SURVEY.md A11's headline denominator), the
          sustained and the nominal fractions beside it
append / combine = the same library event pairs around the KV append and the split-KV combine kernels
cpu_baseline = the fp64 oracle, as it stands, on a bounded row sample of layer 0 on the host cores.
Multi-GPU: the path has no exchange step -> replicas only: each rank runs its own batch (weak scaling), no collective
on the data path; torch.distributed is used for the barrier and the max over ranks of the device time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "chunk_attention_tflops"
UNIT = "TFLOP/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="cfg5", choices=["cfg2", "cfg3", "cfg4", "cfg5", "cfg5b"])
    ap.add_argument("--no-others", action="store_true", help="skip the supplementary blocks under config.others")
    ap.add_argument("--dtype", default="bf16", choices=["bf16", "fp8"],
                    help="fp8: FP8 (e4m3) K/V pools, quantising append, FP8 attention (NEXT-3; never the headline line)")
    ap.add_argument("--kv-chunks", type=int, default=7, help="cfg5: visible chunks (1..7)")
    ap.add_argument("--layers", type=int, default=30)
    ap.add_argument("--force-splits", type=int, default=0)
    ap.add_argument("--cta-pairs", type=int, default=0, choices=[0, 1, 2],
                    help="slack_plan_opts.cta_pairs: 0 = automatic, 1 = one CTA per item, 2 = CTA pairs (cta_group::2)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-rows", type=int, default=768, help="query rows of the oracle sample")
    ap.add_argument("--transfer-bench", action="store_true",
                    help="also time slack_kv_transfer (state-plane page transfer, NEXT-4) of stream 0 over all layers")
    ap.add_argument("--sparsity", type=float, default=0.0, help="block-sparse variant: fraction of visible key blocks dropped")
    return ap.parse_args()


def make_descriptors(args, seed_shift=0, workload=None):
    """The workload's stream descriptors WITHOUT drawing tensors (layers are filled on the device)."""
    import unittest.mock as m
    from paper_2606_15319_b200 import workloads as W
    name = workload or args.workload
    makers = {"cfg2": lambda: W.config2(seed=2000 + seed_shift), "cfg3": lambda: W.config3(seed=3000 + seed_shift),
              "cfg4": lambda: W.config4(seed=4000 + seed_shift),
              "cfg5": lambda: W.config5(kv_chunks=args.kv_chunks, seed=5000 + seed_shift),
              "cfg5b": lambda: W.config5b(seed=5500 + seed_shift)}
    with m.patch.object(W, "_draw", lambda rng, shape, amp, dtype: np.zeros((0,), dtype=np.uint16)):
        return makers[name]()


def reduce_job(dist, ms, flops, device=None):
    """N > 1 (replicas only): whole-job time = MAX over ranks of the device time, whole-job work = SUM over ranks of the
    flops each rank's own batch holds (ragged configs draw different batches per rank)."""
    if dist is None:
        return float(ms), float(flops)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    f = torch.tensor([flops], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(f, op=dist.ReduceOp.SUM)
    return float(t.item()), float(f.item())


def workload_label(args, w, workload=None):
    names = {"cfg2": "BASELINE.json configs[1]: 1 stream, Lq=4680, 4 prior chunks (Lk=23400), H=12, D=128, bf16, P=256",
             "cfg3": "BASELINE.json configs[2]: ragged batch of 8 streams, priors U{0..6}",
             "cfg4": "BASELINE.json configs[3]: 16 streams mixed fidelity, 21-frame window",
             "cfg5": f"BASELINE.json configs[4]: 4 streams, Lq=4680, Lk={args.kv_chunks * 4680}"
                     + (" (full 21-frame window)" if args.kv_chunks == 7 else "") + ", H=12, D=128, bf16, P=256",
             "cfg5b": "supplementary decode-like: 64 streams, Lq=72, Lk=8190"}
    return names[workload or args.workload]


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 20 ms DURING the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "20"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for n, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        os.unlink(self.f.name)
        if sm:
            # "under load" = samples drawing real power; the median over those is what the timed region saw
            load = [s for s, p in zip(sm, pw) if p >= 0.5 * max(pw)] or sm
            out.update(sm_mhz=float(np.median(load)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                       reasons=sorted(reasons), samples=len(sm))
        return out


# ---------------------------------------------------------------------------------------------------------------------
# CPU baseline: the oracle as it stands, on a bounded row sample
# ---------------------------------------------------------------------------------------------------------------------

def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        n = [d.get("num_threads", 0) for d in threadpool_info() if d.get("user_api") == "blas"]
        if n:
            return int(max(n))
    except Exception:
        pass
    return int(os.cpu_count() or 1)


def sample_rows(streams, n_rows, seed=17):
    """n_rows query rows spread over the streams in proportion to their chunk length (seeded)."""
    rng = np.random.default_rng(seed)
    total = sum(s.q_len for s in streams)
    rows = []
    for s in streams:
        k = min(s.q_len, max(1, int(round(n_rows * s.q_len / max(total, 1))))) if s.q_len else 0
        rows.append(np.sort(rng.choice(s.q_len, size=k, replace=False)) if k else np.zeros(0, dtype=np.int64))
    return rows


def sample_flops(streams, rows, n_heads, head_dim):
    from paper_2606_15319_b200 import metrics
    return 4.0 * n_heads * head_dim * sum(len(r) * lk for r, lk in zip(rows, metrics.visible_keys(streams)))


def selected_pairs(w, masks, rows=None):
    """(query, key) pairs, summed over heads, that a block mask leaves: sum over query rows of the visible keys in selected
    blocks.  `rows`: optional per-stream sampled rows (else every row)."""
    from paper_2606_15319_b200 import workloads as W
    total = 0
    for si, (s, m) in enumerate(zip(w.streams, masks)):
        if s.q_len == 0:
            continue
        n = s.cache_len + s.q_len
        lo = max(0, n - s.window) if s.window > 0 else 0
        sink = min(s.sink_len, n)
        lo = max(lo, sink)
        toks = np.concatenate([np.arange(0, sink), np.arange(lo, n)])
        keys_per_block = np.bincount((s.base + toks) // W.MASK_BLOCK_K, minlength=m.shape[2])
        per_qb = (m * keys_per_block[None, None, :]).sum(axis=(0, 2))           # [n_qb], summed over heads
        r = np.arange(s.q_len) if rows is None else np.asarray(rows[si])
        total += int(per_qb[r // W.MASK_BLOCK_Q].sum())
    return total


def time_oracle(w, k_pool, v_pool, q, n_rows, masks=None):
    """Runs oracle.chunk_attention on `n_rows` sampled rows; returns (seconds, flops, rows, out, lse)."""
    import oracle
    rows = sample_rows(w.streams, n_rows)
    t0 = time.perf_counter()
    out, lse = oracle.chunk_attention(k_pool, v_pool, w.streams, q, w.scale, w.dtype, rows=rows, block_masks=masks)
    dt = time.perf_counter() - t0
    fl = sample_flops(w.streams, rows, w.n_heads, w.head_dim) if masks is None else 4.0 * w.head_dim * selected_pairs(w, masks, rows)
    return dt, fl, rows, out, lse


def host_layer(w, seed):
    """Seeded host-side pools / Q for one layer (bf16 bit patterns), pool pages filled directly with N(0,1)*0.5."""
    from paper_2606_15319_b200 import workloads as W
    rng = np.random.default_rng(seed)
    shape = (w.n_pages, w.n_heads, w.page_size, w.head_dim)
    draw = lambda shp: W.f32_to_bf16_bits(rng.standard_normal(shp, dtype=np.float32) * np.float32(0.5))
    return draw(shape), draw(shape), draw((w.total_q, w.n_heads, w.head_dim))


def run_reference(args):
    """--impl reference: the oracle (kind "oracle") on the host cores; each step is a bounded row sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_descriptors(args)
    k_pool, v_pool, q = host_layer(w, seed=12345)
    masks = None
    if args.sparsity > 0:
        from paper_2606_15319_b200 import workloads as W
        masks = W.random_block_masks(w, args.sparsity, seed=9000)
    # size the per-step sample so that warmup+steps finish within a few minutes (about 4 s of CPU per step)
    time_oracle(w, k_pool, v_pool, q, 64, masks)                                   # cold pass (imports, page faults)
    dt, fl, *_ = time_oracle(w, k_pool, v_pool, q, 64, masks)
    n_rows = int(max(64, min(w.total_q, 64 * 4.0 / max(dt, 1e-3))))
    for _ in range(args.warmup):
        time_oracle(w, k_pool, v_pool, q, n_rows, masks)
    t, f = 0.0, 0.0
    for _ in range(args.steps):
        dt, fl, *_ = time_oracle(w, k_pool, v_pool, q, n_rows, masks)
        t += dt
        f += fl
    val = f / t / 1e12
    cores = blas_threads()
    sample = f"{n_rows} seeded query rows x all heads x all visible keys of one layer per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(args, w), "sample": sample, "sparsity": args.sparsity},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


# ---------------------------------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------------------------------

# dram__bytes_read.sum + dram__bytes_write.sum per attention-kernel launch, from the committed `ncu --set full` capture
# of that workload (ncu cannot run inside a timed bench; profiles/ names the command): null where none was taken.
NCU_TRAFFIC_BYTES = {
    "cfg2": (216167680, "profiles/r01_ncu_full_cfg2.md"),
    "cfg5": (1038073088, "profiles/r02_ncu_full_cfg5_final.md"),   # Lk = 32760 only
}


def load_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


def measure(ctx, args, name, steps, warmup, rank, world, local, dist, *, want_e2e, want_cpu, want_xfer, sparsity=0.0,
            sample_clocks=True, dtype=None):
    """One workload: fills 30 layers of pools on the device, times `steps` steps, returns the pieces of the JSON line."""
    import torch
    from paper_2606_15319_b200 import binding, metrics

    dev = torch.device("cuda", local)
    w = make_descriptors(args, seed_shift=rank, workload=name)       # replicas: each rank has its own batch, same shapes
    L, H, D, P = args.layers, w.n_heads, w.head_dim, w.page_size
    tq = w.total_q
    gen = torch.Generator(device=dev)
    gen.manual_seed(777 + rank)
    rnd = lambda *shape: (torch.randn(*shape, device=dev, dtype=torch.float32, generator=gen) * 0.5).to(torch.bfloat16)
    fp8 = (dtype or args.dtype) == "fp8"
    pools, qs, kns, vns, outs = [], [], [], [], []
    for l in range(L):
        if fp8:
            # e4m3 codes of the same N(0, 0.25) values under one scale per block (5 sigma / 448, saturating: torch's cast
            # alone turns values beyond 448 into the NaN code); torch's cast only builds
            # the synthetic cache contents here - every chunk the bench appends is quantised by slack_kv_append itself
            sc = 2.5 / 448.0
            kp = torch.empty(w.n_pages, H, P, D, device=dev, dtype=torch.uint8)
            vp = torch.empty_like(kp)
            for t in (kp, vp):
                for a in range(0, w.n_pages, 64):
                    t[a:a + 64] = (rnd(min(64, w.n_pages - a), H, P, D).float() / sc).clamp_(-448.0, 448.0).to(torch.float8_e4m3fn).view(torch.uint8)
            ks = torch.full((w.n_pages, H, P // 128), sc, device=dev, dtype=torch.float32)
            pools.append(binding.Pool(kp, vp, w.n_pages, H, D, P, "fp8", k_scale=ks, v_scale=ks.clone()))
        else:
            kp = torch.empty(w.n_pages, H, P, D, device=dev, dtype=torch.bfloat16)
            vp = torch.empty_like(kp)
            for t in (kp, vp):                             # fill page by page-block to bound the fp32 temporary
                for a in range(0, w.n_pages, 64):
                    t[a:a + 64] = rnd(min(64, w.n_pages - a), H, P, D)
            pools.append(binding.Pool(kp, vp, w.n_pages, H, D, P, "bf16"))
        qs.append(rnd(tq, H, D)); kns.append(rnd(tq, H, D)); vns.append(rnd(tq, H, D))
        outs.append(torch.empty(tq, H, D, device=dev, dtype=torch.bfloat16))
    main = torch.cuda.current_stream()
    plan0 = ctx.slack_plan(pools[0], w.streams, force_splits=args.force_splits, cta_pairs=args.cta_pairs)
    ws = torch.empty(max(plan0.workspace_bytes, plan0.sparse_workspace_bytes if sparsity > 0 else 0, 256),
                     dtype=torch.uint8, device=dev)
    # block-sparse variant: a seeded mask per layer (the selection rule, Light Forcing's [39] P:319, is outside the path)
    layer_masks, masks_d = None, None
    if sparsity > 0:
        from paper_2606_15319_b200 import workloads as W
        layer_masks = [W.random_block_masks(w, sparsity, seed=9000 + 100 * rank + l) for l in range(L)]
        masks_d = [torch.from_numpy(W.pack_block_masks(w, m).view(np.int32)).to(dev) for m in layer_masks]
    plan_info = {"items": plan0.num_items, "partial_slots": plan0.num_partial_slots, "kernel_kind": plan0.kernel_kind}
    del plan0
    state = {"launches": 0, "plan_s": 0.0}

    def step(q_of=lambda l: qs[l], kn_of=lambda l: kns[l], vn_of=lambda l: vns[l], out_of=lambda l: outs[l],
             pre=lambda l: None, post=lambda l: None):
        t0 = time.perf_counter()
        plan = ctx.slack_plan(pools[0], w.streams, force_splits=args.force_splits, cta_pairs=args.cta_pairs)      # A0 + A2 (host), once per step
        state["plan_s"] += time.perf_counter() - t0
        for l in range(L):
            pre(l)
            ctx.slack_kv_append_planned(plan, pools[l], kn_of(l), vn_of(l), stream=main)             # A1
            state["launches"] += ctx.last_launch_count
            if masks_d is None:
                ctx.slack_chunk_attention(plan, pools[l], q_of(l), out_of(l), w.scale, workspace=ws, stream=main)  # A3 + A4
            else:
                ctx.slack_chunk_attention_sparse(plan, pools[l], q_of(l), out_of(l), w.scale, masks_d[l], workspace=ws,
                                                 stream=main)
            state["launches"] += ctx.last_launch_count
            post(l)
        del plan    # slack_plan_destroy: the tables go back to the ctx arena behind an event, no device synchronisation

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(step_fn, steps, warmup, after=lambda: None):
        """-> (ms of the whole region, [ms of every step]); an event at every step boundary, nothing inside a step."""
        for _ in range(warmup):
            step_fn()
        after()
        barrier()
        state["launches"], state["plan_s"] = 0, 0.0
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        ev[0].record(main)
        for i in range(steps):
            step_fn()
            if i + 1 < steps:
                ev[i + 1].record(main)
        after()
        ev[steps].record(main)
        barrier()
        return ev[0].elapsed_time(ev[steps]), [ev[i].elapsed_time(ev[i + 1]) for i in range(steps)]

    if layer_masks is None:
        flops_layer = metrics.attention_flops(w.streams, H, D)
        flops_step = flops_layer * L
    else:                                             # selected (query, key) pairs only
        per_layer = [4.0 * D * selected_pairs(w, m) for m in layer_masks]
        flops_step = float(sum(per_layer))
        flops_layer = flops_step / L

    # ---- device-resident timing (value) + per-kernel roofline ------------------------------------------------------
    sampler = ClockSampler(local) if (rank == 0 and sample_clocks) else None
    ms_local, step_ms = timed(step, steps, warmup)    # the timed region of `value`: no profiling events inside a step
    launches = state["launches"]
    plan_ms = 1e3 * state["plan_s"] / steps
    ms, job_flops_step = reduce_job(dist, ms_local, flops_step, dev)    # MAX of the time, SUM of the work over ranks
    value = job_flops_step * steps / (ms * 1e-3) / 1e12
    # the same K steps once more with the library's event pairs around every append / attention / combine kernel
    ctx.profile_enable(binding.PROF_ATTENTION | binding.PROF_APPEND | binding.PROF_COMBINE)
    ms_prof, _ = timed(step, steps, 0)
    k_list = ctx.profile_read(binding.PROF_ATTENTION)
    a_list = ctx.profile_read(binding.PROF_APPEND)
    c_list = ctx.profile_read(binding.PROF_COMBINE)
    ctx.profile_enable(0)
    k_ms, k_n = float(sum(k_list)), len(k_list)
    clocks = sampler.stop() if sampler else None

    # ---- end to end: inputs from pinned host memory, output read back, inside the timed region ----------------------
    e2e = None
    if want_e2e:
        pin = lambda t: t.cpu().pin_memory()
        hq, hkn, hvn = [pin(t) for t in qs], [pin(t) for t in kns], [pin(t) for t in vns]
        hout = [torch.empty(tq, H, D, dtype=torch.bfloat16).pin_memory() for _ in range(L)]
        s_in, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        NB = 3                                          # staging depth: copies of layer l+1.. overlap compute of layer l
        dq = [torch.empty_like(qs[0]) for _ in range(NB)]
        dkn, dvn, dout = [torch.empty_like(qs[0]) for _ in range(NB)], [torch.empty_like(qs[0]) for _ in range(NB)], \
            [torch.empty_like(qs[0]) for _ in range(NB)]
        ev_in = [torch.cuda.Event() for _ in range(NB)]
        ev_free_in = [torch.cuda.Event() for _ in range(NB)]
        ev_done = [torch.cuda.Event() for _ in range(NB)]
        ev_free_out = [torch.cuda.Event() for _ in range(NB)]

        def pre(l):
            b = l % NB
            with torch.cuda.stream(s_in):
                s_in.wait_event(ev_free_in[b])          # compute that last read staging buffer b has finished
                dq[b].copy_(hq[l], non_blocking=True)
                dkn[b].copy_(hkn[l], non_blocking=True)
                dvn[b].copy_(hvn[l], non_blocking=True)
                ev_in[b].record(s_in)
            main.wait_event(ev_in[b])
            main.wait_event(ev_free_out[b])             # the previous result in dout[b] has been read back

        def post(l):
            b = l % NB
            ev_free_in[b].record(main)
            ev_done[b].record(main)
            with torch.cuda.stream(s_out):
                s_out.wait_event(ev_done[b])
                hout[l].copy_(dout[b], non_blocking=True)
                ev_free_out[b].record(s_out)

        e2e_step = lambda: step(q_of=lambda l: dq[l % NB], kn_of=lambda l: dkn[l % NB], vn_of=lambda l: dvn[l % NB],
                                out_of=lambda l: dout[l % NB], pre=pre, post=post)
        e2e_steps = max(2, min(steps, 5))               # PCIe-bound: a few steps are a stable sample
        ms_e2e_local, _ = timed(e2e_step, e2e_steps, 2, after=lambda: main.wait_stream(s_out))
        ms_e2e, _ = reduce_job(dist, ms_e2e_local, flops_step, dev)
        bytes_in = 3 * tq * H * D * 2 * L
        bytes_out = tq * H * D * 2 * L
        e2e = {"value": job_flops_step * e2e_steps / (ms_e2e * 1e-3) / 1e12, "unit": UNIT,
               "h2d_bytes_per_step": bytes_in, "d2h_bytes_per_step": bytes_out, "ms_per_step": ms_e2e / e2e_steps,
               "steps": e2e_steps, "pcie_gb_per_s": (bytes_in + bytes_out) * e2e_steps / (ms_e2e * 1e-3) / 1e9,
               "overlap": "H2D / compute / D2H on three streams, 3-deep staging"}
        # the e2e path must produce the same bits as the device-resident path (same inputs, same plan)
        torch.cuda.synchronize()
        assert torch.equal(hout[L - 1].view(torch.int16), outs[L - 1].cpu().view(torch.int16)), "e2e output differs from the device-resident run"
        assert bool(torch.isfinite(outs[L - 1]).all()), "non-finite attention output"
        del hq, hkn, hvn, hout, dq, dkn, dvn, dout

    # ---- state-plane page transfer (NEXT-4): stream 0's pages, all layers, HBM pool -> second HBM pool ----------------
    xfer = None
    peaks = load_peaks()
    if want_xfer and rank == 0:
        s0 = w.streams[0]
        sp = np.asarray(s0.page_table, dtype=np.int32)
        dst_pools = []
        for l in range(L):
            kp = torch.empty(sp.size, H, P, D, device=dev, dtype=torch.bfloat16)
            dst_pools.append(binding.Pool(kp, torch.empty_like(kp), int(sp.size), H, D, P, "bf16"))
        dp = np.random.default_rng(3).permutation(sp.size).astype(np.int32)
        for _ in range(3):
            ctx.slack_kv_transfer(pools, dst_pools, sp, dp, 0, H, stream=main)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 5
        e0.record(main)
        for _ in range(reps):
            ctx.slack_kv_transfer(pools, dst_pools, sp, dp, 0, H, stream=main)
        e1.record(main)
        torch.cuda.synchronize()
        x_ms = e0.elapsed_time(e1) / reps
        x_bytes = 2.0 * 2.0 * sp.size * H * P * D * 2 * L          # K and V, read + write, all layers
        same = all(torch.equal(dst_pools[l].k_pool[int(dp[i])], pools[l].k_pool[int(sp[i])]) for l in (0, L - 1) for i in (0, sp.size - 1))
        xfer = {"pages": int(sp.size), "layers": L, "bytes_moved": x_bytes, "ms": x_ms, "GB_per_s": x_bytes / (x_ms * 1e-3) / 1e9,
                "frac_of_hbm_peak": None, "spot_check_equal": bool(same), "kernel": "kv_transfer_kernel, one launch per layer"}
        if "hbm_gbs" in peaks:
            xfer["frac_of_hbm_peak"] = xfer["GB_per_s"] / float(peaks["hbm_gbs"])
        del dst_pools

    # ---- roofline of the dominant kernel; append and combine beside it ----------------------------------------------
    burst = float(peaks["bf16_tflops"]) if "bf16_tflops" in peaks else 1590.0
    which = "MEASURED_PEAKS.json bf16_tflops (burst: SURVEY.md A11 headline denominator)" if "bf16_tflops" in peaks else \
        "fallback: B200_PROFILING.md 1.59 PFLOP/s burst (MEASURED_PEAKS.json absent)"
    sustained = float(peaks["bf16_tflops_sustained"]) if "bf16_tflops_sustained" in peaks else None
    if fp8:   # a contraction takes the peak of its own dtype: the measured bf16 figure x the nominal fp8 : bf16 ratio of 2
        burst, sustained = 2.0 * burst, (2.0 * sustained if sustained else None)
        which += " x 2 (nominal fp8 : bf16 ratio, B200_PROFILING.md)"
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    hbm_src = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    kernel_ms = k_ms / max(k_n, 1)
    achieved = flops_layer / (kernel_ms * 1e-3) / 1e12 if k_n else None
    # minimal HBM bytes of one launch: Q read, Out written, every visible K and V read once per (stream, head)
    bytes_layer = metrics.attention_min_bytes(w.streams, H, D, 2)
    if fp8:   # K and V are one byte per element; Q and Out stay bf16
        bytes_layer = float(sum((2 * s.q_len * 2 + 2 * lk * 1) * H * D for s, lk in zip(w.streams, metrics.visible_keys(w.streams))))
    intensity = flops_layer / bytes_layer
    traffic, traffic_src = NCU_TRAFFIC_BYTES.get(name if (layer_masks is None and (name != "cfg5" or args.kv_chunks == 7)) else "", (None, None))
    stats = lambda xs: {"ms_avg": float(np.mean(xs)), "ms_median": float(np.median(xs)), "ms_min": float(np.min(xs)),
                        "launches_timed": len(xs)} if len(xs) else None
    if layer_masks is None and intensity < burst * 1e12 / (hbm_peak * 1e9):
        # decode-like short chunks (cfg5b): fewer flops per K/V byte than the ridge point -> HBM-bound
        gbs = bytes_layer / (kernel_ms * 1e-3) / 1e9 if k_n else None
        roofline = {"bound": "hbm", "kernel": "attn_tc_kernel", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s",
                    "frac": (gbs / hbm_peak) if gbs else None, "traffic": traffic, "traffic_source": traffic_src,
                    "peak_source": hbm_src, "kernel_ms_avg": kernel_ms, "kernel_ms": stats(k_list), "launches_timed": k_n,
                    "bytes_per_launch": bytes_layer, "flops_per_byte": intensity,
                    "ridge_flops_per_byte": burst * 1e12 / (hbm_peak * 1e9), "tflops": achieved,
                    "kernel_share_of_step": (k_ms / ms_prof) if k_n else None}
    else:
        roofline = {"bound": "tensor", "kernel": "attn_tc_kernel", "achieved": achieved, "peak": burst, "unit": "TFLOP/s",
                    "frac": (achieved / burst) if achieved else None, "traffic": traffic, "traffic_source": traffic_src,
                    "peak_source": which, "kernel_ms_avg": kernel_ms, "kernel_ms": stats(k_list), "launches_timed": k_n,
                    "flops_per_launch": flops_layer, "algorithmic_bytes_per_launch": bytes_layer,
                    "frac_of_sustained": (achieved / sustained) if achieved and sustained else None,
                    "frac_of_nominal_2250": (achieved / 2250.0) if achieved else None,
                    "kernel_share_of_step": (k_ms / ms_prof) if k_n else None}
    app_bytes = metrics.append_bytes(w.streams, H, D, 2) * (0.75 if fp8 else 1.0)   # fp8: bf16 read, 1-byte codes written
    append = stats(a_list)
    if append:
        append.update(kernel="kv_append_kernel", bytes_per_launch=app_bytes, GB_per_s=app_bytes / (append["ms_avg"] * 1e-3) / 1e9,
                      GB_per_s_best=app_bytes / (append["ms_min"] * 1e-3) / 1e9, peak=hbm_peak, peak_source=hbm_src,
                      share_of_step=float(sum(a_list)) / ms_prof)
        append["frac_of_hbm"] = append["GB_per_s"] / hbm_peak
    combine = stats(c_list)
    if combine:
        combine.update(kernel="combine_kernel", share_of_step=float(sum(c_list)) / ms_prof)

    # ---- CPU baseline: the oracle on layer 0 of this very run (also a live parity spot check) ----------------------
    cpu, parity = None, None
    if want_cpu and rank == 0 and fp8:
        # the FP8 oracle (oracle/fp8_attention.py) on a row sample of layer 0: dequantised operands, exact P
        import oracle
        Fo = oracle.fp8_attention
        img = [t.cpu().numpy() for t in (pools[0].k_pool, pools[0].v_pool, pools[0].k_scale, pools[0].v_scale)]
        q0 = binding.to_numpy(qs[0], "bf16")
        rows = sample_rows(w.streams, 256)
        t0 = time.perf_counter()
        o_want, _ = Fo.chunk_attention_fp8(img[0], img[1], img[2], img[3], w.streams, q0, w.scale, "bf16", rows=rows)
        dt = time.perf_counter() - t0
        fl = sample_flops(w.streams, rows, H, D)
        ma, rf = oracle.error_metrics(outs[0].float().cpu().numpy().astype(np.float64), o_want)
        parity = {"rows": int(sum(len(r) for r in rows)), "max_abs": ma, "rel_fro": rf, "pass": bool(ma <= 2e-2 and rf <= 4e-2),
                  "against": "oracle.fp8_attention.chunk_attention_fp8 (dequantised Q, K, V; exact P); gate rel-Fro 4e-2"}
        cpu = {"value": fl / dt / 1e12, "unit": UNIT, "cores": blas_threads(), "kind": "oracle", "seconds": dt,
               "sample": f"{parity['rows']} seeded query rows x {H} heads x all visible keys of layer 0 (fp64 numpy, incl. dequantising the pool)"}
    elif want_cpu and rank == 0:
        kp0 = binding.to_numpy(pools[0].k_pool, "bf16")
        vp0 = binding.to_numpy(pools[0].v_pool, "bf16")
        q0 = binding.to_numpy(qs[0], "bf16")
        m0 = layer_masks[0] if layer_masks is not None else None
        time_oracle(w, kp0, vp0, q0, 64, m0)                                # cold pass (imports, page faults)
        dt, fl, rows, o_want, _ = time_oracle(w, kp0, vp0, q0, 64, m0)      # calibration pass
        dt, *_ = time_oracle(w, kp0, vp0, q0, 256, m0)                      # second calibration point (per-stream set-up amortised)
        n_rows = int(max(64, min(tq, 256 * 20.0 / max(dt, 1e-3), args.cpu_rows * 64)))   # about 20 s of CPU work
        dt, fl, rows, o_want, _ = time_oracle(w, kp0, vp0, q0, n_rows, m0)
        import oracle
        ma, rf = oracle.error_metrics(outs[0].float().cpu().numpy().astype(np.float64), o_want)
        parity = {"rows": int(sum(len(r) for r in rows)), "max_abs": ma, "rel_fro": rf, "pass": bool(ma <= 2e-2 and rf <= 1e-2)}
        cpu = {"value": fl / dt / 1e12, "unit": UNIT, "cores": blas_threads(), "kind": "oracle", "seconds": dt,
               "sample": f"{parity['rows']} seeded query rows x {H} heads x all visible keys of layer 0 (fp64 numpy)"}

    n_streams_job = world * len(w.streams)
    return {
        "value": value, "ms_per_step": ms / steps, "flops_step": flops_step, "job_flops_step": job_flops_step,
        "step_ms": {"median": float(np.median(step_ms)), "min": float(np.min(step_ms)), "max": float(np.max(step_ms)),
                    "of": "rank 0's per-step CUDA-event times"},
        "launches": launches, "plan_ms": plan_ms, "plan_info": plan_info, "clocks": clocks, "e2e": e2e, "xfer": xfer,
        "roofline": roofline, "append": append, "combine": combine, "cpu": cpu, "parity": parity, "w": w, "layers": L,
        "chunk_layers_per_s": n_streams_job * L * steps / (ms * 1e-3),
        "chunks_per_s": n_streams_job * steps / (ms * 1e-3) * (L / 30.0),
        "dense_flops_step": metrics.attention_flops(w.streams, H, D) * L, "sparse": layer_masks is not None,
    }


def run_ours(args):
    import gc
    import torch
    from paper_2606_15319_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device - the product path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    ctx = binding.Context(local)

    r = measure(ctx, args, args.workload, args.steps, args.warmup, rank, world, local, dist,
                want_e2e=not args.no_e2e, want_cpu=not args.no_cpu_baseline, want_xfer=args.transfer_bench,
                sparsity=args.sparsity)
    w = r["w"]

    # ---- supplementary blocks (N = 1 only): the other things `metric` / `north_star` name, a few steps each -----------
    others = {}
    if world == 1 and not args.no_others and args.sparsity == 0 and args.workload == "cfg5" and args.dtype == "bf16":
        blocks = (("cfg4", "cfg4", "bf16", 0.0, "configs[3] mixed streams: chunks/s"),
                  ("cfg3", "cfg3", "bf16", 0.0, "configs[2]: the 460 MB append"),
                  ("cfg5b", "cfg5b", "bf16", 0.0, "decode-like short chunks: HBM GB/s"),
                  ("cfg5_sparse_0.8", "cfg5", "bf16", 0.8, "block-sparse variant (P:88 knob (2)), selected flops"),
                  ("cfg5_fp8", "cfg5", "fp8", 0.0, "FP8 pool variant (P:88 knob (4)): peak = 2 x the bf16 burst figure"),
                  ("cfg5b_fp8", "cfg5b", "fp8", 0.0, "FP8 pool variant, decode-like: GB/s of 1-byte K/V"))
        for key, name, dt, rho, why in blocks:
            gc.collect()
            torch.cuda.empty_cache()
            o = measure(ctx, args, name, 5, 3, rank, world, local, dist, want_e2e=False, want_cpu=False, want_xfer=False,
                        sample_clocks=True, dtype=dt, sparsity=rho)
            rf, ap = o["roofline"], o["append"]
            others[key] = {"workload": workload_label(args, o["w"], name), "why": why, "dtype": dt, "sparsity": rho, "steps": 5,
                           "warmup": 3, "tflops": o["value"], "ms_per_step": o["ms_per_step"], "step_ms": o["step_ms"],
                           "chunks_per_s_30_layers_1_step": o["chunks_per_s"], "streams": len(o["w"].streams),
                           "attention": {k: rf.get(k) for k in ("bound", "achieved", "unit", "peak", "frac", "kernel_ms_avg",
                                                                "kernel_share_of_step", "tflops", "bytes_per_launch")},
                           "append": {k: ap.get(k) for k in ("ms_avg", "ms_min", "bytes_per_launch", "GB_per_s", "frac_of_hbm")} if ap else None,
                           "combine_ms_avg": o["combine"]["ms_avg"] if o["combine"] else None,
                           "clocks": o["clocks"]}
            del o

    if dist is not None:
        dist.barrier()
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    line = {"metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16" if args.dtype == "bf16" else "fp8_e4m3 (K/V pool codes, Q and P quantised online; fp32 accumulation; bf16 in/out)",
            "data": "synthetic",
            "config": {"workload": workload_label(args, w) + ("" if args.dtype == "bf16" else " [FP8 pool variant, NEXT-3]"), "layers_per_step": r["layers"], "streams": len(w.streams),
                       "l2": "inputs larger than L2: every layer has its own pools (no flush needed)",
                       "parallelism": "replicas only" if world > 1 else "1 GPU", "plan": r["plan_info"],
                       "flops_per_step": r["job_flops_step"], "chunk_layers_per_s": r["chunk_layers_per_s"],
                       "chunks_per_s_30_layers_1_step": r["chunks_per_s"],
                       "plan_ms_per_step_host": r["plan_ms"], "step_ms": r["step_ms"],
                       "sparsity": args.sparsity if r["sparse"] else 0.0,
                       "dense_flops_per_step": r["dense_flops_step"], "others": others or None},
            "clocks": r["clocks"], "e2e": r["e2e"], "gpu_launches": r["launches"], "roofline": r["roofline"],
            "append": r["append"], "combine": r["combine"], "cpu_baseline": r["cpu"], "parity_spot_check": r["parity"]}
    if r["xfer"] is not None:
        line["transfer"] = r["xfer"]
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
