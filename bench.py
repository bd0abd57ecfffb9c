#!/usr/bin/env python
"""bench.py -- node embeddings / s of K-layer PinSage inference (BASELINE.json's metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload all|cfg2|cfg3|cfg4|cfg5|tiny]
                    [--impl ours|reference]

A step = one pass of the whole hot path (S1..S6 of include/pinsage.h: K layers + head over all
N nodes of the workload) = one ``pinsage_embed_all`` call.  One JSON line is printed by rank 0.

The default run (``--workload all``) times BASELINE.json's largest single-GPU configuration, config 5
(N = 5e7, T = 100, K = 3; BASELINE.json's ``metric`` names no configuration), as the headline and carries
configs 2, 3 and 4 in ``per_config`` (fewer steps each, same timing rules), so that every roofline claim
is measured by the same command:

  value        nodes embedded per second, inputs already resident in HBM, CUDA-event timed on the
               context's stream, max over ranks.
  e2e          the same call with HOST (pinned) features / tables / output: H2D and D2H copies are
               inside the timed region.
  roofline     the dominant kernel (S2 pool): algorithmic bytes per launch / event-measured launch
               duration inside the timed region, against MEASURED_PEAKS.json's HBM figure; next to it the
               calibration ceilings measured in this very run (``calib``: m1 read-only stream, m2 random-row
               gather from HBM, m3 random-row gather from L2 -- SURVEY.md 8(d)).
  roofline_gemm  S1 and S3 at the paper-shaped config 3, the one place the GEMMs are tensor-bound.
  per_config[*].gemm  per GEMM kind: TFLOP/s, its own bound min(sustained bf16 peak, AI x HBM GB/s) and
               the fraction of that bound.
  cpu_baseline the fp64 oracle (oracle/, as it stands) on this box's host cores on a bounded
               sample of the headline workload.  A reported baseline, not the target.

N > 1 (torchrun): the path does not shard in this library (replicas only),
so every rank embeds its own replica of the workload; scaling is "weak".
``--impl reference`` times the oracle itself (rank 0 only).
"""
from __future__ import annotations

import argparse
import dataclasses
import gc
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "node embeddings/sec for K-layer inference"
UNIT = "nodes/s"
HEADLINE = "cfg5"                      # the largest single-GPU configuration of BASELINE.json
SIDE_CONFIGS = ("cfg2", "cfg3", "cfg4")


def _peaks():
    """(hbm GB/s, bf16 TFLOP/s burst, bf16 TFLOP/s sustained, source)."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        burst = float(d["bf16_tflops"])
        return float(d["hbm_gbs"]), burst, float(d.get("bf16_tflops_sustained", burst)), "measured"
    return 6650.0, 1590.0, 1400.0, "fallback"   # B200_PROFILING.md fallback figures


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML (nvidia-ml-py) every few ms while the
    timed region runs; falls back to polling nvidia-smi if NVML is unavailable."""
    REASONS = (("hw_slowdown", 0x8), ("sw_power_cap", 0x4), ("sw_thermal_slowdown", 0x20),
               ("hw_thermal_slowdown", 0x40))

    def __init__(self, index: int):
        self.index, self.sm, self.mask, self.max_mhz = index, [], 0, None
        self.stop_flag, self.th, self.nv = threading.Event(), None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self.h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        while not self.stop_flag.is_set():
            try:
                if self.nv is not None:
                    self.sm.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
                    self.mask |= int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                    self.stop_flag.wait(0.004)
                else:
                    r = subprocess.run(
                        ["nvidia-smi", "-i", str(self.index),
                         "--query-gpu=clocks.sm,clocks.max.sm,clocks_throttle_reasons.active",
                         "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5)
                    c = [x.strip() for x in r.stdout.strip().split(",")]
                    self.sm.append(float(c[0]))
                    self.max_mhz = float(c[1])
                    self.mask |= int(c[2], 16)
            except Exception:
                self.stop_flag.wait(0.05)

    def start(self):
        self.th = threading.Thread(target=self._run, daemon=True)
        self.th.start()

    def stop(self):
        self.stop_flag.set()
        if self.th:
            self.th.join(timeout=10)
        sm = sorted(self.sm)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(n for n, bit in self.REASONS if self.mask & bit),
                "samples": len(sm)}


def pool_bytes_per_node(T, m, e):
    """Algorithmic bytes of S2 per destination node: T gathered rows of P,
    the node's T (id, weight) pairs, one output row."""
    return T * m * e + 8 * T + m * e


def gemm_flops_per_node(cfg):
    f = 0
    for d_in, m, d in cfg.layer_dims():
        f += 2 * d_in * m + 2 * (d_in + m) * d
    f += 2 * cfg.hidden * cfg.g1 + 2 * cfg.g1 * cfg.d_out
    return f


def gemm_kinds(cfg, linear_pool: int):
    """The GEMMs of one step as (name, profile kind, layer, flops per node, HBM bytes per node): what the
    method must compute and move per node (weights amortise to zero; e = 2 bytes).  In the linear-pool
    schedule (m > d) S3 keeps only H W1^T and the projection P W2^T is its own launch."""
    e = 2 if cfg.dtype == "bf16" else 4
    out = []
    dims = cfg.layer_dims()
    for k, (d_in, m, d) in enumerate(dims, start=1):
        lin = linear_pool == 1 or (linear_pool == -1 and m > d)
        out.append((f"S1 layer {k}", 1, k, 2 * d_in * m, (d_in + m) * e))
        if lin:
            out.append((f"P W2^T layer {k}", 5, k, 2 * m * d, (m + d) * e))
            out.append((f"S3 layer {k}", 2, k, 2 * d_in * d, (d_in + 2 * d) * e))
        else:
            out.append((f"S3 layer {k}", 2, k, 2 * (d_in + m) * d, (d_in + m + d) * e))
    K = len(dims)
    out.append(("S4 head", 3, K, 2 * cfg.hidden * cfg.g1, (cfg.hidden + cfg.g1) * e))
    out.append(("S5 head", 4, K, 2 * cfg.g1 * cfg.d_out, (cfg.g1 + cfg.d_out) * e))
    return out


# ----------------------------------------------------------------------------- oracle legs
def oracle_sample_run(cfg, n_cpu: int):
    """Oracle mode B (layer-wise, fp64) on the n_cpu-node sibling of cfg.  Returns seconds."""
    import numpy as np
    import torch
    from oracle import oracle as O
    from paper_1806_01973_b200 import synth
    small = cfg.scaled(n_cpu)
    X = synth.make_features(small).to(torch.float64).numpy()
    layers, head = synth.make_params(small)
    idx, counts = synth.make_graph(small)
    Lf = [{k: v.to(torch.float64).numpy() for k, v in lp.items()} for lp in layers]
    Hf = {k: v.to(torch.float64).numpy() for k, v in head.items()}
    idx_np, cnt_np = idx.numpy(), counts.numpy()
    t0 = time.perf_counter()
    alpha = O.normalize_counts(cnt_np)
    out = O.embed_all(X, idx_np, alpha, Lf, Hf)
    dt = time.perf_counter() - t0
    assert np.isfinite(out).all()
    return dt


def cpu_baseline(cfg, target_s: float = 15.0):
    from oracle import oracle as O
    probe_n = 2000
    t_probe = oracle_sample_run(cfg, probe_n)
    n_cpu = int(max(probe_n, min(cfg.N, probe_n * target_s / max(t_probe, 1e-3))))
    n_cpu = max(cfg.T + 1, n_cpu // 1000 * 1000)
    dt = oracle_sample_run(cfg, n_cpu)
    return {"value": n_cpu / dt, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
            "sample": f"{n_cpu}-node sibling of {cfg.name} (same dims, T, K, value laws), "
                      f"fp64 layer-wise oracle, {dt:.1f} s"}, n_cpu


def run_reference(args, cfg):
    """--impl reference: the oracle as it stands, each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    probe_n = 2000
    t_probe = oracle_sample_run(cfg, probe_n)
    total_steps = args.steps + args.warmup
    per_step = max(1.0, min(20.0, 150.0 / total_steps))
    n_cpu = int(max(probe_n, min(cfg.N, probe_n * per_step / max(t_probe, 1e-3))))
    n_cpu = max(cfg.T + 1, n_cpu // 1000 * 1000)
    for _ in range(args.warmup):
        oracle_sample_run(cfg, n_cpu)
    t = [oracle_sample_run(cfg, n_cpu) for _ in range(args.steps)]
    tot = sum(t)
    value = n_cpu * args.steps / tot
    sample = f"{n_cpu}-node sibling of {cfg.name} per step, fp64 layer-wise oracle"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": workload_config(cfg, args, n_cpu),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def workload_config(cfg, args, n_nodes=None):
    return {"workload": f"{cfg.name}: N={n_nodes or cfg.N} nodes, d0={cfg.d0}, T={cfg.T}, K={cfg.K}, "
                        f"hidden={cfg.hidden}, head {cfg.hidden}->{cfg.g1}->{cfg.d_out}, {cfg.dtype}",
            "N": n_nodes or cfg.N, "T": cfg.T, "K": cfg.K, "d0": cfg.d0, "hidden": cfg.hidden,
            "g1": cfg.g1, "d_out": cfg.d_out, "parallelism": f"replicas x{args.gpus}",
            "l2": "inputs larger than L2 (features + tables + P exceed 126 MB; no flush needed)"}


# ----------------------------------------------------------------------------- multi-rank host logic
def replica_config(cfg, rank: int):
    """Replicas only: rank r embeds its own graph, drawn with seed + r."""
    return cfg if rank == 0 else dataclasses.replace(cfg, seed=cfg.seed + rank)


def max_over_ranks(ms: float, world: int, device) -> float:
    """The step time of the job is the slowest rank's (all-reduce MAX; identity at world 1)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(n_per_rank: int, steps: int, world: int, ms_max: float) -> float:
    """Whole-job nodes/s: every rank embeds n_per_rank nodes per step (weak scaling)."""
    return n_per_rank * steps * world / (ms_max * 1e-3)


def e2e_nodes(cfg, world: int, avail_bytes: int) -> int:
    """Nodes of the e2e leg: the whole workload when its pinned host buffers (features, both tables,
    output) fit 60 % of this rank's share of the available host memory, else the largest sibling that does
    (a multiple of 10^6 nodes; the copy volume per node is the same)."""
    e = 2 if cfg.dtype == "bf16" else 4
    per_node = cfg.d0 * e + 8 * cfg.T + cfg.d_out * e
    fit = int(0.6 * avail_bytes / max(world, 1) / per_node)
    if fit >= cfg.N:
        return cfg.N
    return max(min(cfg.N, 1_000_000), fit // 1_000_000 * 1_000_000)


# ----------------------------------------------------------------------------- the CUDA arm
def calibrate(ctx, dev):
    """Calibration kernels m1 / m2 / m3 (include/pinsage.h pinsage_calibrate): the read,
    random-row-gather (HBM) and random-row-gather (L2) ceilings of this device, in GB/s of gathered +
    written bytes, measured in this run."""
    import torch
    T = 50
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    table = torch.zeros(10 << 30, dtype=torch.uint8, device=dev)          # 10 GiB >> L2
    sink = torch.empty(sms * 8 * 256 * 16, dtype=torch.uint8, device=dev)
    res = {"how": f"pinsage_calibrate, 5 launches each after one warm-up; m1 streams a 10 GiB buffer; m2 gathers "
                  f"T = {T} hashed rows per destination from a 10 GiB table, m3 from a 32 MiB one; GB/s of "
                  f"gathered + written bytes"}
    ms = ctx.pinsage_calibrate(0, table, 0, 0, 0, sink, reps=5)
    res["m1_stream_read_gbs"] = table.numel() / (ms * 1e-3) / 1e9
    res["m2_gather_hbm_gbs"], res["m3_gather_l2_gbs"] = {}, {}
    small = table[: 32 << 20]
    for row in (256, 512, 1024, 2048):
        n_dst = int(16e9 / (T * row))
        out = torch.empty(n_dst * row, dtype=torch.uint8, device=dev)
        moved = n_dst * (T * row + row)
        for name, tab in (("m2_gather_hbm_gbs", table), ("m3_gather_l2_gbs", small)):
            ms = ctx.pinsage_calibrate(1, tab, row, n_dst, T, out, reps=5)
            res[name][str(row)] = moved / (ms * 1e-3) / 1e9
        del out
    del table, sink, small
    torch.cuda.empty_cache()
    return res


def _pool_traffic(cfg_name):
    """DRAM bytes per destination node of the pool from the committed ncu --set full capture of this
    config (profiles/pool_traffic.csv: name, chunk_nodes, dram_bytes, nodes, source), or None."""
    tp = os.path.join(ROOT, "profiles", "pool_traffic.csv")
    if not os.path.exists(tp):
        return None, None
    for ln in open(tp).read().splitlines()[1:]:
        f = [x.strip() for x in ln.split(",")]
        if len(f) >= 4 and f[0] == cfg_name:
            return float(f[2]) / float(f[3]), (f[4] if len(f) > 4 else "profiles/pool_traffic.csv")
    return None, None


def run_config(cfg, args, steps, warmup, env, with_clocks=False, e2e_steps=0):
    """Times `steps` calls of pinsage_embed_all on cfg (device-resident inputs) after `warmup` calls, reads
    the per-kernel event records, optionally runs the host-buffer (e2e) leg, and frees everything."""
    import psutil
    import torch
    from paper_1806_01973_b200 import binding, synth
    rank, world, local, dev, barrier = env
    hbm, burst, sustained, src = _peaks()

    t_gen = time.time()
    rcfg = replica_config(cfg, rank)
    X = synth.make_features(rcfg, device=dev)
    layers, head = synth.make_params(rcfg, device=dev)
    idx, counts = synth.make_graph(rcfg, device=dev)
    ctx = binding.Context(local)
    ctx.pinsage_set_option("gemm_impl", args.gemm_impl)
    ctx.pinsage_set_option("overlap", args.overlap)
    ctx.pinsage_set_option("gemm_cg", args.gemm_cg)
    ctx.pinsage_set_option("pool_slab", args.pool_slab)
    ctx.pinsage_set_option("gemm_gx", args.gemm_gx)
    ctx.pinsage_set_option("gemm_bres", args.gemm_bres)
    ctx.pinsage_set_option("head_fused", args.head_fused)
    if args.pool_hubs is not None:
        ctx.pinsage_set_option("pool_hubs", args.pool_hubs)
    ctx.pinsage_set_option("linear_pool", args.linear_pool)
    alpha = ctx.pinsage_normalize_counts(counts)
    torch.cuda.synchronize()
    del counts
    torch.cuda.empty_cache()     # generator temporaries back to the driver: the library cudaMallocs
    out = torch.empty((cfg.N, cfg.d_out), dtype=X.dtype, device=dev)
    e = X.element_size()
    t_gen = time.time() - t_gen

    def step():
        ctx.pinsage_embed_all(X, idx, alpha, layers, head, out=out, chunk_nodes=args.chunk_nodes)

    for _ in range(warmup):
        step()
    barrier()

    # ---- timed region: CUDA events on the context's stream (= torch's current stream) -------------
    sampler = ClockSampler(local) if (with_clocks and rank == 0) else None
    if sampler:
        sampler.start()
    ctx.pinsage_set_option("profile", 1)
    ctx.pinsage_profile_read(-1)
    l0 = ctx.pinsage_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(steps):
        step()
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = ctx.pinsage_launch_count() - l0
    kinds = gemm_kinds(cfg, args.linear_pool)
    pool_ms, pool_n = ctx.pinsage_profile_read(0)
    gemm_ms = {name: ctx.pinsage_profile_read(kind, layer) for name, kind, layer, _, _ in kinds}
    ctx.pinsage_set_option("profile", 0)
    ctx.pinsage_profile_read(-1)
    clocks = sampler.stop() if sampler else None
    ms_max = max_over_ranks(ms, world, dev)
    assert torch.isfinite(out[:: max(1, cfg.N // 4096)].float()).all()

    # ---- roofline of the dominant kernel (S2 pool) from the live event records --------------------
    lin = args.linear_pool
    pool_bytes_step = sum(cfg.N * pool_bytes_per_node(cfg.T, d if (lin == 1 or (lin == -1 and m > d)) else m, e)
                          for _, m, d in cfg.layer_dims())
    pool_gbs = pool_bytes_step * steps / (pool_ms * 1e-3) / 1e9 if pool_ms > 0 else 0.0
    per_node, tsrc = _pool_traffic(cfg.name)
    n_layers = len(cfg.layer_dims())
    traffic = per_node * cfg.N * n_layers * steps / max(pool_n, 1) if per_node else None
    roof = {"bound": "hbm", "kernel": "pool_kernel (S2)", "achieved": pool_gbs, "peak": hbm, "unit": "GB/s",
            "frac": pool_gbs / hbm, "traffic": traffic, "traffic_from": tsrc,
            "peak_source": f"{src} (MEASURED_PEAKS.json hbm_gbs: a copy, half reads half writes)"
            if src == "measured" else "fallback (B200_PROFILING.md)",
            "algorithmic_bytes_per_launch": pool_bytes_step * steps / max(pool_n, 1),
            "avg_launch_ms": pool_ms / max(pool_n, 1), "launches": pool_n,
            "ms_per_step": pool_ms / steps,
            "traffic_over_algorithmic": (traffic / (pool_bytes_step * steps / max(pool_n, 1))) if traffic else None}
    gemm = {}
    if gemm_ms["S5 head"][1] == 0 and gemm_ms["S4 head"][1] > 0:
        # the head ran as ONE launch (gemm_head.cu): its bytes are H read + out written, `a` stays on chip / in L2
        f4, f5 = kinds[-2][3], kinds[-1][3]
        kinds = kinds[:-2] + [("S4+S5 head (one launch)", 3, kinds[-1][2], f4 + f5, (cfg.hidden + cfg.d_out) * e)]
        gemm_ms["S4+S5 head (one launch)"] = gemm_ms["S4 head"]
    for name, kind, layer, flops, nbytes in kinds:
        kms, kn = gemm_ms[name]
        if kms <= 0:
            continue
        tf = flops * cfg.N * steps / (kms * 1e-3) / 1e12
        ai = flops / nbytes
        bound = min(sustained, ai * hbm / 1e3)
        gemm[name] = {"ms_per_step": kms / steps, "launches_per_step": kn / steps, "tflops": tf,
                      "ai_flop_per_byte": ai, "bound_tflops": bound,
                      "bound": "tensor" if bound == sustained else "hbm", "frac_of_bound": tf / bound,
                      "frac_of_nominal_2250": tf / 2250.0}
    plan = ctx.pinsage_last_plan()
    if "hubs=" in plan and "hubs=off" not in plan:
        roof["note"] = ("hub-split pool: the list entries that name a hub are not gathered (they enter S3 as a third K "
                        "segment), so `achieved` -- the plain definition's bytes over the pool's time -- is not a "
                        "bandwidth; the launch itself moves `traffic` bytes")
    rec = {"workload": workload_config(cfg, args)["workload"], "steps": steps, "warmup": warmup, "plan": plan,
           "ms_per_step": ms_max / steps, "value": job_throughput(cfg.N, steps, world, ms_max), "unit": UNIT,
           "roofline": roof, "gemm": gemm, "gpu_launches": int(launches), "gen_s": round(t_gen, 1)}
    if clocks is not None:
        rec["clocks"] = clocks

    # ---- e2e: the same public call with pinned HOST buffers, copies inside the timed region -------
    if e2e_steps > 0:
        n_e = e2e_nodes(cfg, world, psutil.virtual_memory().available)
        ref_rows = out[:1024].cpu()
        bits = torch.int16 if e == 2 else torch.int32
        try:
            hX = torch.empty((n_e, cfg.d0), dtype=X.dtype, pin_memory=True)
            hX.copy_(X[:n_e])
            del X
            hI = torch.empty((n_e, cfg.T), dtype=idx.dtype, pin_memory=True)
            hI.copy_(idx[:n_e])
            if n_e < cfg.N:                      # a sibling: ids must stay inside it
                hI.remainder_(n_e)
            del idx
            hW = torch.empty((n_e, cfg.T), dtype=alpha.dtype, pin_memory=True)
            hW.copy_(alpha[:n_e])
            del alpha, out
            torch.cuda.empty_cache()
            hO = torch.empty((n_e, cfg.d_out), dtype=hX.dtype, pin_memory=True)
            h2d = hX.numel() * e + hI.numel() * 4 + hW.numel() * 4
            d2h = hO.numel() * e

            def step_host():
                ctx.pinsage_embed_all(hX, hI, hW, layers, head, out=hO, chunk_nodes=args.chunk_nodes)

            step_host()
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(e2e_steps):
                step_host()
            e1.record()
            barrier()
            te_max = max_over_ranks(e0.elapsed_time(e1), world, dev)
            if n_e == cfg.N:
                assert torch.equal(hO[:1024].view(bits), ref_rows.view(bits)), "e2e output differs"
            rec["e2e"] = {"value": job_throughput(n_e, e2e_steps, world, te_max), "unit": UNIT,
                          "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
                          "ms_per_step": te_max / e2e_steps, "nodes": n_e,
                          "workload": "the headline workload" if n_e == cfg.N else
                          f"{n_e}-node sibling (pinned host buffers of the full workload exceed this host's memory)"}
            del hX, hI, hW, hO
        except RuntimeError as ex:           # pinned allocation refused
            rec["e2e"] = {"value": None, "unit": UNIT, "error": str(ex)[:200]}
    ctx.close()
    del ctx
    X = idx = alpha = out = layers = head = None
    gc.collect()
    torch.cuda.empty_cache()
    return rec


def run_extras(local, dev, which=("walks", "embed_nodes", "topk")):
    """The steps around the hot path, timed briefly so that their numbers reach
    the same record: the neighbourhood builder (the step before the path), targeted inference (Algorithm 2
    on a minibatch) and the exact top-K lookup (the step after it).  CUDA events, best of 3 after a warm-up.
    `--workload extras [--extras walks,topk]` runs these legs alone (the command the ncu captures use)."""
    import torch
    from paper_1806_01973_b200 import binding, synth
    res = {}

    def best_ms(fn, reps=3, warm=1):
        best = float("inf")
        for it in range(warm + reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize()
            if it >= warm:
                best = min(best, e0.elapsed_time(e1))
        return best

    g = torch.Generator(device=dev).manual_seed(5)
    with binding.Context(local) as ctx:
        if "walks" in which:
            # pinsage_build_neighbourhoods: N = 10^6, out-degrees uniform on [1, 40], 200 walks x 5 steps, T = 50
            N, walks, wlen, T = 1_000_000, 200, 5, 50
            row_ptr, col = synth.make_csr(N, 1, 40, law="uniform", seed=1, device=dev)
            ms = best_ms(lambda: ctx.pinsage_build_neighbourhoods(row_ptr, col, walks, wlen, T, 0))
            res["build_neighbourhoods"] = {"value": N / (ms * 1e-3), "unit": "neighbourhoods/s", "ms": ms,
                                           "walk_steps_per_s": N * walks * wlen / (ms * 1e-3),
                                           "config": {"N": N, "edges": int(col.numel()), "n_walks": walks,
                                                      "walk_len": wlen, "T": T}}
            del row_ptr, col
        if "embed_nodes" in which:
            # pinsage_embed_nodes on config 2's graph: 1 / 1024 / 16384 targets
            cfg = synth.CONFIGS["cfg2"]
            X = synth.make_features(cfg, device=dev)
            layers, head = synth.make_params(cfg, device=dev)
            idx, counts = synth.make_graph(cfg, device=dev)
            alpha = ctx.pinsage_normalize_counts(counts)
            del counts
            res["embed_nodes"] = {"graph": "cfg2", "unit": "ms per call"}
            for m in (1, 1024, 16384):
                t = torch.randint(0, cfg.N, (m,), generator=g, device=dev, dtype=torch.int32)
                res["embed_nodes"][str(m)] = best_ms(lambda: ctx.pinsage_embed_nodes(X, idx, alpha, layers, head, t))
            del X, idx, alpha, layers, head
            torch.cuda.empty_cache()
        if "topk" in which:
            # pinsage_topk at the paper's evaluation shape: K = 500 of 5 * 10^6 candidates, d = 1024
            nq, nc, d, k = 4096, 5_000_000, 1024, 500
            Z = torch.empty((nc, d), dtype=torch.bfloat16, device=dev)
            for s0 in range(0, nc, 1 << 20):
                e1 = min(nc, s0 + (1 << 20))
                z = torch.randn((e1 - s0, d), generator=g, device=dev)
                Z[s0:e1] = (z / z.norm(dim=1, keepdim=True)).to(torch.bfloat16)
            Q = Z[torch.randint(0, nc, (nq,), generator=g, device=dev)].clone()
            ms = best_ms(lambda: ctx.pinsage_topk(Q, Z, k), reps=2)
            res["topk"] = {"value": nq / (ms * 1e-3), "unit": "queries/s", "ms": ms,
                           "gemm_tflops_incl_selection": 2.0 * nq * nc * d / (ms * 1e-3) / 1e12,
                           "config": {"queries": nq, "candidates": nc, "dim": d, "k": k, "dtype": "bf16"}}
            del Z, Q
    torch.cuda.empty_cache()
    return res


def run_libgemm(local, dev, reps=10, rounds=3, only=None):
    """`--workload libgemm`: context for the GEMM rooflines, NOT part of the path or of the contract line.
    The plain GEMMs of configs 3-5 (no epilogue: the library routine has none) as pinsage_dense and as
    torch.matmul (cuBLAS), interleaved in one process on the same HBM-resident operands, in 2^20-row chunks as
    the layer driver issues them: what a vendor GEMM reaches on these streaming shapes under the same power
    cap.  TFLOP/s per round; CUDA events around `reps` back-to-back passes over all rows."""
    import torch
    from paper_1806_01973_b200 import binding
    shapes = [("cfg4 S1 / S4", 20_000_000, 512, 512), ("cfg4 S3 without the hub segment", 20_000_000, 1024, 512),
              ("cfg4 S3 with 256 hubs", 20_000_000, 1280, 512), ("cfg4 S5", 20_000_000, 512, 256),
              ("cfg3 S1", 5_000_000, 2048, 1024), ("cfg3 S3", 5_000_000, 3072, 1024),
              ("cfg3 S4 / S5", 5_000_000, 1024, 1024), ("cfg5 S1 / S4 / S5", 50_000_000, 256, 256),
              ("cfg5 S3", 50_000_000, 512, 256)]
    g = torch.Generator(device=dev).manual_seed(1)
    out_recs = []
    with binding.Context(local) as ctx:
        for si, (name, M, K, N) in enumerate(shapes):
            if only is not None and si not in only:
                continue
            A = torch.empty((M, K), dtype=torch.bfloat16, device=dev)
            for s0 in range(0, M, 1 << 21):
                A[s0:s0 + (1 << 21)].normal_(generator=g)
            W = (torch.randn((N, K), generator=g, device=dev) * K ** -0.5).to(torch.bfloat16)
            Wt = W.t()
            out = torch.empty((M, N), dtype=torch.bfloat16, device=dev)
            chunk = 1 << 20

            def lib():
                for s0 in range(0, M, chunk):
                    torch.matmul(A[s0:s0 + chunk], Wt, out=out[s0:s0 + chunk])

            def ours():
                for s0 in range(0, M, chunk):
                    ctx.pinsage_dense(A[s0:s0 + chunk], W, None, False, out=out[s0:s0 + chunk])

            rec = {"shape": name, "M": M, "K": K, "N": N, "unit": "TFLOP/s", "pinsage_dense": [], "torch_matmul": []}
            for _ in range(rounds):
                for key, fn in (("torch_matmul", lib), ("pinsage_dense", ours)):
                    fn()
                    torch.cuda.synchronize()
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record()
                    for _ in range(reps):
                        fn()
                    e1.record()
                    torch.cuda.synchronize()
                    rec[key].append(round(2.0 * M * K * N * reps / e0.elapsed_time(e1) / 1e9, 1))
            out_recs.append(rec)
            del A, W, Wt, out
            torch.cuda.empty_cache()
    return out_recs


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1806_01973_b200 import binding, synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}: launch with torchrun")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (B200); there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.workload == "extras":      # the legs around the path alone (profiles/: the ncu captures of walks / top-K)
        if rank == 0:
            print(json.dumps({"extras": run_extras(local, dev, tuple(args.extras.split(",")))}))
        if world > 1:
            dist.destroy_process_group()
        return
    if args.workload == "libgemm":     # context only: the library GEMM on the path's shapes (profiles/r02_gemm.md)
        if rank == 0:
            only = None if args.libgemm_shapes == "all" else {int(x) for x in args.libgemm_shapes.split(",")}
            print(json.dumps({"libgemm": run_libgemm(local, dev, reps=args.libgemm_reps, only=only)}))
        if world > 1:
            dist.destroy_process_group()
        return
    env = (rank, world, local, dev, barrier)
    everything = args.workload == "all"
    head_cfg = synth.CONFIGS[HEADLINE if everything else args.workload]
    if args.nodes:
        head_cfg = head_cfg.scaled(args.nodes)

    # ---- calibration ceilings of the day (rank 0's device; a few seconds) -------------------------
    calib = None
    if (everything or args.calib) and not args.no_calib:
        c = binding.Context(local)
        try:
            calib = calibrate(c, dev)
        finally:
            c.close()
        barrier()

    # ---- the headline workload, then the other BASELINE configs -----------------------------------
    e2e_steps = 0 if args.no_e2e else max(1, min(args.steps, 3))
    head = run_config(head_cfg, args, args.steps, args.warmup, env, with_clocks=True, e2e_steps=e2e_steps)
    per_config = []
    if everything:
        for name in SIDE_CONFIGS:
            rec = run_config(synth.CONFIGS[name], args, args.side_steps, max(3, min(args.warmup, 3)), env)
            rec["config"] = name
            per_config.append(rec)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    hbm, burst, sustained, src = _peaks()

    def against_calib(roof, cfg):
        """The pool against the ceilings measured in this run: m2 at its own row width (HBM-bound
        configs), m3 (the power-law config, whose gathers hit L2-resident hub rows), m1."""
        if not calib:
            return
        row = str(min(2048, max(256, cfg.hidden * 2)))
        roof["calib"] = {"row_bytes": int(row), "frac_of_m1_stream_read": roof["achieved"] / calib["m1_stream_read_gbs"],
                         "frac_of_m2_gather_hbm": roof["achieved"] / calib["m2_gather_hbm_gbs"][row],
                         "frac_of_m3_gather_l2": roof["achieved"] / calib["m3_gather_l2_gbs"][row]}

    against_calib(head["roofline"], head_cfg)
    for rec in per_config:
        against_calib(rec["roofline"], synth.CONFIGS[rec["config"]])

    line = {
        "metric": METRIC, "value": head["value"], "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16" if head_cfg.dtype == "bf16" else "f32",
        "data": "synthetic", "config": workload_config(head_cfg, args),
        "roofline": head["roofline"], "gemm": head["gemm"], "plan": head.get("plan"),
        "e2e": head.get("e2e"), "gpu_launches": head["gpu_launches"], "clocks": head.get("clocks"),
        "gemm_impl": "tcgen05" if args.gemm_impl == 0 and head_cfg.dtype == "bf16" else "simt",
        "peaks": {"hbm_gbs": hbm, "bf16_tflops_burst": burst, "bf16_tflops_sustained": sustained, "source": src},
    }
    if calib:
        line["calib"] = calib
    if per_config:
        line["per_config"] = per_config
        c3 = next((r for r in per_config if r["config"] == "cfg3"), None)
        if c3:      # the GEMM roofline where the GEMMs are tensor-bound: the paper-shaped config
            line["roofline_gemm"] = {
                "workload": c3["workload"], "bound": "tensor", "unit": "TFLOP/s", "peak": sustained,
                "peak_source": f"{src} (MEASURED_PEAKS.json bf16_tflops_sustained: the kernels are timed inside a long step)",
                "kernels": {k: {"achieved": v["tflops"], "frac": v["tflops"] / sustained,
                                "frac_of_nominal_2250": v["frac_of_nominal_2250"], "ms_per_step": v["ms_per_step"]}
                            for k, v in c3["gemm"].items()}}
    if everything and world == 1 and not args.no_extras:
        line["extras"] = run_extras(local, dev)
    if not args.no_cpu and world == 1:
        line["cpu_baseline"], _ = cpu_baseline(head_cfg, args.cpu_seconds)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="all",
                    help="all (default: cfg5 headline + cfg2-4 in per_config + calibration) | tiny | cfg2 | cfg3 | "
                         "cfg4 | cfg5 | paper (one workload at full N) | extras (only the legs around the path, "
                         "one JSON object; not the contract line) | libgemm (context: pinsage_dense and torch.matmul "
                         "on the path's GEMM shapes)")
    ap.add_argument("--side-steps", type=int, default=5, help="timed steps of each per_config entry")
    ap.add_argument("--nodes", type=int, default=0, help="override N (a '-small' sibling)")
    ap.add_argument("--chunk-nodes", type=int, default=0)
    ap.add_argument("--gemm-impl", type=int, default=0, help="0 tcgen05, 1 SIMT reference kernels")
    ap.add_argument("--overlap", type=int, default=0)
    ap.add_argument("--gemm-cg", type=int, default=0, help="0 auto (CTA pairs), 1 single CTAs, 2 pairs")
    ap.add_argument("--linear-pool", type=int, default=-1, help="-1 auto (m > d), 0 off, 1 on")
    ap.add_argument("--pool-slab", type=int, default=-1, help="-1 auto, 0 whole rows, 32/64/128")
    ap.add_argument("--gemm-gx", type=int, default=1,
                    help="wide S3 row norms: 1 global-memory exchange (cooperative launch), 2 the same with a plain "
                         "launch (for ncu, which cannot replay a cooperative one), 0 cluster exchange")
    ap.add_argument("--head-fused", type=int, default=1, help="1 S4 -> S5 in one launch where the shape allows, 2 its single-CTA form only, 0 two launches")
    ap.add_argument("--gemm-bres", type=int, default=1, help="1 stationary weights in shared memory at short K, 0 off")
    ap.add_argument("--pool-hubs", type=int, default=None,
                    help="hub-split pool: 0 off, -1 automatic, 64..512 forced (default: the library's)")
    ap.add_argument("--calib", action="store_true", help="run the calibration kernels with a single workload too")
    ap.add_argument("--no-calib", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the neighbourhood builder / embed_nodes / top-K legs")
    ap.add_argument("--extras", default="walks,embed_nodes,topk",
                    help="with --workload extras: which of the legs to run (comma-separated)")
    ap.add_argument("--libgemm-shapes", default="all", help="with --workload libgemm: indices 0..8 of the shapes to run")
    ap.add_argument("--libgemm-reps", type=int, default=10, help="with --workload libgemm: passes per timed figure")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3          # timing rule: at least 3 warm-up steps
    if args.impl == "reference":
        from paper_1806_01973_b200 import synth
        cfg = synth.CONFIGS[HEADLINE if args.workload in ("all", "extras", "libgemm") else args.workload]
        if args.nodes:
            cfg = cfg.scaled(args.nodes)
        run_reference(args, cfg)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
