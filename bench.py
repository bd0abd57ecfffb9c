#!/usr/bin/env python
"""bench.py -- node embeddings / s of K-layer PinSage inference (BASELINE.json's metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl ours|reference]

A step = one pass of the whole hot path (S1..S6 of include/pinsage.h: K layers + head over all
N nodes of the workload) = one ``pinsage_embed_all`` call.  One JSON line is printed by rank 0.

  value      nodes embedded per second, inputs already resident in HBM, CUDA-event timed on the
             context's stream, max over ranks.
  e2e        the same call with HOST (pinned) features / tables / output: H2D and D2H copies are
             inside the timed region.
  roofline   the dominant kernel (S2 pool): algorithmic bytes per launch / event-measured launch
             duration inside the timed region, against MEASURED_PEAKS.json's HBM figure.
  cpu_baseline  the fp64 oracle (oracle/, as it stands) on this box's host cores on a bounded
             sample of the same workload.  A reported baseline, not the target.

N > 1 (torchrun): the path does not shard in this library (replicas only),
so every rank embeds its own replica of the workload; scaling is "weak".
``--impl reference`` times the oracle itself (rank 0 only).
"""
from __future__ import annotations

import argparse
import dataclasses
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


def _peaks():
    """(hbm GB/s, bf16 TFLOP/s sustained, source)."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "measured"
    return 6650.0, 1400.0, "fallback"   # B200_PROFILING.md fallback figures


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


# ----------------------------------------------------------------------------- the CUDA arm
def run_ours(args, cfg):
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

    # ---- seeded synthetic inputs of the workload's shape, generated on the device -------------
    rcfg = replica_config(cfg, rank)
    X = synth.make_features(rcfg, device=dev)
    layers, head = synth.make_params(rcfg, device=dev)
    idx, counts = synth.make_graph(rcfg, device=dev)
    ctx = binding.Context(local)
    ctx.pinsage_set_option("gemm_impl", args.gemm_impl)
    ctx.pinsage_set_option("overlap", args.overlap)
    ctx.pinsage_set_option("gemm_cg", args.gemm_cg)
    ctx.pinsage_set_option("gemm_ns", args.gemm_ns)
    ctx.pinsage_set_option("gemm_epi", args.gemm_epi)
    ctx.pinsage_set_option("pool_slab", args.pool_slab)
    ctx.pinsage_set_option("gemm_nl", args.gemm_nl)
    ctx.pinsage_set_option("gemm_gx", args.gemm_gx)
    if args.pool_hubs is not None:
        ctx.pinsage_set_option("pool_hubs", args.pool_hubs)
    ctx.pinsage_set_option("linear_pool", args.linear_pool)
    alpha = ctx.pinsage_normalize_counts(counts)
    torch.cuda.synchronize()
    del counts
    torch.cuda.empty_cache()     # generator temporaries back to the driver: the library cudaMallocs
    out = torch.empty((cfg.N, cfg.d_out), dtype=X.dtype, device=dev)
    e = X.element_size()

    def step():
        ctx.pinsage_embed_all(X, idx, alpha, layers, head, out=out, chunk_nodes=args.chunk_nodes)

    for _ in range(args.warmup):
        step()
    barrier()

    # ---- timed region: K steps, CUDA events on the context's stream (= torch's current) -------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ctx.pinsage_set_option("profile", 1)
    ctx.pinsage_profile_read(-1)
    l0 = ctx.pinsage_launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = ctx.pinsage_launch_count() - l0
    prof = {name: ctx.pinsage_profile_read(kind) for kind, name in
            ((0, "pool"), (1, "dense"), (2, "combine"))}
    ctx.pinsage_set_option("profile", 0)
    ctx.pinsage_profile_read(-1)
    clocks = sampler.stop() if rank == 0 else None
    ms_max = max_over_ranks(ms, world, dev)
    assert torch.isfinite(out[:: max(1, cfg.N // 4096)].float()).all()

    # ---- e2e: the same public call with pinned HOST buffers, copies inside the timed region ---
    e2e = None
    if not args.no_e2e:
        hX = torch.empty(X.shape, dtype=X.dtype).pin_memory()
        hX.copy_(X)
        hI = torch.empty(idx.shape, dtype=idx.dtype).pin_memory()
        hI.copy_(idx)
        hW = torch.empty(alpha.shape, dtype=alpha.dtype).pin_memory()
        hW.copy_(alpha)
        hO = torch.empty(out.shape, dtype=out.dtype).pin_memory()
        h2d = hX.numel() * e + hI.numel() * 4 + hW.numel() * 4
        d2h = hO.numel() * e

        def step_host():
            ctx.pinsage_embed_all(hX, hI, hW, layers, head, out=hO, chunk_nodes=args.chunk_nodes)

        step_host()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        nrep = max(1, min(args.steps, 5))
        for _ in range(nrep):
            step_host()
        e1.record()
        barrier()
        te_max = max_over_ranks(e0.elapsed_time(e1), world, dev)
        assert torch.equal(hO[:1024].view(torch.int16 if e == 2 else torch.int32),
                           out[:1024].cpu().view(torch.int16 if e == 2 else torch.int32))
        e2e = {"value": job_throughput(cfg.N, nrep, world, te_max), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": nrep}
        del hX, hI, hW, hO

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (S2 pool) from the live event records ---------------
    hbm, tflops, src = _peaks()
    pool_ms, pool_n = prof["pool"]
    # gathered row width: m, or d in the linear-pool schedule (pooling the W2-projection)
    lin = args.linear_pool
    pool_bytes_step = sum(cfg.N * pool_bytes_per_node(cfg.T, d if (lin == 1 or (lin == -1 and m > d)) else m, e)
                          for _, m, d in cfg.layer_dims())
    pool_gbs = pool_bytes_step * args.steps / (pool_ms * 1e-3) / 1e9 if pool_ms > 0 else 0.0
    traffic = None      # DRAM bytes per launch from the committed ncu --set full capture, if any
    tp = os.path.join(ROOT, "profiles", "pool_traffic.csv")
    if os.path.exists(tp):
        for ln in open(tp).read().splitlines()[1:]:
            f = ln.split(",")
            if f and f[0] == cfg.name and int(f[1]) == (args.chunk_nodes or 0):
                # the capture is one full driver chunk: scale to the average launch of this run
                per_node = float(f[2]) / float(f[3])
                traffic = per_node * cfg.N * len(cfg.layer_dims()) * args.steps / max(pool_n, 1)
    kernels = {}
    for name, (kms, kn) in prof.items():
        kernels[name] = {"ms_per_step": kms / args.steps, "launches_per_step": kn / args.steps}
    dense_f = sum(2 * d_in * m for d_in, m, _ in cfg.layer_dims()) + 2 * cfg.hidden * cfg.g1 \
        + 2 * cfg.g1 * cfg.d_out
    comb_f = sum(2 * (d_in + m) * d for d_in, m, d in cfg.layer_dims())
    for d_in, m, d in cfg.layer_dims():          # linear pool: P W2^T is a dense launch, S3 keeps H W1^T
        if lin == 1 or (lin == -1 and m > d):
            dense_f += 2 * m * d
            comb_f -= 2 * m * d
    for name, f in (("dense", dense_f), ("combine", comb_f)):
        kms = prof[name][0]
        if kms > 0:
            kernels[name]["tflops"] = f * cfg.N * args.steps / (kms * 1e-3) / 1e12
            kernels[name]["frac_of_bf16_peak"] = kernels[name]["tflops"] / tflops
    kernels["pool"]["gbs"] = pool_gbs

    line = {
        "metric": METRIC, "value": job_throughput(cfg.N, args.steps, world, ms_max), "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16" if cfg.dtype == "bf16" else "f32",
        "data": "synthetic", "config": workload_config(cfg, args),
        "roofline": {"bound": "hbm", "kernel": "pool_kernel (S2)", "achieved": pool_gbs,
                     "peak": hbm, "unit": "GB/s", "frac": pool_gbs / hbm, "traffic": traffic,
                     "peak_source": f"{src} (MEASURED_PEAKS.json hbm_gbs)" if src == "measured"
                     else "fallback (B200_PROFILING.md)",
                     "algorithmic_bytes_per_launch": pool_bytes_step * args.steps / max(pool_n, 1),
                     "avg_launch_ms": pool_ms / max(pool_n, 1), "launches": pool_n,
                     # the same launch measured in DRAM bytes (ncu traffic / live duration): what is
                     # above 1.0 in `frac` is gathers served by L2, not work skipped
                     "dram_gbs": (traffic / (pool_ms / max(pool_n, 1) * 1e-3) / 1e9) if traffic and pool_ms > 0 else None,
                     "frac_dram": (traffic / (pool_ms / max(pool_n, 1) * 1e-3) / 1e9 / hbm) if traffic and pool_ms > 0 else None},
        "kernels": kernels,
        "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "gemm_impl": "tcgen05" if args.gemm_impl == 0 and cfg.dtype == "bf16" else "simt",
    }
    if not args.no_cpu and world == 1:
        line["cpu_baseline"], _ = cpu_baseline(cfg, args.cpu_seconds)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", help="tiny | cfg2 | cfg3 | cfg4 | cfg5 (full N)")
    ap.add_argument("--nodes", type=int, default=0, help="override N (a '-small' sibling)")
    ap.add_argument("--chunk-nodes", type=int, default=0)
    ap.add_argument("--gemm-impl", type=int, default=0, help="0 tcgen05, 1 SIMT reference kernels")
    ap.add_argument("--overlap", type=int, default=0)
    ap.add_argument("--gemm-cg", type=int, default=0, help="0 auto (CTA pairs), 1 single CTAs, 2 pairs")
    ap.add_argument("--gemm-ns", type=int, default=0, help="slab width without row norm: 0/256/512")
    ap.add_argument("--gemm-epi", type=int, default=0, help="0 auto (8 epilogue warps), 1 four")
    ap.add_argument("--linear-pool", type=int, default=-1, help="-1 auto (m > d), 0 off, 1 on")
    ap.add_argument("--pool-slab", type=int, default=-1, help="-1 auto, 0 whole rows, 32/64/128")
    ap.add_argument("--gemm-gx", type=int, default=1, help="wide S3 row norms: 1 global-memory exchange (cooperative launch), 2 same with a plain "
                         "launch (for ncu), 0 cluster exchange")
    ap.add_argument("--gemm-nl", type=int, default=0, help="row-norm GEMM slab width: 0/512 or 256")
    ap.add_argument("--pool-hubs", type=int, default=None,
                    help="hub-split pool: 0 off, -1 automatic, 64..512 forced (default: the library's)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3          # timing rule: at least 3 warm-up steps
    from paper_1806_01973_b200 import synth
    cfg = synth.CONFIGS[args.workload]
    if args.nodes:
        cfg = cfg.scaled(args.nodes)
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
