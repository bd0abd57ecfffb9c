"""Throughput of the exact top-K lookup (pinsage_topk) at the paper's evaluation shape (PAPER.md:289:
K = 500 neighbours of each query among 5 million candidates).

    python -m paper_1806_01973_b200.topk_bench [--queries Q] [--cands N] [--dim D] [--k K] [--dtype bf16|f32]

Prints one JSON line: queries/s, the GEMM's TFLOP/s share and the bytes the selection pass reads."""
import argparse
import json

import torch

from . import binding


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--queries", type=int, default=4096)
    ap.add_argument("--cands", type=int, default=5_000_000)
    ap.add_argument("--dim", type=int, default=1024)
    ap.add_argument("--k", type=int, default=500)
    ap.add_argument("--dtype", choices=["bf16", "f32"], default="bf16",
                    help="f32: fp32 embeddings, scores from the split (3 x bf16) tensor-core GEMM")
    ap.add_argument("--f32-split", type=int, default=-1, help="option f32_split (-1 auto, 0 SIMT, 1 split)")
    a = ap.parse_args()
    dev = "cuda:0"
    ctx = binding.Context(0)
    g = torch.Generator(device=dev).manual_seed(0)
    dt = torch.bfloat16 if a.dtype == "bf16" else torch.float32
    ctx.pinsage_set_option("f32_split", a.f32_split)
    Z = torch.empty((a.cands, a.dim), dtype=dt, device=dev)
    for s in range(0, a.cands, 1 << 20):
        e = min(a.cands, s + (1 << 20))
        z = torch.randn((e - s, a.dim), generator=g, device=dev)
        Z[s:e] = (z / z.norm(dim=1, keepdim=True)).to(dt)
    Q = Z[torch.randint(0, a.cands, (a.queries,), generator=g, device=dev)].clone()
    ctx.pinsage_set_option("profile", 1)
    best = float("inf")
    for it in range(3):
        ctx.pinsage_profile_read(-1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        idx, score = ctx.pinsage_topk(Q, Z, a.k)
        e1.record()
        torch.cuda.synchronize()
        if it >= 1:
            best = min(best, e0.elapsed_time(e1))
            gemm_ms, n_gemm = ctx.pinsage_profile_read(1)
    assert bool((idx[:, 0].long() >= 0).all())
    flops = 2.0 * a.queries * a.cands * a.dim
    print(json.dumps({"metric": "top-K queries/sec", "value": a.queries / (best * 1e-3), "ms": best,
                      "gemm_ms": gemm_ms, "gemm_tflops": flops / (gemm_ms * 1e-3) / 1e12,
                      "select_ms": best - gemm_ms,
                      "select_gbs": a.queries * a.cands * 4 / ((best - gemm_ms) * 1e-3) / 1e9,
                      "config": {"queries": a.queries, "candidates": a.cands, "dim": a.dim, "k": a.k,
                                 "dtype": a.dtype}}))
    ctx.close()


if __name__ == "__main__":
    main()
