"""Throughput of the neighbourhood builder (pinsage_build_neighbourhoods) on a synthetic CSR graph.

    python -m paper_1806_01973_b200.walk_bench [--nodes N] [--law uniform|zipf] [--walks R] [--len L] [--T T]

Prints one JSON line: nodes/s and walk steps/s (CUDA events, 2 warm-up calls, best of 3).  This is the
step BEFORE the hot path that bench.py measures (it runs once per graph, not once per inference)."""
import argparse
import json

import torch

from . import binding, synth


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--nodes", type=int, default=1_000_000)
    ap.add_argument("--law", default="uniform")
    ap.add_argument("--walks", type=int, default=200)
    ap.add_argument("--len", type=int, default=5, dest="walk_len")
    ap.add_argument("--T", type=int, default=50)
    ap.add_argument("--deg", type=int, default=40, help="out-degrees uniform on [1, deg]")
    a = ap.parse_args()
    dev = "cuda:0"
    ctx = binding.Context(0)
    row_ptr, col = synth.make_csr(a.nodes, 1, a.deg, law=a.law, seed=1, device=dev)
    best = float("inf")
    for it in range(5):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        idx, cnt = ctx.pinsage_build_neighbourhoods(row_ptr, col, a.walks, a.walk_len, a.T, 0)
        e1.record()
        torch.cuda.synchronize()
        if it >= 2:
            best = min(best, e0.elapsed_time(e1))
    print(json.dumps({"metric": "neighbourhoods built/sec", "value": a.nodes / (best * 1e-3),
                      "walk_steps_per_s": a.nodes * a.walks * a.walk_len / (best * 1e-3), "ms": best,
                      "config": {"N": a.nodes, "edges": int(col.numel()), "law": a.law, "n_walks": a.walks,
                                 "walk_len": a.walk_len, "T": a.T},
                      "non_padding_fraction": float((cnt > 0).float().mean())}))
    ctx.close()


if __name__ == "__main__":
    main()
