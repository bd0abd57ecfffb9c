"""Host logic of the N > 1 bench path on CPU: two gloo ranks, replicas only.
No kernel runs here; the ranks check the per-rank replica seeding, the max-over-ranks step time
and the whole-job throughput that bench.py prints."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    from paper_1806_01973_b200 import synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = bench.replica_config(synth.CONFIGS["tiny"], rank)
        idx, _ = synth.make_graph(cfg)                       # every rank draws its own replica
        ms = 10.0 + 5.0 * rank                               # rank 1 is the slow one
        ms_max = bench.max_over_ranks(ms, world, "cpu")
        q.put((rank, cfg.seed, int(idx.sum()), ms_max,
               bench.job_throughput(cfg.N, 4, world, ms_max)))
    finally:
        dist.destroy_process_group()


def test_two_rank_replicas_max_time_and_aggregate_throughput():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, seed0, sum0, max0, thr0), (r1, seed1, sum1, max1, thr1) = res
    assert (r0, r1) == (0, 1) and (seed0, seed1) == (0, 1)
    assert sum0 != sum1                                      # different replicas
    assert max0 == max1 == 15.0                              # the slowest rank's time, on both
    assert thr0 == thr1 == 2000 * 4 * 2 / 15e-3              # whole-job nodes/s


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(7.5, 1, "cpu") == 7.5
    assert bench.job_throughput(1000, 10, 1, 500.0) == 1000 * 10 / 0.5
