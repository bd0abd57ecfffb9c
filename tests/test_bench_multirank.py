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


def test_bench_accounting_matches_survey_tables():
    """The algorithmic bytes / flops bench.py divides by are SURVEY.md 8(a) / 8(d)'s per-node figures:
    pool bytes T m e + 8 T + m e, GEMM flops 2 K N per row, arithmetic intensity per GEMM."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_1806_01973_b200 import synth
    # pool bytes per node: 26.5 KB / 104.8 KB / 52.6 KB / 52.5 KB at configs 2-5
    assert bench.pool_bytes_per_node(50, 256, 2) == 26_512
    assert bench.pool_bytes_per_node(50, 1024, 2) == 104_848
    assert bench.pool_bytes_per_node(50, 512, 2) == 52_624
    assert bench.pool_bytes_per_node(100, 256, 2) == 52_512
    # GEMM flops per node (SURVEY 8(a) totals): 9.83e5 / 2.10e7 / 3.93e6 / 1.44e6
    for name, flops in (("cfg2", 983_040), ("cfg3", 20_971_520), ("cfg4", 3_932_160), ("cfg5", 1_441_792)):
        cfg = synth.CONFIGS[name]
        assert bench.gemm_flops_per_node(cfg) == flops
        kinds = bench.gemm_kinds(cfg, -1)
        assert sum(k[3] for k in kinds) == flops                 # the per-kind split adds up
    # arithmetic intensities of SURVEY 8(d): S1 / S3 / S4 / S5 at config 2 = 128 / 171 / 128 / 85
    ai = {k[0]: k[3] / k[4] for k in bench.gemm_kinds(synth.CONFIGS["cfg2"], -1)}
    assert ai["S1 layer 1"] == 128 and round(ai["S3 layer 1"]) == 171 and ai["S4 head"] == 128
    assert round(ai["S5 head"]) == 85
    # the paper's geometry takes the linear-pool schedule (m = 2048 > d = 1024): P W2^T is its own GEMM
    names = [k[0] for k in bench.gemm_kinds(synth.CONFIGS["paper"], -1)]
    assert "P W2^T layer 1" in names and "P W2^T layer 2" in names
    assert sum(k[3] for k in bench.gemm_kinds(synth.CONFIGS["paper"], -1)) == bench.gemm_flops_per_node(
        synth.CONFIGS["paper"])


def test_e2e_leg_fits_the_host():
    """The e2e leg pins features, both tables and the output: the whole workload when that fits 60 % of the
    rank's share of host memory, else the largest sibling (a multiple of 10^6 nodes) that does."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_1806_01973_b200 import synth
    cfg = synth.CONFIGS["cfg5"]                                  # 512 + 800 + 512 bytes per node = 91.2 GB
    assert bench.e2e_nodes(cfg, 1, 196 << 30) == cfg.N
    n8 = bench.e2e_nodes(cfg, 8, 196 << 30)                      # eight ranks share the host
    assert 1_000_000 <= n8 < cfg.N and n8 % 1_000_000 == 0
    assert n8 * 1824 <= 0.6 * (196 << 30) / 8
