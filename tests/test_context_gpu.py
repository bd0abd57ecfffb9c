"""Context life cycle: buffers a context owns survive each other's growth and are all released by
pinsage_destroy (regression tests for the round-1 bug where growing the fp32 split buffer freed the
hub-split pool's storage, and for storage that outlived the context)."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_1806_01973_b200 import binding, synth
from tests.parity import assert_rows_close, to_f64

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _skewed(N=120_000):
    cfg = synth.CONFIGS["cfg4"].scaled(N)
    X = synth.make_features(cfg, device=DEV)
    layers, head = synth.make_params(cfg, device=DEV)
    idx, counts = synth.make_graph(cfg, device=DEV)
    return cfg, X, layers, head, idx, counts


def _f32_dense(ctx, M, k, n, seed, out=None):
    g = torch.Generator().manual_seed(seed)
    A = torch.randn((M, k), generator=g).to(DEV)
    W = (torch.randn((n, k), generator=g) * k ** -0.5).to(DEV)
    got = ctx.pinsage_dense(A, W, None, False, out=out)
    return A, W, got


def test_hub_storage_survives_growth_of_the_split_buffer():
    """hub-split pool -> fp32 GEMMs that grow the split buffer twice -> hub-split pool again, one context:
    same bits as the first call and as a fresh context's."""
    cfg, X, layers, head, idx, counts = _skewed()
    with binding.Context(0) as ctx:
        ctx.pinsage_set_option("pool_hubs", 64)
        alpha = ctx.pinsage_normalize_counts(counts)
        first = ctx.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=32768).clone()
        ctx.pinsage_set_option("f32_split", 1)
        for M, k, n, seed in ((4096, 256, 256, 1), (16384, 1024, 512, 2)):     # the second one grows the buffer
            A, W, got = _f32_dense(ctx, M, k, n, seed)
            ref = O.dense(to_f64(A), to_f64(W), None, False)
            err = np.abs(to_f64(got) - ref).max() / np.abs(ref).max()
            assert err < 1e-5, err
        again = ctx.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=32768)
        torch.cuda.synchronize()
        assert torch.equal(first.view(torch.int16), again.view(torch.int16))
    with binding.Context(0) as fresh:
        fresh.pinsage_set_option("pool_hubs", 64)
        ref = fresh.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=32768)
        torch.cuda.synchronize()
        assert torch.equal(first.view(torch.int16), ref.view(torch.int16))


def test_destroy_releases_everything_the_context_allocated():
    """Free device memory before pinsage_create and after pinsage_destroy agrees to within a few MB after
    the hub-split pool, the fp32 split GEMM, pinsage_embed_nodes, a d = 1024 S3 (grid-wide norm exchange
    buffers), the host-buffer pipeline and pinsage_topk have all run.  Every output is preallocated so that
    torch's caching allocator does not move between the two readings."""
    cfg, X, layers, head, idx, counts = _skewed()
    alpha = torch.empty((cfg.N, cfg.T), dtype=torch.float32, device=DEV)
    out = torch.empty((cfg.N, cfg.d_out), dtype=torch.bfloat16, device=DEV)
    targets = torch.tensor([0, 5, cfg.N - 1], dtype=torch.int32, device=DEV)
    out_t = torch.empty((3, cfg.d_out), dtype=torch.bfloat16, device=DEV)
    g = torch.Generator().manual_seed(3)
    A32 = torch.randn((8192, 512), generator=g).to(DEV)
    W32 = torch.randn((512, 512), generator=g).to(DEV)
    o32 = torch.empty((8192, 512), dtype=torch.float32, device=DEV)
    H = torch.randn((20_000, 512), generator=g).to(torch.bfloat16).to(DEV)
    n = torch.randn((20_000, 512), generator=g).abs().to(torch.bfloat16).to(DEV)
    W = (torch.randn((1024, 1024), generator=g) / 32).to(torch.bfloat16).to(DEV)
    w = torch.zeros(1024, device=DEV)
    o3 = torch.empty((20_000, 1024), dtype=torch.bfloat16, device=DEV)
    hX = X[:30_000].cpu().pin_memory()
    hI = (idx[:30_000] % 30_000).cpu().pin_memory()
    hO = torch.empty((30_000, cfg.d_out), dtype=torch.bfloat16).pin_memory()
    torch.cuda.synchronize()
    # a first context warms up everything that is per-process (module loading, function attributes)
    for attempt in range(2):
        free0, _ = torch.cuda.mem_get_info(0)
        ctx = binding.Context(0)
        ctx.pinsage_normalize_counts(counts, out=alpha)
        ctx.pinsage_set_option("pool_hubs", 128)
        ctx.pinsage_embed_all(X, idx, alpha, layers, head, out=out)
        ctx.pinsage_set_option("pool_hubs", 0)
        ctx.pinsage_embed_nodes(X, idx, alpha, layers, head, targets, out=out_t)
        ctx.pinsage_set_option("f32_split", 1)
        ctx.pinsage_dense(A32, W32, None, True, out=o32)
        ctx.pinsage_combine(H, n, W, w, out=o3)
        hW = alpha[:30_000].cpu().pin_memory()
        ctx.pinsage_embed_all(hX, hI, hW, layers, head, out=hO)
        torch.cuda.synchronize()
        ctx.close()
        free1, _ = torch.cuda.mem_get_info(0)
    assert abs(free0 - free1) < (8 << 20), f"context leaked {(free0 - free1) / 2**20:.1f} MiB"


def test_pooled_width_is_checked_before_anything_runs():
    """fp32 rows wider than 4 KB are outside the pool kernels: UNSUPPORTED_SHAPE up front, for every entry."""
    N, T, d = 300, 5, 2048
    X = torch.zeros((N, 64), device=DEV)
    idx = torch.zeros((N, T), dtype=torch.int32, device=DEV)
    w = torch.zeros((N, T), device=DEV)
    lp = {"Q": torch.zeros((d, 64), device=DEV), "q": torch.zeros(d, device=DEV),
          "W": torch.zeros((d, 64 + d), device=DEV), "w": torch.zeros(d, device=DEV)}
    hp = {"G1": torch.zeros((64, d), device=DEV), "g": torch.zeros(64, device=DEV),
          "G2": torch.zeros((64, 64), device=DEV)}
    with binding.Context(0) as ctx:
        l0 = ctx.pinsage_launch_count()
        for call in (lambda: ctx.pinsage_layer(X, idx, w, lp),
                     lambda: ctx.pinsage_embed_all(X, idx, w, [lp], hp),
                     lambda: ctx.pinsage_embed_nodes(X, idx, w, [lp], hp,
                                                     torch.zeros(1, dtype=torch.int32, device=DEV)),
                     lambda: ctx.pinsage_pool(torch.zeros((N, d), device=DEV), idx, w)):
            with pytest.raises(binding.PinsageError) as e:
                call()
            assert e.value.status_name == "UNSUPPORTED_SHAPE", e.value
        assert ctx.pinsage_launch_count() == l0


def test_fp32_kernel_choice_follows_the_call_not_the_chunk():
    """In F32 the automatic split / SIMT choice is taken from the rows of the whole call, so small chunks,
    the automatic chunk and pinsage_embed_nodes (hint: the whole graph) give the same bits -- at a size
    where the whole graph takes the split tensor-core path (N x 64 x 64 >= 2^28)."""
    cfg = synth.CONFIGS["tiny"].scaled(70_000)
    X = synth.make_features(cfg, device=DEV)
    layers, head = synth.make_params(cfg, device=DEV)
    idx, counts = synth.make_graph(cfg, device=DEV)
    with binding.Context(0) as ctx:
        alpha = ctx.pinsage_normalize_counts(counts)
        whole = ctx.pinsage_embed_all(X, idx, alpha, layers, head)
        small = ctx.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=4096)
        t = torch.tensor([0, 69_999, 4095, 4096, 31_337], dtype=torch.int32, device=DEV)
        sub = ctx.pinsage_embed_nodes(X, idx, alpha, layers, head, t)
        torch.cuda.synchronize()
        assert torch.equal(whole.view(torch.int32), small.view(torch.int32))
        assert torch.equal(sub.view(torch.int32), whole[t.long()].view(torch.int32))
        # and it is the split path that ran: SIMT-only gives (slightly) different bits, same function
        ctx.pinsage_set_option("f32_split", 0)
        simt = ctx.pinsage_embed_all(X, idx, alpha, layers, head)
        torch.cuda.synchronize()
        assert not torch.equal(simt.view(torch.int32), whole.view(torch.int32))
        rows = np.array([0, 17, 69_999])
        assert_rows_close(to_f64(whole[rows]), to_f64(simt[rows]), torch.float32, "split vs SIMT rows")


def test_two_contexts_on_two_threads_share_nothing():
    """include/pinsage.h: different contexts may be used from different threads.  Two threads, each with its
    own context on its own stream, run different graphs at the same time (ctypes releases the GIL during a
    call) -- a uniform graph at d = 1024 (CTA pairs, the cooperative grid-wide norm exchange, cached tensor
    maps) and a skewed one (hub selection with its pinned read-back, hub-split pool, fused head) -- several
    times over; every result equals, bit for bit, what the same context configuration gives when it runs
    alone."""
    import threading
    jobs = []
    for name, N, opts in (("cfg3", 20_000, {}), ("cfg4", 150_000, {"pool_hubs": 64})):
        cfg = synth.CONFIGS[name].scaled(N)
        X = synth.make_features(cfg, device=DEV)
        layers, head = synth.make_params(cfg, device=DEV)
        idx, counts = synth.make_graph(cfg, device=DEV)
        with binding.Context(0) as ctx:
            for k, v in opts.items():
                ctx.pinsage_set_option(k, v)
            alpha = ctx.pinsage_normalize_counts(counts)
            alone = ctx.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=8192).clone()
        torch.cuda.synchronize()
        jobs.append(dict(X=X, idx=idx, alpha=alpha, layers=layers, head=head, opts=opts, alone=alone,
                         outs=[torch.empty_like(alone) for _ in range(4)], err=None))

    start = threading.Barrier(len(jobs))

    def work(job):
        try:
            s = torch.cuda.Stream(device=DEV)
            with binding.Context(0, stream=s.cuda_stream) as ctx:
                for k, v in job["opts"].items():
                    ctx.pinsage_set_option(k, v)
                start.wait()
                for out in job["outs"]:
                    ctx.pinsage_embed_all(job["X"], job["idx"], job["alpha"], job["layers"], job["head"],
                                          chunk_nodes=8192, out=out)
                s.synchronize()
        except Exception as ex:     # surfaced in the main thread
            job["err"] = ex

    threads = [threading.Thread(target=work, args=(j,)) for j in jobs]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=300)
        assert not t.is_alive(), "a worker thread hangs"
    torch.cuda.synchronize()
    for j in jobs:
        assert j["err"] is None, j["err"]
        for out in j["outs"]:
            assert torch.equal(out.view(torch.int16), j["alone"].view(torch.int16))
