"""The layer driver (S6) of pinsage_embed_all: memory plan, buffer aliasing, host streaming.

SURVEY.md sec. 7.4 / PAPER.md:124 ("control the memory footprint"), BASELINE config 5 ("node chunks sized
to fit HBM"): P and one H are resident, everything else is per chunk; a device `out` as wide as every layer
doubles as H; host inputs are staged whole when that fits and streamed through rings of chunk slots when
it does not; the chunk shrinks before the call gives up.  Whatever the plan, the result is the same bits."""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_1806_01973_b200 import binding, synth
from tests.parity import assert_rows_close, params_f64, to_f64

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _inputs(cfg):
    X = synth.make_features(cfg)
    layers, head = synth.make_params(cfg)
    idx, counts = synth.make_graph(cfg)
    alpha = O.normalize_counts(counts.numpy())
    Ld = [{k: v.to(DEV) for k, v in lp.items()} for lp in layers]
    Hd = {k: v.to(DEV) for k, v in head.items()}
    return X, idx, torch.from_numpy(alpha), layers, head, Ld, Hd


def _oracle(X, idx, alpha, layers, head):
    Lf, Hf = params_f64(layers, head)
    return O.embed_all(to_f64(X), idx.numpy(), alpha.numpy(), Lf, Hf)


def test_out_serves_as_H_and_poisoned_buffers_are_never_read():
    """K = 3 at equal widths with d_out = d (config 5's shape): the caller's `out` is the one H buffer
    (plan says H=out), every layer after the first runs in place, the head of a chunk follows its last S3.
    With debug_poison every buffer is filled with NaN patterns the moment the plan says it is dead: the
    result must not change, and must match the oracle on every row."""
    cfg = synth.CONFIGS["cfg5"].scaled(9_000)
    X, idx, alpha, layers, head, Ld, Hd = _inputs(cfg)
    ref = _oracle(X, idx, alpha, layers, head)
    with binding.Context(0) as ctx:
        a = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), alpha.to(DEV), Ld, Hd, chunk_nodes=2048)
        assert "H=out" in ctx.pinsage_last_plan(), ctx.pinsage_last_plan()
        assert_rows_close(to_f64(a), ref, X.dtype, "H = out, K = 3")
        ctx.pinsage_set_option("debug_poison", 1)
        b = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), alpha.to(DEV), Ld, Hd, chunk_nodes=2048)
        c = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), alpha.to(DEV), Ld, Hd)            # one chunk
        torch.cuda.synchronize()
        assert torch.equal(a.view(torch.int16), b.view(torch.int16))
        assert torch.equal(a.view(torch.int16), c.view(torch.int16))
        # host output: H lives in the workspace again, out leaves through two chunk slots
        hO = torch.empty((cfg.N, cfg.d_out), dtype=X.dtype).pin_memory()
        ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), alpha.to(DEV), Ld, Hd, out=hO, chunk_nodes=2048)
        assert "H=workspace" in ctx.pinsage_last_plan() and "out=ring" in ctx.pinsage_last_plan()
        assert torch.equal(hO.view(torch.int16), a.cpu().view(torch.int16))


def test_changing_layer_widths_use_two_H_buffers_poisoned():
    """K = 3 with widths 128 -> 256 -> 256 -> 384 and d_out = 32: `out` cannot serve as H, layers 1 and 3 change
    width (ping-pong between two H buffers, the replaced one is poisoned), layer 2 runs in place."""
    N, T = 5_003, 10
    g = torch.Generator().manual_seed(77)

    def rn(*shape, std=1.0):
        return torch.randn(shape, generator=g) * std

    dims, ms, g1, d_out = [128, 256, 256, 384], [128, 256, 128], 136, 32
    X = rn(N, dims[0]).to(torch.bfloat16)
    layers = [{"Q": rn(ms[k], dims[k], std=dims[k] ** -0.5).to(torch.bfloat16), "q": rn(ms[k], std=0.01),
               "W": rn(dims[k + 1], dims[k] + ms[k], std=(dims[k] + ms[k]) ** -0.5).to(torch.bfloat16),
               "w": rn(dims[k + 1], std=0.01)} for k in range(3)]
    head = {"G1": rn(g1, dims[-1], std=dims[-1] ** -0.5).to(torch.bfloat16), "g": rn(g1, std=0.01),
            "G2": rn(d_out, g1, std=g1 ** -0.5).to(torch.bfloat16)}
    idx = torch.randint(0, N, (N, T), generator=g, dtype=torch.int32)
    alpha = torch.from_numpy(O.normalize_counts(torch.randint(1, 50, (N, T), generator=g, dtype=torch.int32).numpy()))
    ref = _oracle(X, idx, alpha, layers, head)
    Ld = [{k: v.to(DEV) for k, v in lp.items()} for lp in layers]
    Hd = {k: v.to(DEV) for k, v in head.items()}
    with binding.Context(0) as ctx:
        a = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), alpha.to(DEV), Ld, Hd, chunk_nodes=1024)
        assert "H=workspace+second" in ctx.pinsage_last_plan(), ctx.pinsage_last_plan()
        assert_rows_close(to_f64(a), ref, torch.bfloat16, "changing widths, K = 3")
        ctx.pinsage_set_option("debug_poison", 1)
        b = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), alpha.to(DEV), Ld, Hd, chunk_nodes=1024)
        torch.cuda.synchronize()
        assert torch.equal(a.view(torch.int16), b.view(torch.int16))


def test_memory_cap_gives_a_smaller_plan_not_an_error():
    """Config 5's shape (K = 3, T = 100) on 200 000 nodes with HOST inputs and output under an artificial
    memory cap (option mem_limit_mb): staged whole -> tables staged, features through a ring -> everything
    through rings; each plan gives the bits of the uncapped call.  Only a cap below what P and H need is
    PINSAGE_ERR_OOM.  Device inputs under a cap: the chunk shrinks."""
    cfg = synth.CONFIGS["cfg5"].scaled(200_000)
    X, idx, alpha, layers, head, Ld, Hd = _inputs(cfg)
    hX, hI, hW = X.pin_memory(), idx.pin_memory(), alpha.pin_memory()
    hO = torch.empty((cfg.N, cfg.d_out), dtype=X.dtype).pin_memory()
    with binding.Context(0) as ctx:
        ctx.pinsage_set_option("debug_poison", 1)
        dev = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), alpha.to(DEV), Ld, Hd)
        torch.cuda.synchronize()
        rows = np.random.default_rng(5).integers(0, cfg.N, 300)
        Lf, Hf = params_f64(layers, head)
        ref = O.minibatch_embed(rows, lambda ids: to_f64(X[ids]), lambda ids: (idx.numpy()[ids], alpha.numpy()[ids]),
                                Lf, Hf)
        assert_rows_close(to_f64(dev[rows]), ref, X.dtype, "cfg5-shaped sibling vs oracle")
        seen = []
        for cap, feats, tables in ((0, "staged", "staged"), (500, "ring", "staged"), (420, "ring", "ring")):
            ctx.pinsage_set_option("mem_limit_mb", cap)
            hO.zero_()
            ctx.pinsage_embed_all(hX, hI, hW, Ld, Hd, out=hO)
            plan = ctx.pinsage_last_plan()
            seen.append(plan)
            assert f"feats={feats}" in plan and f"tables={tables}" in plan and "out=ring" in plan, (cap, plan)
            assert torch.equal(hO.view(torch.int16), dev.cpu().view(torch.int16)), f"cap {cap} MiB changed the result"
        ctx.pinsage_set_option("mem_limit_mb", 150)       # below P + H
        with pytest.raises(binding.PinsageError) as e:
            ctx.pinsage_embed_all(hX, hI, hW, Ld, Hd, out=hO)
        assert e.value.status_name == "OOM" and "resident" in str(e.value)
        # device inputs: 210 MiB hold P (98) + the n and a chunks, with `out` as H, only at a smaller chunk
        ctx.pinsage_set_option("mem_limit_mb", 0)
        ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), alpha.to(DEV), Ld, Hd)
        big = int(ctx.pinsage_last_plan().split("chunk=")[1].split()[0])
        ctx.pinsage_set_option("mem_limit_mb", 120)
        small_out = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), alpha.to(DEV), Ld, Hd)
        small = int(ctx.pinsage_last_plan().split("chunk=")[1].split()[0])
        torch.cuda.synchronize()
        assert small < big, (small, big, seen)
        assert torch.equal(small_out.view(torch.int16), dev.view(torch.int16))


def test_hub_split_with_host_tables_matches_device_tables():
    """The hub-split pool picks its hubs from the same sampled rows whether the table lives on the device
    or on the host (one strided copy of the sample), and remaps host tables in their staging slots -- staged
    whole or through a ring: same bits as with device tables."""
    cfg = synth.CONFIGS["cfg4"].scaled(130_000)
    X = synth.make_features(cfg, device=DEV)
    layers, head = synth.make_params(cfg, device=DEV)
    idx, counts = synth.make_graph(cfg, device=DEV)
    with binding.Context(0) as ctx:
        alpha = ctx.pinsage_normalize_counts(counts)
        l0 = ctx.pinsage_launch_count()
        dev = ctx.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=32_768)
        n_dev = ctx.pinsage_launch_count() - l0
        ctx.pinsage_set_option("pool_hubs", 0)
        l0 = ctx.pinsage_launch_count()
        ctx.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=32_768)
        assert n_dev > ctx.pinsage_launch_count() - l0 + 4, "the hub split did not run on this graph"
        ctx.pinsage_set_option("pool_hubs", -1)
        hI, hW = idx.cpu().pin_memory(), alpha.cpu().pin_memory()
        hO = torch.empty((cfg.N, cfg.d_out), dtype=torch.bfloat16).pin_memory()
        for cap, chunk_nodes in ((0, 32_768), (340, 0)):
            ctx.pinsage_set_option("mem_limit_mb", cap)
            hO.zero_()
            ctx.pinsage_embed_all(X, hI, hW, layers, head, out=hO, chunk_nodes=chunk_nodes)
            assert torch.equal(hO.view(torch.int16), dev.cpu().view(torch.int16)), ctx.pinsage_last_plan()
        assert "tables=ring" in ctx.pinsage_last_plan(), ctx.pinsage_last_plan()


@pytest.mark.parametrize("K,chunk_nodes,cap", [(1, 700, 0), (2, 512, 14), (3, 1000, 14), (2, 0, 0)])
def test_host_pipeline_rings_many_chunks_repeated(K, chunk_nodes, cap):
    """The copy / compute pipeline of host buffers under stress: many small chunks (ragged last one), rings
    forced by a small memory cap, every mix of host and device arrays, K = 1 (layer 1 is also the last
    layer: the head follows the S3 that consumed a streamed feature chunk), pageable as well as pinned
    host memory -- ten calls in a row on one context, each bit-identical to the device-buffer result."""
    cfg = dataclasses.replace(synth.CONFIGS["cfg2"].scaled(9_973), K=K)
    X, idx, alpha, layers, head, Ld, Hd = _inputs(cfg)
    with binding.Context(0) as ctx:
        dev = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), alpha.to(DEV), Ld, Hd).cpu()
        ctx.pinsage_set_option("mem_limit_mb", cap)
        ctx.pinsage_set_option("debug_poison", 1)
        hO = torch.empty((cfg.N, cfg.d_out), dtype=X.dtype).pin_memory()
        pinned = (X.pin_memory(), idx.pin_memory(), alpha.pin_memory())
        for it in range(10):
            if it % 5 == 4:      # pageable host memory
                args = (X.clone(), idx.clone(), alpha.clone())
            elif it % 5 == 3:    # device features, host tables
                args = (X.to(DEV), pinned[1], pinned[2])
            elif it % 5 == 2:    # host features, device tables
                args = (pinned[0], idx.to(DEV), alpha.to(DEV))
            else:
                args = pinned
            hO.zero_()
            ctx.pinsage_embed_all(*args, Ld, Hd, out=hO, chunk_nodes=chunk_nodes)
            assert torch.equal(hO.view(torch.int16), dev.view(torch.int16)), (it, ctx.pinsage_last_plan())
        if cap:
            assert "ring" in ctx.pinsage_last_plan().split("out=")[0], ctx.pinsage_last_plan()
