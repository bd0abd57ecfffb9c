"""Parity of the hub-split pool (option ``pool_hubs``; hubs.cu): on a power-law graph the entries of the
neighbour lists that point at the few hundred most listed nodes are not gathered; their term enters S3 as
a third K segment on the tensor cores.  Same function as Algorithm 1 lines 1-2 in real arithmetic;
checked against the fp64 oracle on sampled destinations (Algorithm 2 on their K-hop closure) and against
the plain pool on every row."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_1806_01973_b200 import binding, synth
from tests.parity import assert_rows_close, params_f64, row_errors, to_f64

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def ctx():
    """The split is automatic by default (pool_hubs = -1); these tests start from "off" and switch it on
    explicitly, so that each has the plain pool to compare with."""
    c = binding.Context(0)
    c.pinsage_set_option("pool_hubs", 0)
    yield c
    c.close()


def _setup(cfg):
    X = synth.make_features(cfg, device=DEV)
    layers, head = synth.make_params(cfg, device=DEV)
    idx, counts = synth.make_graph(cfg, device=DEV)
    return X, layers, head, idx, counts


def _oracle_rows(X, idx, alpha, layers, head, rows):
    Lf, Hf = params_f64([{k: v.cpu() for k, v in lp.items()} for lp in layers], {k: v.cpu() for k, v in head.items()})

    def fetch_x(ids):
        t = torch.from_numpy(np.asarray(ids, dtype=np.int64)).to(DEV)
        return X[t].to(torch.float64).cpu().numpy()

    def fetch_nbr(ids):
        t = torch.from_numpy(np.asarray(ids, dtype=np.int64)).to(DEV)
        return idx[t].cpu().numpy(), alpha[t].cpu().numpy()

    return O.minibatch_embed(rows, fetch_x, fetch_nbr, Lf, Hf)


@pytest.mark.parametrize("hubs", [256, 64, -1])
def test_power_law_graph_with_hub_split_pool(ctx, hubs):
    cfg = synth.CONFIGS["cfg4"].scaled(150_000)
    X, layers, head, idx, counts = _setup(cfg)
    alpha = ctx.pinsage_normalize_counts(counts)
    plain = ctx.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=65536)
    l0 = ctx.pinsage_launch_count()
    ctx.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=65536)
    plain_launches = ctx.pinsage_launch_count() - l0
    ctx.pinsage_set_option("pool_hubs", hubs)
    try:
        l0 = ctx.pinsage_launch_count()
        out = ctx.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=65536)
        hub_launches = ctx.pinsage_launch_count() - l0
    finally:
        ctx.pinsage_set_option("pool_hubs", 0)
    torch.cuda.synchronize()
    assert hub_launches > plain_launches + 4, "the hub path did not run"
    # the lists really are dominated by a few ids (what the path is for)
    share = float((idx < 256).float().mean())
    assert share > 0.3, share
    rows = np.concatenate([[0, 1, 255, 256, cfg.N - 1], np.random.default_rng(3).integers(0, cfg.N, 123)])
    ref = _oracle_rows(X, idx, alpha, layers, head, rows)
    t = torch.from_numpy(rows).to(DEV)
    assert_rows_close(to_f64(out[t]), ref, torch.bfloat16, f"hub-split pool H={hubs} vs oracle")
    assert_rows_close(to_f64(plain[t]), ref, torch.bfloat16, "plain pool vs oracle")
    rel, cos = row_errors(to_f64(out), to_f64(plain))
    assert rel.max() <= 1e-2 and cos.min() >= 0.999, (rel.max(), cos.min())


def test_uniform_graph_finds_no_hubs(ctx):
    """No id reaches the candidate threshold on a uniform graph: forced on, the remapped table equals the
    original and the hub GEMM adds zero -> bit-identical output; automatic -> the path is not taken."""
    cfg = synth.CONFIGS["cfg2"].scaled(120_000)
    X, layers, head, idx, counts = _setup(cfg)
    alpha = ctx.pinsage_normalize_counts(counts)
    plain = ctx.pinsage_embed_all(X, idx, alpha, layers, head)
    l0 = ctx.pinsage_launch_count()
    ctx.pinsage_embed_all(X, idx, alpha, layers, head)
    plain_launches = ctx.pinsage_launch_count() - l0
    for hubs in (128, -1):
        ctx.pinsage_set_option("pool_hubs", hubs)
        try:
            l0 = ctx.pinsage_launch_count()
            out = ctx.pinsage_embed_all(X, idx, alpha, layers, head)
            n = ctx.pinsage_launch_count() - l0
        finally:
            ctx.pinsage_set_option("pool_hubs", 0)
        assert torch.equal(out.view(torch.int16), plain.view(torch.int16))
        if hubs == -1:
            assert n == plain_launches + 3          # histogram, candidates, selection -- and nothing else
        else:
            assert n > plain_launches + 4


def test_pool_hubs_option_values(ctx):
    for bad in (1, 63, 576, -2):
        with pytest.raises(binding.PinsageError):
            ctx.pinsage_set_option("pool_hubs", bad)


@pytest.mark.parametrize("d0,hidden,T,hubs,chunk", [(264, 264, 37, 64, 30_000), (136, 520, 50, 512, 0),
                                                     (512, 128, 64, 128, 50_048)])
def test_hub_split_pool_odd_shapes(ctx, d0, hidden, T, hubs, chunk):
    """Widths that are not multiples of 64 (ragged K blocks in all three S3 segments, inexact row
    chunks in the gather), a row narrow enough for two nodes per warp (hidden = 128: the separate
    matrix kernel), T beyond one 32-entry batch, ragged driver chunks."""
    import dataclasses
    cfg = dataclasses.replace(synth.CONFIGS["cfg4"].scaled(130_003), d0=d0, hidden=hidden, g1=hidden, d_out=64, T=T)
    X, layers, head, idx, counts = _setup(cfg)
    alpha = ctx.pinsage_normalize_counts(counts)
    plain = ctx.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=chunk)
    ctx.pinsage_set_option("pool_hubs", hubs)
    try:
        out = ctx.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=chunk)
    finally:
        ctx.pinsage_set_option("pool_hubs", 0)
    torch.cuda.synchronize()
    rows = np.concatenate([[0, 1, hubs - 1, hubs, cfg.N - 1], np.random.default_rng(5).integers(0, cfg.N, 59)])
    ref = _oracle_rows(X, idx, alpha, layers, head, rows)
    t = torch.from_numpy(rows).to(DEV)
    assert_rows_close(to_f64(out[t]), ref, torch.bfloat16, "hub-split pool vs oracle")
    rel, cos = row_errors(to_f64(out), to_f64(plain))
    assert rel.max() <= 1e-2 and cos.min() >= 0.999, (rel.max(), cos.min())
    assert not torch.equal(out.view(torch.int16), plain.view(torch.int16)), "the hub path did not run"


def test_default_context_takes_the_split_and_all_paths_agree_bit_for_bit():
    """A fresh context (pool_hubs = -1, the default) on the power-law graph: the split is taken, the result is
    the same run to run (no atomics: the hub weights are summed in table order), and the one-call path, the
    layer-by-layer path and targeted inference (pinsage_embed_nodes, which picks the hubs from the whole
    graph's table and remaps only its sub-tables) agree bit for bit -- with lists that name a hub several
    times (reading A7) and with the hub weights summed across 32-entry batches (T = 50)."""
    cfg = synth.CONFIGS["cfg4"].scaled(140_000)
    X, layers, head, idx, counts = _setup(cfg)
    idx[7, 5] = idx[7, 0]            # node 7 names its first (hub) neighbour three times, across two batches
    idx[7, 40] = idx[7, 0]
    idx[9, :] = idx[9, 0]            # node 9 names one hub 50 times
    with binding.Context(0) as c:
        alpha = c.pinsage_normalize_counts(counts)
        l0 = c.pinsage_launch_count()
        a = c.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=40_000)
        n_split = c.pinsage_launch_count() - l0
        b = c.pinsage_embed_all(X, idx, alpha, layers, head)            # automatic chunk
        torch.cuda.synchronize()
        assert torch.equal(a.view(torch.int16), b.view(torch.int16))
        for _ in range(3):
            again = c.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=40_000)
            assert torch.equal(a.view(torch.int16), again.view(torch.int16)), "not bit-reproducible"
        H = X
        for lp in layers:
            H = c.pinsage_layer(H, idx, alpha, lp)
        by_layer = c.pinsage_head(H, head)
        assert torch.equal(a.view(torch.int16), by_layer.view(torch.int16)), "layer-by-layer path differs"
        rows = np.concatenate([[0, 7, 9, 127, 128, cfg.N - 1], np.random.default_rng(11).integers(0, cfg.N, 200)])
        t = torch.from_numpy(rows).to(DEV).to(torch.int32)
        sub = c.pinsage_embed_nodes(X, idx, alpha, layers, head, t)
        torch.cuda.synchronize()
        assert torch.equal(sub.view(torch.int16), a[t.long()].view(torch.int16)), "targeted rows differ"
        ref = _oracle_rows(X, idx, alpha, layers, head, rows[:70])
        assert_rows_close(to_f64(a[t.long()[:70]]), ref, torch.bfloat16, "default (hub-split) path vs oracle")
        c.pinsage_set_option("pool_hubs", 0)
        l0 = c.pinsage_launch_count()
        plain = c.pinsage_embed_all(X, idx, alpha, layers, head, chunk_nodes=40_000)
        n_plain = c.pinsage_launch_count() - l0
        assert n_split > n_plain + 4, "the default context did not take the hub-split pool"
        assert not torch.equal(plain.view(torch.int16), a.view(torch.int16))
