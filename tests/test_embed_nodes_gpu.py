"""Targeted inference (pinsage_embed_nodes = Algorithm 2 on a minibatch) against the
oracle's Algorithm 2 and against the full-graph path, whose rows it must reproduce bit for bit."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_1806_01973_b200 import binding, synth
from tests.parity import assert_rows_close, params_f64, to_f64

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def ctx():
    c = binding.Context(0)
    yield c
    c.close()


def _setup(cfg):
    X = synth.make_features(cfg)
    layers, head = synth.make_params(cfg)
    idx, counts = synth.make_graph(cfg)
    alpha = O.normalize_counts(counts.numpy())
    Ld = [{k: v.to(DEV) for k, v in lp.items()} for lp in layers]
    Hd = {k: v.to(DEV) for k, v in head.items()}
    return X, idx, alpha, layers, head, Ld, Hd


@pytest.mark.parametrize("name,N,targets", [
    ("tiny", 2000, [5, 0, 1999, 5, 17, 1024]),
    ("cfg2", 20011, [0, 20010, 127, 128, 4096, 4095, 7, 7, 7, 12345]),
    ("cfg2", 3000, list(range(0, 3000, 3))),           # a closure that is the whole graph
    ("cfg5", 4001, [4000, 1, 2]),                      # K = 3, T = 100
])
def test_embed_nodes_matches_oracle_and_full_graph(ctx, name, N, targets):
    cfg = synth.CONFIGS[name].scaled(N)
    X, idx, alpha, layers, head, Ld, Hd = _setup(cfg)
    Xd, idd, wd = X.to(DEV), idx.to(DEV), torch.from_numpy(alpha).to(DEV)
    t = torch.tensor(targets, dtype=torch.int32, device=DEV)
    got = ctx.pinsage_embed_nodes(Xd, idd, wd, Ld, Hd, t)
    torch.cuda.synchronize()
    Lf, Hf = params_f64(layers, head)
    Xf = to_f64(X)
    ref = O.minibatch_embed(np.array(targets), lambda ids: Xf[ids],
                            lambda ids: (idx.numpy()[ids], alpha[ids]), Lf, Hf)
    assert_rows_close(to_f64(got), ref, X.dtype, f"embed_nodes {name}")
    full = ctx.pinsage_embed_all(Xd, idd, wd, Ld, Hd)
    bits = torch.int16 if X.dtype == torch.bfloat16 else torch.int32
    assert torch.equal(got.view(bits), full[t.long()].view(bits)), "targeted rows differ from full-graph rows"


def test_embed_nodes_variants_and_errors(ctx):
    cfg = synth.CONFIGS["cfg2"].scaled(5000)
    X, idx, alpha, layers, head, Ld, Hd = _setup(cfg)
    Xd, idd, wd = X.to(DEV), idx.to(DEV), torch.from_numpy(alpha).to(DEV)
    t = torch.tensor([3, 4999, 42], dtype=torch.int32, device=DEV)
    base = ctx.pinsage_embed_nodes(Xd, idd, wd, Ld, Hd, t)
    ctx.pinsage_set_option("linear_pool", 1)           # the linear-pool schedule on the closure
    try:
        lin = ctx.pinsage_embed_nodes(Xd, idd, wd, Ld, Hd, t)
    finally:
        ctx.pinsage_set_option("linear_pool", -1)
    Lf, Hf = params_f64(layers, head)
    Xf = to_f64(X)
    ref = O.minibatch_embed(np.array([3, 4999, 42]), lambda ids: Xf[ids],
                            lambda ids: (idx.numpy()[ids], alpha[ids]), Lf, Hf)
    assert_rows_close(to_f64(lin), ref, X.dtype, "embed_nodes linear pool")
    assert_rows_close(to_f64(base), ref, X.dtype, "embed_nodes")
    bad = torch.tensor([3, 5000], dtype=torch.int32, device=DEV)
    with pytest.raises(binding.PinsageError) as e:
        ctx.pinsage_embed_nodes(Xd, idd, wd, Ld, Hd, bad)
    assert e.value.status_name == "BAD_INDEX"
