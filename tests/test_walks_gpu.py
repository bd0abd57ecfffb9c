"""Parity of the importance-neighbourhood builder (pinsage_build_neighbourhoods)
with the oracle's simulated walks: integer work, compared bit for bit."""
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


def _both(ctx, row_ptr, col, R, L, T, seed):
    gi, gc = ctx.pinsage_build_neighbourhoods(row_ptr.to(DEV), col.to(DEV), R, L, T, seed)
    oi, oc = O.walk_neighbourhoods(row_ptr.numpy(), col.numpy(), R, L, T, seed)
    np.testing.assert_array_equal(gi.cpu().numpy(), oi)
    np.testing.assert_array_equal(gc.cpu().numpy(), oc)
    return gi, gc


@pytest.mark.parametrize("law", ["uniform", "zipf"])
@pytest.mark.parametrize("R,L,T", [(1, 1, 1), (50, 3, 10), (200, 5, 50), (64, 32, 100), (33, 7, 20),
                                   (2048, 1, 8), (3, 300, 40), (200, 5, 128), (200, 5, 65), (256, 4, 64),
                                   (200, 5, 129), (300, 5, 50)])
def test_walk_neighbourhoods_bit_exact(ctx, law, R, L, T):
    """Random graphs with dead ends, self loops and repeated edges; ragged N (not a multiple of the
    warps per CTA); slot counts from 32 to the 2048 maximum."""
    row_ptr, col = synth.make_csr(3001, 0, 9, law=law, seed=R + L)
    _both(ctx, row_ptr, col, R, L, T, seed=17)


def test_walks_on_a_cycle_and_tiny_graphs(ctx):
    N = 257
    row_ptr = torch.arange(N + 1, dtype=torch.int64)
    col = ((torch.arange(N) + 1) % N).to(torch.int32)
    gi, gc = _both(ctx, row_ptr, col, 9, 5, 8, seed=1)
    assert gc[0].tolist() == [9] * 5 + [0] * 3 and gi[0].tolist() == [1, 2, 3, 4, 5, 0, 0, 0]
    one = torch.zeros(2, dtype=torch.int64)                      # a single isolated node
    gi, gc = _both(ctx, one, torch.zeros(0, dtype=torch.int32), 4, 4, 3, seed=0)
    assert gi.tolist() == [[0, 0, 0]] and gc.tolist() == [[0, 0, 0]]
    assert torch.equal(ctx.pinsage_normalize_counts(gc), torch.zeros((1, 3), device=DEV))


def test_graph_to_embeddings_end_to_end(ctx):
    """CSR graph -> walks -> L1-normalised counts -> K layers + head, all on the GPU, against the
    same chain in the oracle (the tables agree bit for bit, the embeddings within tolerance)."""
    cfg = synth.CONFIGS["cfg2"].scaled(5003)
    row_ptr, col = synth.make_csr(cfg.N, 1, 12, law="zipf", seed=3)
    X = synth.make_features(cfg)
    layers, head = synth.make_params(cfg)
    gi, gc = _both(ctx, row_ptr, col, 100, 4, cfg.T, seed=5)
    w = ctx.pinsage_normalize_counts(gc)
    alpha = O.normalize_counts(gc.cpu().numpy())
    np.testing.assert_array_equal(w.cpu().numpy(), alpha)
    assert ctx.pinsage_validate_graph(gi, w, cfg.N) == -1
    Lf, Hf = params_f64(layers, head)
    ref = O.embed_all(to_f64(X), gi.cpu().numpy(), alpha, Lf, Hf)
    out = ctx.pinsage_embed_all(X.to(DEV), gi, w, [{k: v.to(DEV) for k, v in lp.items()} for lp in layers],
                                {k: v.to(DEV) for k, v in head.items()})
    assert_rows_close(to_f64(out), ref, X.dtype, "graph -> embeddings")


def test_walk_argument_errors(ctx):
    row_ptr, col = synth.make_csr(64, 1, 3, seed=1)
    with pytest.raises(binding.PinsageError) as e:
        ctx.pinsage_build_neighbourhoods(row_ptr.to(DEV), col.to(DEV), 300, 7, 10)
    assert e.value.status_name == "UNSUPPORTED_SHAPE"
    with pytest.raises(binding.PinsageError) as e:
        ctx.pinsage_build_neighbourhoods(row_ptr.to(DEV), col.to(DEV), 0, 7, 10)
    assert e.value.status_name == "INVALID_ARG"
