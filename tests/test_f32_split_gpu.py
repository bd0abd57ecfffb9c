"""Parity of the fp32 mode on the tensor cores (three-way bf16 operand splitting, option
``f32_split``) with the fp64 oracle, at the fp32 bar of BASELINE.json's
north_star (relative L2 error per row <= 1e-4; the split path is held to 2e-5, a tenth of a
single-bf16 product's error, so a dropped term of the six cannot pass)."""
import dataclasses

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


class _split:
    def __init__(self, ctx, mode):
        self.ctx, self.mode = ctx, mode

    def __enter__(self):
        self.ctx.pinsage_set_option("f32_split", self.mode)

    def __exit__(self, *exc):
        self.ctx.pinsage_set_option("f32_split", -1)


def _rand(shape, seed, scale=1.0):
    g = torch.Generator().manual_seed(seed)
    return torch.randn(shape, generator=g) * scale


@pytest.mark.parametrize("M,k,n_out", [(1, 8, 8), (127, 64, 40), (1000, 256, 256), (4099, 104, 72),
                                       (300, 4360, 2048), (20_000, 512, 1024), (513, 1032, 264)])
def test_dense_split_matches_oracle(ctx, M, k, n_out):
    A = _rand((M, k), 20)
    Wt = _rand((n_out, k), 21, scale=k ** -0.5)
    b = _rand((n_out,), 22, scale=0.1)
    with _split(ctx, 1):
        for bias, relu in [(b, True), (None, False)]:
            got = ctx.pinsage_dense(A.to(DEV), Wt.to(DEV), None if bias is None else bias.to(DEV), relu)
            ref = O.dense(to_f64(A), to_f64(Wt), None if bias is None else to_f64(bias), relu)
            err = np.abs(to_f64(got) - ref).max(axis=1)
            scale = np.abs(ref).max(axis=1) + 1e-3
            assert (err / scale).max() < 2e-5, (relu, (err / scale).max())


@pytest.mark.parametrize("M,d_in,m,d", [(1, 8, 8, 8), (130, 64, 64, 64), (1000, 256, 256, 256),
                                        (515, 512, 512, 512), (300, 2048, 1024, 1024), (257, 24, 40, 16),
                                        (5000, 264, 120, 520), (70_001, 128, 128, 128)])
def test_combine_split_matches_oracle(ctx, M, d_in, m, d):
    H = _rand((M, d_in), 30)
    n = _rand((M, m), 31).abs()
    W = _rand((d, d_in + m), 32, scale=(d_in + m) ** -0.5)
    w = _rand((d,), 33, scale=0.01)
    ref = O.combine(to_f64(H), to_f64(n), to_f64(W), to_f64(w))
    with _split(ctx, 1):
        got = ctx.pinsage_combine(H.to(DEV), n.to(DEV), W.to(DEV), w.to(DEV))
    assert_rows_close(to_f64(got), ref, torch.float32, "split combine", tol=2e-5)
    nrm = np.linalg.norm(to_f64(got), axis=1)
    assert np.all((np.abs(nrm - 1) < 1e-5) | (nrm == 0))


def test_split_is_exact_on_small_integers(ctx):
    """Entries in {-3..3}: the second and third planes are zero and every sum is exact in fp32, so the
    split path, the SIMT path and the oracle agree bit for bit (a mis-ordered plane would show)."""
    M, k, n_out = 700, 96, 80
    g = torch.Generator().manual_seed(3)
    A = torch.randint(-3, 4, (M, k), generator=g).float()
    Wt = torch.randint(-3, 4, (n_out, k), generator=g).float()
    ref = O.dense(to_f64(A), to_f64(Wt), None, False)
    for mode in (0, 1):
        with _split(ctx, mode):
            got = ctx.pinsage_dense(A.to(DEV), Wt.to(DEV), None, False)
        np.testing.assert_array_equal(to_f64(got), ref)


def test_split_carries_every_term(ctx):
    """x = 1 + 2^-9 + 2^-17 has the planes (1, 2^-9, 2^-17); x^2 = 1 + 2^-8 + 2^-16 + 2^-18 + ... and each
    of the six kept terms is worth at least 2^-18, eight times the bound below: a dropped, doubled or
    mis-paired term fails.  One non-zero product per output isolates the splitting from the summing."""
    x = 1.0 + 2.0 ** -9 + 2.0 ** -17
    assert float(np.float32(x)) == x
    A = torch.zeros((256, 8))
    Wt = torch.zeros((8, 8))
    A[:, 0] = x
    Wt[:, 0] = x
    with _split(ctx, 1):
        got = to_f64(ctx.pinsage_dense(A.to(DEV), Wt.to(DEV), None, False))
    assert np.abs(got - x * x).max() < 2.0 ** -21


def test_combine_split_zero_rows_stay_zero(ctx):
    M, d = 1300, 64
    H = _rand((M, d), 34).abs()
    n = _rand((M, d), 35).abs()
    W = -_rand((d, 2 * d), 36).abs()
    with _split(ctx, 1):
        got = ctx.pinsage_combine(H.to(DEV), n.to(DEV), W.to(DEV), torch.zeros(d).to(DEV))
    assert torch.equal(got.cpu(), torch.zeros((M, d)))


@pytest.mark.parametrize("name,N,chunk", [("tiny", 2000, 0), ("cfg2", 20_011, 4096), ("cfg3", 3000, 2048)])
def test_whole_path_fp32_split(ctx, name, N, chunk):
    """The whole path in fp32 with every GEMM on the tensor cores, every row, <= 1e-4 (north_star's
    fp32 bar), layer by layer and in one call; the automatic choice gives the same result."""
    cfg = dataclasses.replace(synth.CONFIGS[name].scaled(N), dtype="f32")
    X = synth.make_features(cfg)
    layers, head = synth.make_params(cfg)
    idx, counts = synth.make_graph(cfg)
    alpha = O.normalize_counts(counts.numpy())
    Lf, Hf = params_f64(layers, head)
    ref_out, ref_hidden = O.embed_all(to_f64(X), idx.numpy(), alpha, Lf, Hf, return_hidden=True)
    Ld = [{k: v.to(DEV) for k, v in lp.items()} for lp in layers]
    Hd = {k: v.to(DEV) for k, v in head.items()}
    w = torch.from_numpy(alpha).to(DEV)
    ctx.pinsage_set_option("linear_pool", 0)
    try:
        with _split(ctx, 1):
            H = X.to(DEV)
            for k, lp in enumerate(Ld):
                H = ctx.pinsage_layer(H, idx.to(DEV), w, lp)
                assert_rows_close(to_f64(H), ref_hidden[k], torch.float32, f"{name} fp32 split H_{k + 1}")
            out = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), w, Ld, Hd, chunk_nodes=chunk)
            assert_rows_close(to_f64(out), ref_out, torch.float32, f"{name} fp32 split embed_all")
        auto = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), w, Ld, Hd, chunk_nodes=chunk)
        assert_rows_close(to_f64(auto), ref_out, torch.float32, f"{name} fp32 auto embed_all")
    finally:
        ctx.pinsage_set_option("linear_pool", -1)


def test_topk_fp32_split(ctx):
    """fp32 embeddings, scores from the split GEMM: same acceptance as the bf16 lookup (unique part
    identical, returned scores are the scores), at an fp32-accurate tolerance."""
    nq, N, d, k = 200, 100_003, 128, 500
    g = torch.Generator().manual_seed(5)
    Z = torch.randn((N, d), generator=g)
    Z = Z / Z.norm(dim=1, keepdim=True)
    Q = Z[torch.randint(0, N, (nq,), generator=g)].clone()
    with _split(ctx, 1):
        idx, score = ctx.pinsage_topk(Q.to(DEV), Z.to(DEV), k)
    idx, score = idx.cpu().numpy(), score.cpu().numpy().astype(np.float64)
    S = to_f64(Q) @ to_f64(Z).T
    tol = 1e-6
    for q in range(nq):
        np.testing.assert_allclose(score[q], S[q, idx[q]], atol=tol)
        assert len(set(idx[q])) == k and np.all(np.diff(score[q]) <= 0)
        kth = np.sort(S[q])[-k]
        assert np.all(S[q, idx[q]] >= kth - tol)
        assert np.isin(np.nonzero(S[q] > kth + tol)[0], idx[q]).all()
    # integer embeddings: exact products, ids identical to the oracle's (ties included)
    Qi = torch.randint(-2, 3, (130, 64), generator=g).float()
    Zi = torch.randint(-2, 3, (70_001, 64), generator=g).float()
    with _split(ctx, 1):
        idx, score = ctx.pinsage_topk(Qi.to(DEV), Zi.to(DEV), 50)
    ref_idx, ref_score = O.topk(to_f64(Qi), to_f64(Zi), 50)
    np.testing.assert_array_equal(idx.cpu().numpy(), ref_idx)
    np.testing.assert_array_equal(score.cpu().numpy().astype(np.float64), ref_score)


def test_split_forced_on_uncovered_gemm_fails_loudly(ctx):
    """f32_split = 1 is a demand, not a hint: the one GEMM the split path does not take (the addend
    of the linear-pool schedule) is an error, while the automatic choice falls back to the SIMT kernel."""
    cfg = dataclasses.replace(synth.CONFIGS["tiny"], m_proj=128)          # m = 128 > d = 64
    X = synth.make_features(cfg)
    layers, _ = synth.make_params(cfg)
    idx, counts = synth.make_graph(cfg)
    alpha = O.normalize_counts(counts.numpy())
    lp = {k: v.to(DEV) for k, v in layers[0].items()}
    w = torch.from_numpy(alpha).to(DEV)
    ctx.pinsage_set_option("linear_pool", 1)
    try:
        with _split(ctx, 1):
            with pytest.raises(binding.PinsageError) as e:
                ctx.pinsage_layer(X.to(DEV), idx.to(DEV), w, lp)
            assert e.value.status_name == "UNSUPPORTED_SHAPE"
        H = ctx.pinsage_layer(X.to(DEV), idx.to(DEV), w, lp)
        ref = O.layer_layerwise(to_f64(X), idx.numpy(), alpha, params_f64(layers)[0][0])
        assert_rows_close(to_f64(H), ref, torch.float32, "linear pool, automatic fp32 GEMM choice")
    finally:
        ctx.pinsage_set_option("linear_pool", -1)
    with pytest.raises(binding.PinsageError):
        ctx.pinsage_set_option("f32_split", 2)
