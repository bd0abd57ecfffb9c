"""Parity of the exact top-K lookup (pinsage_topk) with the oracle.

Index work is compared bit for bit where floating point cannot interfere: with small-integer
embeddings every inner product is exact in fp32, so ids, order and tie-breaks must equal the oracle's.
With Gaussian embeddings the GPU's fp32 accumulation can swap candidates whose fp64 scores differ by
less than its rounding error: there the unique part is compared (everything clearly above the k-th
score is present, nothing clearly below it is) and the returned scores must match."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_1806_01973_b200 import binding
from tests.parity import to_f64

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
DTYPES = [torch.bfloat16, torch.float32]


@pytest.fixture(scope="module")
def ctx():
    c = binding.Context(0)
    yield c
    c.close()


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("nq,N,d,k", [(1, 1, 8, 1), (5, 37, 8, 7), (130, 5000, 64, 50), (300, 70001, 32, 500),
                                      (7, 3000, 256, 1024), (257, 66000, 128, 10)])
def test_topk_exact_on_integer_embeddings(ctx, dtype, nq, N, d, k):
    """Entries in {-2..2}: products and sums are exact, ties are everywhere -> ids must be identical."""
    k = min(k, N)
    g = torch.Generator().manual_seed(nq + N)
    Q = torch.randint(-2, 3, (nq, d), generator=g).to(dtype)
    Z = torch.randint(-2, 3, (N, d), generator=g).to(dtype)
    ref_idx, ref_score = O.topk(to_f64(Q), to_f64(Z), k)
    for cg, fused in ([(1, 1), (0, 1), (0, 0)] if dtype == torch.bfloat16 else [(0, 1)]):
        ctx.pinsage_set_option("gemm_cg", cg)
        ctx.pinsage_set_option("topk_fused", fused)
        try:
            idx, score = ctx.pinsage_topk(Q.to(DEV), Z.to(DEV), k)
        finally:
            ctx.pinsage_set_option("gemm_cg", 0)
            ctx.pinsage_set_option("topk_fused", 1)
        np.testing.assert_array_equal(idx.cpu().numpy(), ref_idx)
        np.testing.assert_array_equal(score.cpu().numpy().astype(np.float64), ref_score)


@pytest.mark.parametrize("k", [100, 1024])
def test_topk_many_blocks_fused_selection(ctx, k):
    """Several candidate blocks, so that most of them go through the GEMM's selection epilogue (only the
    first one or two are scanned from stored scores); integer embeddings -> identical to the oracle, and
    identical to the two-pass form."""
    nq, N, d = 50, 400_003, 32
    g = torch.Generator().manual_seed(11)
    Q = torch.randint(-2, 3, (nq, d), generator=g).to(torch.bfloat16)
    Z = torch.randint(-2, 3, (N, d), generator=g).to(torch.bfloat16)
    ref_idx, ref_score = O.topk(to_f64(Q), to_f64(Z), k)
    for fused in (1, 0):
        ctx.pinsage_set_option("topk_fused", fused)
        try:
            idx, score = ctx.pinsage_topk(Q.to(DEV), Z.to(DEV), k)
        finally:
            ctx.pinsage_set_option("topk_fused", 1)
        np.testing.assert_array_equal(idx.cpu().numpy(), ref_idx)
        np.testing.assert_array_equal(score.cpu().numpy().astype(np.float64), ref_score)


def test_topk_fused_selection_overflow_is_redone(ctx):
    """Adversarial order: candidate scores ascend with the id (ties of 32), so for the "ascending"
    queries EVERY score of every later block beats the running k-th score, the 1024-key buffers of the
    selection epilogue overflow in every block, and those (block, query) pairs must be redone from
    stored scores -- while the "descending" queries of the same blocks keep nothing.  Exact products."""
    N, d, k = 250_000, 16, 500
    t = torch.arange(N) // 32
    Z = torch.zeros((N, d))
    Z[:, 0], Z[:, 1] = (t // 64).float(), (t % 64).float()      # 64 * Z0 + Z1 = t, all exact in bf16
    Q = torch.zeros((6, d))
    Q[0::2, 0], Q[0::2, 1] = 64.0, 1.0                          # score = t: ascending
    Q[1::2, 0], Q[1::2, 1] = -64.0, -1.0                        # score = -t: descending
    Q, Z = Q.to(torch.bfloat16), Z.to(torch.bfloat16)
    ref_idx, ref_score = O.topk(to_f64(Q), to_f64(Z), k)
    assert ref_idx[0, 0] == N - N % 32 - (32 if N % 32 == 0 else 0) or ref_idx[0, 0] >= N - 32
    idx, score = ctx.pinsage_topk(Q.to(DEV), Z.to(DEV), k)
    np.testing.assert_array_equal(idx.cpu().numpy(), ref_idx)
    np.testing.assert_array_equal(score.cpu().numpy().astype(np.float64), ref_score)


@pytest.mark.parametrize("dtype", DTYPES)
def test_topk_on_unit_embeddings(ctx, dtype):
    """Row-normalised Gaussian embeddings (what the path produces), K = 500 as in the paper's evaluation."""
    nq, N, d, k = 200, 100_003, 128, 500
    g = torch.Generator().manual_seed(5)
    Z = torch.randn((N, d), generator=g)
    Z = (Z / Z.norm(dim=1, keepdim=True)).to(dtype)
    Q = Z[torch.randint(0, N, (nq,), generator=g)].clone()
    idx, score = ctx.pinsage_topk(Q.to(DEV), Z.to(DEV), k)
    idx, score = idx.cpu().numpy(), score.cpu().numpy().astype(np.float64)
    S = to_f64(Q) @ to_f64(Z).T
    tol = 2e-6                                           # fp32 accumulation of d = 128 products of size <= 1
    for q in range(nq):
        np.testing.assert_allclose(score[q], S[q, idx[q]], atol=tol)         # returned scores are the scores
        assert len(set(idx[q])) == k
        assert np.all(np.diff(score[q]) <= 0)                                # descending
        kth = np.sort(S[q])[-k]
        assert np.all(S[q, idx[q]] >= kth - tol)                             # nothing clearly below the k-th
        must = np.nonzero(S[q] > kth + tol)[0]
        assert np.isin(must, idx[q]).all()                                   # everything clearly above it
    ref_idx, _ = O.topk(to_f64(Q), to_f64(Z), k)
    assert (idx[:, 0] == ref_idx[:, 0]).all()            # the query itself (score 1) comes first


def test_topk_argument_errors(ctx):
    Q = torch.zeros((4, 16), dtype=torch.bfloat16, device=DEV)
    Z = torch.zeros((100, 16), dtype=torch.bfloat16, device=DEV)
    for k, name in ((0, "INVALID_ARG"), (101, "INVALID_ARG")):
        with pytest.raises(binding.PinsageError) as e:
            ctx.pinsage_topk(Q, Z, k)
        assert e.value.status_name == name
    Zb = torch.zeros((5000, 16), dtype=torch.bfloat16, device=DEV)
    with pytest.raises(binding.PinsageError) as e:
        ctx.pinsage_topk(Q, Zb, 2000)
    assert e.value.status_name == "UNSUPPORTED_SHAPE"


def test_topk_full_size_sampled(ctx):
    """The shape bench.py's `extras` leg times (K = 500 among 5 million candidates; 4 096 queries,
    d = 1024, bf16), in the launch configuration it times (88 candidate blocks, 87 of them through the
    GEMM's selection epilogue).  Sampled queries are checked against fp64 scores computed on the host
    from the stored bf16 values, block of candidates by block of candidates (numpy), then ordered as
    the oracle orders (score descending, id ascending)."""
    free, _ = torch.cuda.mem_get_info(0)
    if free < 30e9:
        pytest.skip("needs 30 GB of free HBM")
    nq, N, d, k = 4096, 5_000_000, 1024, 500
    g = torch.Generator(device=DEV).manual_seed(0)
    Z = torch.empty((N, d), dtype=torch.bfloat16, device=DEV)
    for s in range(0, N, 1 << 20):
        e = min(N, s + (1 << 20))
        z = torch.randn((e - s, d), generator=g, device=DEV)
        Z[s:e] = (z / z.norm(dim=1, keepdim=True)).to(torch.bfloat16)
    Q = Z[torch.randint(0, N, (nq,), generator=g, device=DEV)].clone()
    idx, score = ctx.pinsage_topk(Q, Z, k)
    torch.cuda.synchronize()
    sample = [0, 1, 777, 2048, 4095]
    Qs = to_f64(Q[sample])
    S = np.empty((len(sample), N))
    for s in range(0, N, 500_000):
        e = min(N, s + 500_000)
        S[:, s:e] = Qs @ to_f64(Z[s:e]).T
    idx, score = idx[sample].cpu().numpy(), score[sample].cpu().numpy().astype(np.float64)
    tol = 4e-6                                           # fp32 accumulation of d = 1024 products, |score| <= 1
    for q in range(len(sample)):
        np.testing.assert_allclose(score[q], S[q, idx[q]], atol=tol)
        assert len(set(idx[q])) == k and np.all(np.diff(score[q]) <= 0)
        order = np.lexsort((np.arange(N), -S[q]))[:k + 50]            # the oracle's order
        kth = S[q, order[k - 1]]
        assert np.all(S[q, idx[q]] >= kth - tol)
        must = order[:k][S[q, order[:k]] > kth + tol]
        assert np.isin(must, idx[q]).all()
        assert idx[q, 0] == order[0]


def test_topk_many_queries_in_groups(ctx):
    """More queries than one group (16 384): the groups are independent lookups with the same result."""
    nq, N, d, k = 40_000, 30_011, 16, 20
    g = torch.Generator().manual_seed(9)
    Q = torch.randint(-2, 3, (nq, d), generator=g).to(torch.bfloat16)
    Z = torch.randint(-2, 3, (N, d), generator=g).to(torch.bfloat16)
    idx, score = ctx.pinsage_topk(Q.to(DEV), Z.to(DEV), k)
    pick = np.r_[0, 16383, 16384, 32767, 32768, nq - 1, np.random.default_rng(1).integers(0, nq, 200)]
    ref_idx, ref_score = O.topk(to_f64(Q[pick]), to_f64(Z), k)
    np.testing.assert_array_equal(idx.cpu().numpy()[pick], ref_idx)
    np.testing.assert_array_equal(score.cpu().numpy().astype(np.float64)[pick], ref_score)
