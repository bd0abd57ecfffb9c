"""Parity tests proper: the CUDA path (through the C-ABI binding) against the fp64 CPU oracle,
element by element on the same seeded inputs.  Integer / index work is bit-exact; floating
point is within north_star's tolerances (tests/parity.py)."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_1806_01973_b200 import binding, synth
from tests.parity import assert_rows_close, params_f64, row_errors, to_f64

pytestmark = pytest.mark.gpu

DEV = "cuda:0"
DTYPES = [torch.bfloat16, torch.float32]


@pytest.fixture(scope="module")
def ctx():
    c = binding.Context(0)
    yield c
    c.close()


def _rand(shape, dtype, seed, scale=1.0):
    g = torch.Generator().manual_seed(seed)
    return (torch.randn(shape, generator=g) * scale).to(dtype)


def _graph(N, T, seed, n_src=None):
    g = torch.Generator().manual_seed(seed)
    idx = torch.randint(0, n_src or N, (N, T), generator=g, dtype=torch.int32)
    counts = torch.randint(1, 101, (N, T), generator=g, dtype=torch.int32)
    return idx, counts


def _both_impls(ctx, dtype):
    """(gemm_impl, gemm_cg): bf16 runs through the tcgen05 kernel with single-CTA tiles, with CTA
    pairs (cta_group::2) and through the SIMT reference kernels; fp32 takes the automatic choice here
    (SIMT at these sizes; the split tensor-core path has its own file, test_f32_split_gpu.py)."""
    return [(0, 1), (0, 2), (1, 0)] if dtype == torch.bfloat16 else [(0, 0)]


class _impl:
    def __init__(self, ctx, impl, cg):
        self.ctx, self.impl, self.cg = ctx, impl, cg

    def __enter__(self):
        self.ctx.pinsage_set_option("gemm_impl", self.impl)
        self.ctx.pinsage_set_option("gemm_cg", self.cg)

    def __exit__(self, *exc):
        self.ctx.pinsage_set_option("gemm_impl", 0)
        self.ctx.pinsage_set_option("gemm_cg", 0)


# ------------------------------------------------------------------ helpers of the path
def test_normalize_counts_bit_exact(ctx):
    for N, T in [(1, 1), (1000, 50), (777, 100), (33, 7)]:
        _, counts = _graph(N, T, 5)
        got = ctx.pinsage_normalize_counts(counts.to(DEV)).cpu().numpy()
        np.testing.assert_array_equal(got, O.normalize_counts(counts.numpy()))


def test_validate_graph(ctx):
    idx, counts = _graph(500, 20, 6)
    w = torch.from_numpy(O.normalize_counts(counts.numpy()))
    assert ctx.pinsage_validate_graph(idx.to(DEV), w.to(DEV), 500) == -1
    bad = idx.clone()
    bad[123, 7] = 500
    bad[400, 0] = -1
    with pytest.raises(binding.PinsageError) as e:
        ctx.pinsage_validate_graph(bad.to(DEV), w.to(DEV), 500)
    assert e.value.status_name == "BAD_INDEX" and ctx.first_bad == 123 * 20 + 7
    wb = w.clone()
    wb[9, 3] = float("nan")
    with pytest.raises(binding.PinsageError):
        ctx.pinsage_validate_graph(idx.to(DEV), wb.to(DEV), 500)
    assert ctx.first_bad == 9 * 20 + 3


# ------------------------------------------------------------------ S2 pool
def _encode_rows(n, m, dtype):
    """Row i holds the base-128 digits of i in columns 0..3 (exact in bf16), zeros elsewhere."""
    i = torch.arange(n, dtype=torch.int64)
    P = torch.zeros((n, m), dtype=torch.float32)
    for c in range(4):
        P[:, c] = ((i >> (7 * c)) & 127).to(torch.float32)
    return P.to(dtype)


@pytest.mark.parametrize("dtype", DTYPES)
def test_pool_index_handling_bit_exact(ctx, dtype):
    """Exact arithmetic gather: T=1 decodes to the id; T=4 with alpha=1/4 sums exactly."""
    n_src, m, n_dst = 300_000, 16, 5000
    P = _encode_rows(n_src, m, dtype).to(DEV)
    g = torch.Generator().manual_seed(7)
    idx = torch.randint(0, n_src, (n_dst, 1), generator=g, dtype=torch.int32)
    idx[0, 0], idx[1, 0], idx[2, 0] = 0, n_src - 1, 2    # first row, last row
    w = torch.ones((n_dst, 1), dtype=torch.float32)
    out = ctx.pinsage_pool(P, idx.to(DEV), w.to(DEV)).cpu().to(torch.float32)
    dec = sum(out[:, c].to(torch.int64) << (7 * c) for c in range(4))
    assert torch.equal(dec, idx[:, 0].to(torch.int64))
    assert torch.equal(out[:, 4:], torch.zeros_like(out[:, 4:]))
    # T = 4, alpha = 0.25, with self / repeated ids: sums of <= 4*127 quarter-integers are exact
    idx4 = torch.randint(0, n_src, (n_dst, 4), generator=g, dtype=torch.int32)
    idx4[5] = idx4[5, 0]                                    # repeated ids are legal (A7)
    w4 = torch.full((n_dst, 4), 0.25, dtype=torch.float32)
    out4 = ctx.pinsage_pool(P, idx4.to(DEV), w4.to(DEV)).cpu()
    ref = O.pool(to_f64(P), idx4.numpy(), w4.numpy())
    exp = torch.from_numpy(ref).to(dtype)                   # exact values; bf16 rounds them once
    assert torch.equal(out4.view(torch.int16 if dtype == torch.bfloat16 else torch.int32),
                       exp.view(torch.int16 if dtype == torch.bfloat16 else torch.int32))


def test_pool_large_ids_and_64bit_offsets(ctx):
    """ids > 2^24 (a float-cast id would break) and a P larger than 2^32 bytes (32-bit
    offset arithmetic would break): n_src = 17M rows of 128 bf16 = 4.35 GB."""
    n_src, m, n_dst = 17_000_000, 128, 4096
    P = torch.zeros((n_src, m), dtype=torch.bfloat16, device=DEV)
    i = torch.arange(n_src, dtype=torch.int64, device=DEV)
    for c in range(4):
        P[:, c] = ((i >> (7 * c)) & 127).to(torch.bfloat16)
    del i
    g = torch.Generator().manual_seed(8)
    idx = torch.randint(0, n_src, (n_dst, 1), generator=g, dtype=torch.int32)
    idx[0, 0], idx[1, 0], idx[2, 0] = n_src - 1, (1 << 24) + 1, (1 << 32) // (m * 2) + 3
    idx[3, 0], idx[4, 0] = (1 << 32) // (m * 2) - 1, (1 << 32) // (m * 2)
    w = torch.ones((n_dst, 1), dtype=torch.float32)
    out = ctx.pinsage_pool(P, idx.to(DEV), w.to(DEV)).cpu().to(torch.float32)
    dec = sum(out[:, c].to(torch.int64) << (7 * c) for c in range(4))
    assert torch.equal(dec, idx[:, 0].to(torch.int64))


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("n_dst,n_src,T,m", [
    (1, 1, 1, 8), (257, 300, 3, 8), (1000, 1000, 10, 64), (3001, 2000, 50, 256),
    (515, 4000, 100, 256), (300, 900, 50, 512), (130, 500, 20, 1024), (77, 300, 7, 2048),
    (999, 999, 33, 24), (640, 640, 50, 192), (200, 200, 5, 320), (50, 3000, 1024, 64),
])
def test_pool_matches_oracle(ctx, dtype, n_dst, n_src, T, m):
    if dtype == torch.float32 and m > 1024:
        pytest.skip("fp32 rows above 4 KB are outside the compiled set")
    P = _rand((n_src, m), dtype, 10 + m)
    idx, counts = _graph(n_dst, T, 11 + T, n_src=n_src)
    w = O.normalize_counts(counts.numpy())
    got = ctx.pinsage_pool(P.to(DEV), idx.to(DEV), torch.from_numpy(w).to(DEV))
    ref = O.pool(to_f64(P), idx.numpy(), w)
    # one RNE rounding of an fp32 sum: unit roundoff u = 2^-8 per element in bf16 (8-bit
    # significand), so a row's relative L2 error is at most u = 3.91e-3 (+ fp32 sum error)
    assert_rows_close(to_f64(got), ref, dtype, f"pool {dtype} T={T} m={m}",
                      tol=4e-3 if dtype == torch.bfloat16 else 2e-6)


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("slab", [32, 64, 128])
@pytest.mark.parametrize("n_dst,n_src,T,m", [(3001, 2000, 50, 256), (515, 4000, 100, 256),
                                             (77, 300, 7, 512), (1, 9, 1, 128), (640, 640, 33, 192)])
def test_pool_column_slab_mode_is_bit_identical(ctx, dtype, slab, n_dst, n_src, T, m):
    """The L2-resident column-slab schedule (option pool_slab) keeps the per-element summation
    order t = 0..T-1, so it must reproduce the whole-row kernel bit for bit (and hence the oracle
    within the same tolerance)."""
    P = _rand((n_src, m), dtype, 40 + m).to(DEV)
    idx, counts = _graph(n_dst, T, 41 + T, n_src=n_src)
    w = torch.from_numpy(O.normalize_counts(counts.numpy())).to(DEV)
    bits = torch.int16 if dtype == torch.bfloat16 else torch.int32
    try:
        ctx.pinsage_set_option("pool_slab", 0)
        whole = ctx.pinsage_pool(P, idx.to(DEV), w)
        ctx.pinsage_set_option("pool_slab", slab)
        slabbed = ctx.pinsage_pool(P, idx.to(DEV), w)
    finally:
        ctx.pinsage_set_option("pool_slab", -1)
    assert torch.equal(whole.view(bits), slabbed.view(bits))
    ref = O.pool(to_f64(P), idx.numpy(), w.cpu().numpy())
    assert_rows_close(to_f64(slabbed), ref, dtype, f"slab pool {slab}",
                      tol=4e-3 if dtype == torch.bfloat16 else 2e-6)


def test_pool_is_deterministic_and_order_invariant_within_tolerance(ctx):
    P = _rand((5000, 256), torch.bfloat16, 12).to(DEV)
    idx, counts = _graph(4000, 50, 13, n_src=5000)
    w = torch.from_numpy(O.normalize_counts(counts.numpy()))
    a = ctx.pinsage_pool(P, idx.to(DEV), w.to(DEV))
    b = ctx.pinsage_pool(P, idx.to(DEV), w.to(DEV))
    assert torch.equal(a.view(torch.int16), b.view(torch.int16))
    perm = torch.stack([torch.randperm(50) for _ in range(4000)])
    c = ctx.pinsage_pool(P, torch.gather(idx, 1, perm).to(DEV), torch.gather(w, 1, perm).to(DEV))
    rel, _ = row_errors(to_f64(c), to_f64(a))
    assert rel.max() < 5e-3


# ------------------------------------------------------------------ S1 / S4 / S5 dense
DENSE_SHAPES = [(1, 8, 8), (130, 64, 64), (1000, 256, 256), (777, 256, 128), (300, 2048, 1024),
                (515, 512, 512), (129, 1024, 1024), (257, 24, 40), (64, 512, 256), (4100, 128, 256)]


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("M,k,n_out", DENSE_SHAPES)
def test_dense_matches_oracle(ctx, dtype, M, k, n_out):
    A = _rand((M, k), dtype, 20)
    Wt = _rand((n_out, k), dtype, 21, scale=k ** -0.5)
    b = _rand((n_out,), torch.float32, 22, scale=0.1)
    ran = 0
    for impl, cg in _both_impls(ctx, dtype):
        with _impl(ctx, impl, cg):
            for bias, relu in [(b, True), (None, False), (b, False)]:
                try:
                    got = ctx.pinsage_dense(A.to(DEV), Wt.to(DEV),
                                            None if bias is None else bias.to(DEV), relu)
                except binding.PinsageError as e:
                    if e.status_name == "UNSUPPORTED_SHAPE" and impl == 0:
                        break                      # e.g. CTA pairs need M > 128 and N % 16 == 0
                    raise
                ran += 1
                ref = O.dense(to_f64(A), to_f64(Wt), None if bias is None else to_f64(bias), relu)
                # absolute comparison per row against the row scale (ReLU rows can be tiny)
                err = np.abs(to_f64(got) - ref).max(axis=1)
                scale = np.abs(ref).max(axis=1) + 1e-3
                tol = 8e-3 if dtype == torch.bfloat16 else 2e-5
                assert (err / scale).max() < tol, (impl, cg, relu, (err / scale).max())
    assert ran >= 3


@pytest.mark.parametrize("M,k,n_out,cg", [(40_000, 512, 512, 2), (40_000, 512, 256, 0), (38_001, 256, 256, 1),
                                          (50_000, 136, 264, 1), (50_000, 520, 208, 2)])
def test_dense_stationary_weights_many_tiles(ctx, M, k, n_out, cg):
    """Short K with more tiles than CTAs: the CTA's share of the weight slab stays in shared memory for the
    whole launch and only the activations stream (diagnostic key gemm_bres; ragged K blocks, ragged slabs
    and ragged last row tiles included).  Against the oracle on every row, and bit-identical to the
    streaming form (the MMAs run in the same order)."""
    A = _rand((M, k), torch.bfloat16, 23)
    Wt = _rand((n_out, k), torch.bfloat16, 24, scale=k ** -0.5)
    b = _rand((n_out,), torch.float32, 25, scale=0.1)
    ref = O.dense(to_f64(A), to_f64(Wt), to_f64(b), True)
    outs = []
    with _impl(ctx, 0, cg):
        for bres in (1, 0):
            ctx.pinsage_set_option("gemm_bres", bres)
            try:
                outs.append(ctx.pinsage_dense(A.to(DEV), Wt.to(DEV), b.to(DEV), True))
            finally:
                ctx.pinsage_set_option("gemm_bres", 1)
    err = np.abs(to_f64(outs[0]) - ref).max(axis=1) / (np.abs(ref).max(axis=1) + 1e-3)
    assert err.max() < 8e-3, err.max()
    assert torch.equal(outs[0].view(torch.int16), outs[1].view(torch.int16))


@pytest.mark.parametrize("M,d,g1,d_out", [(1, 64, 64, 32), (130, 256, 256, 128), (20_011, 256, 256, 128),
                                          (50_000, 256, 256, 256), (3_001, 136, 72, 40), (100_000, 512, 256, 256),
                                          (777, 1024, 128, 8), (40_000, 264, 200, 136),
                                          (256 * 74 + 100, 256, 256, 256), (256 * 74 * 3 + 129, 128, 256, 64),
                                          (300_000, 256, 256, 256)])
def test_head_one_launch_matches_oracle_and_two_launches(ctx, M, d, g1, d_out):
    """S4 -> S5 in one launch (gemm_head.cu; the intermediate a lives in an L2-resident scratch, two row
    tiles software-pipelined over the two TMEM accumulators): against the oracle's head on every row, and
    bit-identical to the two-launch form (same K order, same roundings) -- in both of its forms: CTA pairs
    with the weights stationary in shared memory (taken from ~19 000 rows where the weights fit) and single
    CTAs that stream them.  One tile, a trailing single tile of a pair, a last pair tile whose second half is
    empty, many tiles per CTA, ragged K blocks and ragged widths."""
    h = _rand((M, d), torch.bfloat16, 60)
    hp = {"G1": _rand((g1, d), torch.bfloat16, 61, scale=d ** -0.5), "g": _rand((g1,), torch.float32, 62, scale=0.05),
          "G2": _rand((d_out, g1), torch.bfloat16, 63, scale=g1 ** -0.5)}
    Hd = {k: v.to(DEV) for k, v in hp.items()}
    hd = h.to(DEV)
    outs, counts = {}, {}
    try:
        for mode in (1, 2, 0):
            ctx.pinsage_set_option("head_fused", mode)
            l0 = ctx.pinsage_launch_count()
            outs[mode] = ctx.pinsage_head(hd, Hd)
            counts[mode] = ctx.pinsage_launch_count() - l0
    finally:
        ctx.pinsage_set_option("head_fused", 1)
    torch.cuda.synchronize()
    assert counts == {1: 1, 2: 1, 0: 2}, counts
    assert torch.equal(outs[1].view(torch.int16), outs[0].view(torch.int16))
    assert torch.equal(outs[2].view(torch.int16), outs[0].view(torch.int16))
    ref = O.head(to_f64(h), {k: to_f64(v) for k, v in hp.items()})
    err = np.abs(to_f64(outs[1]) - ref).max(axis=1) / (np.abs(ref).max(axis=1) + 1e-3)
    assert err.max() < 1.2e-2, err.max()          # two bf16 roundings (a, out) of O(1) values, per element


# ------------------------------------------------------------------ S3 combine
@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("M,d_in,m,d", [(1, 8, 8, 8), (130, 64, 64, 64), (1000, 256, 256, 256),
                                        (515, 512, 512, 512), (300, 2048, 1024, 1024),
                                        (257, 24, 40, 16), (129, 256, 512, 128),
                                        (200, 1024, 1024, 1024), (5000, 256, 256, 768),
                                        (1500, 512, 512, 2048)])
def test_combine_matches_oracle(ctx, dtype, M, d_in, m, d):
    H = _rand((M, d_in), dtype, 30)
    n = _rand((M, m), dtype, 31).abs()
    W = _rand((d, d_in + m), dtype, 32, scale=(d_in + m) ** -0.5)
    w = _rand((d,), torch.float32, 33, scale=0.01)
    ref = O.combine(to_f64(H), to_f64(n), to_f64(W), to_f64(w))
    ran = 0
    # rows wider than 512 columns: the slabs of a row exchange their partial norms through global
    # memory (gemm_gx 1: cooperative launch, 2: plain launch) or inside a cluster (0)
    gxs = (1, 0, 2) if (dtype == torch.bfloat16 and d > 512) else (1,)
    for impl, cg in _both_impls(ctx, dtype):
        for gx in (gxs if impl == 0 else (1,)):
            ctx.pinsage_set_option("gemm_gx", gx)
            try:
                with _impl(ctx, impl, cg):
                    try:
                        got = ctx.pinsage_combine(H.to(DEV), n.to(DEV), W.to(DEV), w.to(DEV))
                    except binding.PinsageError as e:
                        if e.status_name == "UNSUPPORTED_SHAPE" and impl == 0:
                            continue
                        raise
            finally:
                ctx.pinsage_set_option("gemm_gx", 1)
            ran += 1
            assert_rows_close(to_f64(got), ref, dtype, f"combine impl={impl} cg={cg} gx={gx}",
                              tol=4e-3 if dtype == torch.bfloat16 else 1e-5)
            nrm = np.linalg.norm(to_f64(got), axis=1)
            assert np.all((np.abs(nrm - 1) < (2.0 ** -7 if dtype == torch.bfloat16 else 1e-5))
                          | (nrm == 0))
    assert ran >= 1


@pytest.mark.parametrize("dtype", DTYPES)
def test_combine_zero_rows_stay_zero(ctx, dtype):
    """A3: all-ReLU-dead rows give exactly 0, never NaN."""
    M, d = 300, 64
    H = _rand((M, d), dtype, 34).abs()
    n = _rand((M, d), dtype, 35).abs()
    W = -_rand((d, 2 * d), dtype, 36).abs()
    w = torch.zeros(d)
    got = ctx.pinsage_combine(H.to(DEV), n.to(DEV), W.to(DEV), w.to(DEV))
    assert torch.equal(got.cpu().to(torch.float32), torch.zeros((M, d)))


# ------------------------------------------------------------------ layers, head, whole path
def _inputs(cfg):
    X = synth.make_features(cfg)
    layers, head = synth.make_params(cfg)
    idx, counts = synth.make_graph(cfg)
    alpha = O.normalize_counts(counts.numpy())
    return X, idx, counts, alpha, layers, head


def _to_dev(layers, head):
    L = [{k: v.to(DEV) for k, v in lp.items()} for lp in layers]
    H = {k: v.to(DEV) for k, v in head.items()}
    return L, H


def _check_whole_path(ctx, cfg, impl=0, chunk_nodes=0, cg=0):
    """chunk_nodes may be a tuple: the one-call path is then run once per value against the same oracle
    pass (0 = the automatic driver chunk, the launch configuration bench.py times)."""
    X, idx, counts, alpha, layers, head = _inputs(cfg)
    Lf, Hf = params_f64(layers, head)
    ref_out, ref_hidden = O.embed_all(to_f64(X), idx.numpy(), alpha, Lf, Hf, return_hidden=True)
    Ld, Hd = _to_dev(layers, head)
    dtype = X.dtype
    ctx.pinsage_set_option("gemm_impl", impl)
    ctx.pinsage_set_option("gemm_cg", cg)
    try:
        w_dev = ctx.pinsage_normalize_counts(counts.to(DEV))
        np.testing.assert_array_equal(w_dev.cpu().numpy(), alpha)
        # layer by layer through pinsage_layer (every intermediate H_k is checked)
        H = X.to(DEV)
        for k, lp in enumerate(Ld):
            H = ctx.pinsage_layer(H, idx.to(DEV), w_dev, lp)
            assert_rows_close(to_f64(H), ref_hidden[k], dtype, f"{cfg.name} H_{k + 1} impl={impl}")
        out_head = ctx.pinsage_head(H, Hd)
        assert_rows_close(to_f64(out_head), ref_out, dtype, f"{cfg.name} head impl={impl}")
        # and in one call
        chunks = chunk_nodes if isinstance(chunk_nodes, (tuple, list)) else (chunk_nodes,)
        first = None
        for cn in chunks:
            out = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), w_dev, Ld, Hd, chunk_nodes=cn)
            stats = assert_rows_close(to_f64(out), ref_out, dtype, f"{cfg.name} embed_all impl={impl} chunk={cn}")
            bits = torch.int16 if dtype == torch.bfloat16 else torch.int32
            if first is None:
                first = out
            else:        # a row's arithmetic does not depend on the chunk it sits in
                assert torch.equal(first.view(bits), out.view(bits)), f"chunk_nodes={cn} changes the result"
        return out, stats
    finally:
        ctx.pinsage_set_option("gemm_impl", 0)
        ctx.pinsage_set_option("gemm_cg", 0)


def test_tiny_config_fp32_exhaustive(ctx):
    """BASELINE config 1 in full: N=2000, fp32, every row, <= 1e-4."""
    _check_whole_path(ctx, synth.CONFIGS["tiny"])


@pytest.mark.parametrize("impl,cg", [(0, 0), (0, 1), (1, 0)])
def test_cfg2_small_exhaustive(ctx, impl, cg):
    """Config 2's shape (256/256/128, T=50, K=2, bf16) on 20 000 nodes, every row; chunked
    so that several chunks, a ragged tail chunk and ragged GEMM tiles are exercised."""
    _check_whole_path(ctx, synth.CONFIGS["cfg2"].scaled(20_011), impl=impl, chunk_nodes=4096, cg=cg)


@pytest.mark.parametrize("name,N,small_chunk", [("cfg3", 50_000, 6144), ("cfg4", 100_000, 12_800),
                                                ("cfg5", 20_000, 2048)])
def test_small_siblings_exhaustive(ctx, name, N, small_chunk):
    """The "-small" siblings of configs 3-5 (same dims, T, K and value laws) at the sizes SURVEY.md 8(d)
    fixes, EVERY row against the oracle, with the automatic driver chunk and with a small one.  At these
    sizes the persistent GEMMs walk several tiles per CTA (pair): config 3's S3 (d = 1024, four 256-column
    slabs, 36 lanes of CTA pairs) runs 196 row tiles = 5-6 per lane with the automatic chunk, so both
    parities of the grid-wide norm exchange and its arrival-count targets for it >= 2 are compared with
    the oracle on every row; the small chunk adds ragged last tiles and chunk edges off the tile grid."""
    cfg = synth.CONFIGS[name].scaled(N)
    _check_whole_path(ctx, cfg, impl=0, chunk_nodes=(0, small_chunk))


def test_embed_all_deterministic_and_overlap_invariant(ctx):
    cfg = synth.CONFIGS["cfg2"].scaled(9000)
    X, idx, counts, alpha, layers, head = _inputs(cfg)
    Ld, Hd = _to_dev(layers, head)
    w = torch.from_numpy(alpha).to(DEV)
    a = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), w, Ld, Hd, chunk_nodes=1024)
    b = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), w, Ld, Hd, chunk_nodes=1024)
    assert torch.equal(a.view(torch.int16), b.view(torch.int16))
    ctx.pinsage_set_option("overlap", 1)       # two-stream schedule, different chunking
    try:
        c = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), w, Ld, Hd, chunk_nodes=3072)
    finally:
        ctx.pinsage_set_option("overlap", 0)
    assert torch.equal(a.view(torch.int16), c.view(torch.int16))
    d = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), w, Ld, Hd)   # automatic chunk (one chunk)
    assert torch.equal(a.view(torch.int16), d.view(torch.int16))


def test_embed_all_host_buffers_match_device_buffers(ctx):
    """The e2e entry: pinned host inputs / output, copies inside the call."""
    cfg = synth.CONFIGS["cfg2"].scaled(5000)
    X, idx, counts, alpha, layers, head = _inputs(cfg)
    Ld, Hd = _to_dev(layers, head)
    w = torch.from_numpy(alpha)
    dev = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), w.to(DEV), Ld, Hd)
    out_h = torch.empty((cfg.N, cfg.d_out), dtype=X.dtype).pin_memory()
    ctx.pinsage_embed_all(X.pin_memory(), idx.pin_memory(), w.pin_memory(), Ld, Hd, out=out_h)
    assert torch.equal(out_h.view(torch.int16), dev.cpu().view(torch.int16))
    # several chunks: the copies are pipelined chunk by chunk with the kernels (ragged last chunk),
    # pinned and pageable host memory, and a mix of host and device buffers
    for pin in (True, False):
        f = (lambda t: t.pin_memory()) if pin else (lambda t: t.clone())
        out_h.zero_()
        ctx.pinsage_embed_all(f(X), f(idx), f(w), Ld, Hd, out=out_h, chunk_nodes=1024)
        assert torch.equal(out_h.view(torch.int16), dev.cpu().view(torch.int16))
    out_h.zero_()
    ctx.pinsage_embed_all(X.to(DEV), idx.pin_memory(), w.to(DEV), Ld, Hd, out=out_h, chunk_nodes=640)
    assert torch.equal(out_h.view(torch.int16), dev.cpu().view(torch.int16))
    out_d = torch.empty_like(dev)            # host inputs, device output
    ctx.pinsage_embed_all(X.pin_memory(), idx.to(DEV), w.pin_memory(), Ld, Hd, out=out_d, chunk_nodes=2048)
    torch.cuda.synchronize()
    assert torch.equal(out_d.view(torch.int16), dev.view(torch.int16))


def test_layer_in_place_and_caller_workspace(ctx):
    cfg = synth.CONFIGS["cfg2"].scaled(3000)
    X, idx, counts, alpha, layers, head = _inputs(cfg)
    Ld, _ = _to_dev(layers, head)
    w = torch.from_numpy(alpha).to(DEV)
    H1 = ctx.pinsage_layer(X.to(DEV), idx.to(DEV), w, Ld[0])
    ref = ctx.pinsage_layer(H1, idx.to(DEV), w, Ld[1])
    nbytes = ctx.pinsage_layer_workspace_bytes(X.dtype, cfg.N, cfg.T, Ld[1])
    ws = torch.empty(nbytes, dtype=torch.uint8, device=DEV)
    inplace = H1.clone()
    ctx.pinsage_layer(inplace, idx.to(DEV), w, Ld[1], out=inplace, ws=ws)   # d == d_in
    assert torch.equal(inplace.view(torch.int16), ref.view(torch.int16))
    with pytest.raises(binding.PinsageError) as e:
        ctx.pinsage_layer(H1, idx.to(DEV), w, Ld[1], ws=ws[:1024])
    assert e.value.status_name == "OOM"


# ------------------------------------------------------------------ argument checking
def test_argument_errors(ctx):
    A = torch.zeros((16, 64), dtype=torch.bfloat16, device=DEV)
    W = torch.zeros((64, 64), dtype=torch.bfloat16, device=DEV)
    with pytest.raises(binding.PinsageError) as e:
        ctx.pinsage_dense(A[:, :60].contiguous(), W[:, :60].contiguous(), None, False)
    assert e.value.status_name == "UNSUPPORTED_SHAPE"
    with pytest.raises(binding.PinsageError) as e:
        ctx.pinsage_dense(A.view(-1)[4:4 + 15 * 64].view(15, 64), W, None, False)
    assert e.value.status_name == "MISALIGNED"
    idx = torch.zeros((16, 4), dtype=torch.int32, device=DEV)
    w = torch.zeros((16, 4), dtype=torch.float32, device=DEV)
    with pytest.raises(binding.PinsageError) as e:
        ctx.pinsage_pool(A, idx, w, out=A)
    assert e.value.status_name == "INVALID_ARG"
    with pytest.raises(binding.PinsageError) as e:
        ctx.pinsage_set_option("no_such_option", 1)
    assert e.value.status_name == "INVALID_ARG"
    lp = {"Q": W, "q": torch.zeros(64, device=DEV), "W": torch.zeros((64, 128), dtype=torch.bfloat16,
                                                                      device=DEV),
          "w": torch.zeros(64, device=DEV)}
    hp = {"G1": torch.zeros((32, 32), dtype=torch.bfloat16, device=DEV),
          "g": torch.zeros(32, device=DEV),
          "G2": torch.zeros((32, 32), dtype=torch.bfloat16, device=DEV)}
    with pytest.raises(binding.PinsageError) as e:       # head.d != layers[-1].d
        ctx.pinsage_embed_all(A, idx, w, [lp], hp)
    assert e.value.status_name == "INVALID_ARG"
    ctx.pinsage_set_option("check_indices", 1)
    try:
        bad = idx.clone()
        bad[3, 1] = 16
        with pytest.raises(binding.PinsageError) as e:
            ctx.pinsage_pool(A, bad, w)
        assert e.value.status_name == "BAD_INDEX"
    finally:
        ctx.pinsage_set_option("check_indices", 0)


# ------------------------------------------------------------------ random shapes (property test)
def _random_case(rng, narrow_ok):
    """A random small instance: dims multiples of 8 with m != d != d_in, odd T, K in 1..3, ragged N.
    narrow_ok=False keeps every normalised width >= 128 (the narrowest bf16 width of BASELINE.json's
    configs is 256; fp32's is 64) and the output width >= 32: with 8-wide rows ReLU regularly leaves a
    nearly dead row whose direction is ill-conditioned (a 1e-3 input rounding becomes a 3 % change of
    z / ||z||), which measures the generator, not the kernels -- those widths are exercised in fp32 mode,
    where they pass at 1e-4, and reported (not gated) in bf16 by test_narrow_bf16_rows_report_only."""
    K = int(rng.integers(1, 4))
    wide = [128, 200, 256, 320]
    any_w = [8, 24, 40, 64, 72] + wide
    dims = [int(rng.choice(any_w))] + [int(rng.choice(any_w if narrow_ok else wide)) for _ in range(K)]
    ms = [int(rng.choice([8, 16, 48, 64, 136, 256, 512] if narrow_ok else [136, 256, 512])) for _ in range(K)]
    g1 = int(rng.choice([8, 32, 64, 128, 264] if narrow_ok else [128, 264]))
    d_out = int(rng.choice([8, 16, 32, 128, 520] if narrow_ok else [32, 128, 520]))
    N = int(rng.integers(60, 3000))
    T = int(rng.choice([1, 2, 3, 7, 10, 33, 50]))
    return N, T, dims, ms, g1, d_out


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("seed", range(12))
def test_random_shapes_whole_path(ctx, dtype, seed):
    """Random (N, T, K, widths) with m != d != d_in, repeated / self neighbour ids allowed (A7):
    pinsage_embed_all against the oracle on every row, with the automatic kernel choices."""
    rng = np.random.default_rng(1000 + seed)
    N, T, dims, ms, g1, d_out = _random_case(rng, narrow_ok=dtype == torch.float32)
    g = torch.Generator().manual_seed(2000 + seed)

    def rn(*shape, std=1.0):
        return torch.randn(shape, generator=g) * std

    X = rn(N, dims[0]).to(dtype)
    layers = [{"Q": rn(ms[k], dims[k], std=dims[k] ** -0.5).to(dtype), "q": rn(ms[k], std=0.01),
               "W": rn(dims[k + 1], dims[k] + ms[k], std=(dims[k] + ms[k]) ** -0.5).to(dtype),
               "w": rn(dims[k + 1], std=0.01)} for k in range(len(ms))]
    head = {"G1": rn(g1, dims[-1], std=dims[-1] ** -0.5).to(dtype), "g": rn(g1, std=0.01),
            "G2": rn(d_out, g1, std=g1 ** -0.5).to(dtype)}
    idx = torch.randint(0, N, (N, T), generator=g, dtype=torch.int32)
    counts = torch.randint(1, 101, (N, T), generator=g, dtype=torch.int32)
    alpha = O.normalize_counts(counts.numpy())
    Lf, Hf = params_f64(layers, head)
    ref = O.embed_all(to_f64(X), idx.numpy(), alpha, Lf, Hf)
    Ld, Hd = _to_dev(layers, head)
    out = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), torch.from_numpy(alpha).to(DEV), Ld, Hd,
                                chunk_nodes=int(rng.choice([0, 128, 1024])))
    # north_star's tolerance as it stands (1e-2 bf16, 1e-4 fp32), for every K and either schedule
    assert_rows_close(to_f64(out), ref, dtype, f"random case {seed}: N={N} T={T} dims={dims} ms={ms}")


@pytest.mark.parametrize("seed", range(6))
def test_narrow_bf16_rows_report_only(ctx, seed):
    """NOT a gate of north_star's tolerance: bf16 with normalised widths below BASELINE.json's minimum
    (8 .. 72 columns).  DESIGN.md sec. 9: with so few columns a row's error is an average over few
    roundings and a nearly dead ReLU row is ill-conditioned, so the worst row of a few thousand sits at
    or above 1e-2 although every stage rounds exactly once.  Asserted here: finite output, exact zero rows,
    cosine >= 0.999 and a relative error below 5e-2 (a wrong index, sign or operand would give O(1));
    the measured maximum is printed."""
    rng = np.random.default_rng(3000 + seed)
    K = int(rng.integers(1, 4))
    narrow = [8, 24, 40, 64, 72]
    dims = [int(rng.choice(narrow)) for _ in range(K + 1)]
    ms = [int(rng.choice([8, 16, 48, 64])) for _ in range(K)]
    g1, d_out = int(rng.choice([8, 32, 64])), int(rng.choice([8, 16, 32]))
    N, T = int(rng.integers(60, 3000)), int(rng.choice([1, 3, 10, 50]))
    g = torch.Generator().manual_seed(4000 + seed)

    def rn(*shape, std=1.0):
        return torch.randn(shape, generator=g) * std

    dtype = torch.bfloat16
    X = rn(N, dims[0]).to(dtype)
    layers = [{"Q": rn(ms[k], dims[k], std=dims[k] ** -0.5).to(dtype), "q": rn(ms[k], std=0.01),
               "W": rn(dims[k + 1], dims[k] + ms[k], std=(dims[k] + ms[k]) ** -0.5).to(dtype),
               "w": rn(dims[k + 1], std=0.01)} for k in range(K)]
    head = {"G1": rn(g1, dims[-1], std=dims[-1] ** -0.5).to(dtype), "g": rn(g1, std=0.01),
            "G2": rn(d_out, g1, std=g1 ** -0.5).to(dtype)}
    idx = torch.randint(0, N, (N, T), generator=g, dtype=torch.int32)
    alpha = O.normalize_counts(torch.randint(1, 101, (N, T), generator=g, dtype=torch.int32).numpy())
    Lf, Hf = params_f64(layers, head)
    ref = O.embed_all(to_f64(X), idx.numpy(), alpha, Lf, Hf)
    Ld, Hd = _to_dev(layers, head)
    out = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), torch.from_numpy(alpha).to(DEV), Ld, Hd)
    rel, cos = row_errors(to_f64(out), ref)
    live = np.linalg.norm(ref, axis=1) > 1e-3          # nearly dead rows: direction is ill-conditioned
    print(f"narrow bf16 case {seed}: dims={dims} ms={ms} K={K} max rel L2 {rel[live].max():.3e} "
          f"(north_star gate 1e-2 applies from 128 columns)")
    assert np.isfinite(to_f64(out)).all() and rel[live].max() < 5e-2 and cos[live].min() >= 0.999


# ------------------------------------------------------------------ aggregator variants (NEXT #1)
@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("gamma,mode", [("mean", 1), ("max", 2)])
@pytest.mark.parametrize("n_dst,n_src,T,m", [(1, 1, 1, 8), (3001, 2000, 50, 256), (515, 4000, 100, 256),
                                             (300, 900, 50, 512), (77, 300, 7, 2048), (999, 999, 33, 24)])
def test_pool_mean_and_max_variants(ctx, dtype, gamma, mode, n_dst, n_src, T, m):
    """gamma = mean / max through pinsage_pool with option pool_mode."""
    if dtype == torch.float32 and m > 1024:
        pytest.skip("fp32 rows above 4 KB are outside the compiled set")
    P = _rand((n_src, m), dtype, 50 + m)
    idx, counts = _graph(n_dst, T, 51 + T, n_src=n_src)
    w = torch.from_numpy(O.normalize_counts(counts.numpy())).to(DEV)
    ctx.pinsage_set_option("pool_mode", mode)
    try:
        got = ctx.pinsage_pool(P.to(DEV), idx.to(DEV), w)
    finally:
        ctx.pinsage_set_option("pool_mode", 0)
    ref = O.pool(to_f64(P), idx.numpy(), gamma=gamma)
    if gamma == "max":      # a max of stored values is a stored value: bit-exact
        exp = torch.from_numpy(ref).to(dtype)
        bits = torch.int16 if dtype == torch.bfloat16 else torch.int32
        assert torch.equal(got.cpu().view(bits), exp.view(bits))
    else:
        assert_rows_close(to_f64(got), ref, dtype, f"mean pool T={T} m={m}",
                          tol=4e-3 if dtype == torch.bfloat16 else 2e-6)


@pytest.mark.parametrize("gamma,mode", [("mean", 1), ("max", 2)])
def test_whole_path_with_mean_and_max_pooling(ctx, gamma, mode):
    """The mean-pooling / max-pooling model variants end to end (config 2's shape, 6 000 nodes)."""
    cfg = synth.CONFIGS["cfg2"].scaled(6001)
    X, idx, counts, alpha, layers, head = _inputs(cfg)
    Lf, Hf = params_f64(layers, head)
    ref = O.embed_all(to_f64(X), idx.numpy(), None, Lf, Hf, gamma=gamma)
    Ld, Hd = _to_dev(layers, head)
    ctx.pinsage_set_option("pool_mode", mode)
    try:
        out = ctx.pinsage_embed_all(X.to(DEV), idx.to(DEV), torch.from_numpy(alpha).to(DEV), Ld, Hd,
                                    chunk_nodes=2048)
    finally:
        ctx.pinsage_set_option("pool_mode", 0)
    assert_rows_close(to_f64(out), ref, X.dtype, f"embed_all gamma={gamma}")


# ------------------------------------------------------------------ linear-pool schedule (NEXT #1)
@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("d0,m,d,N,T", [(64, 128, 64, 3000, 10), (256, 256, 256, 2500, 50),
                                        (520, 2048, 1024, 700, 50), (72, 40, 136, 1111, 7)])
def test_linear_pool_schedule_matches_oracle(ctx, dtype, d0, m, d, N, T):
    """W [h ; sum a p] = W1 h + sum a (W2 p): pooling the W2-projection (width d) gives the same
    layer as pooling P (width m) -- both schedules against the same oracle, incl. the paper's
    m = 2048, d = 1024, and mean pooling (also linear)."""
    if dtype == torch.float32 and m > 1024:
        pytest.skip("fp32 rows above 4 KB are outside the compiled set")
    g = torch.Generator().manual_seed(70 + d)
    X = torch.randn((N, d0), generator=g).to(dtype)
    lp = {"Q": (torch.randn((m, d0), generator=g) * d0 ** -0.5).to(dtype),
          "q": torch.randn((m,), generator=g) * 0.01,
          "W": (torch.randn((d, d0 + m), generator=g) * (d0 + m) ** -0.5).to(dtype),
          "w": torch.randn((d,), generator=g) * 0.01}
    idx, counts = _graph(N, T, 71)
    alpha = O.normalize_counts(counts.numpy())
    Lf, _ = params_f64([lp])
    Ld = {k: v.to(DEV) for k, v in lp.items()}
    for gamma, mode in (("importance", 0), ("mean", 1)):
        ref = O.layer_layerwise(to_f64(X), idx.numpy(), alpha, Lf[0], gamma=gamma)
        for lin in (0, 1):
            ctx.pinsage_set_option("linear_pool", lin)
            ctx.pinsage_set_option("pool_mode", mode)
            try:
                got = ctx.pinsage_layer(X.to(DEV), idx.to(DEV), torch.from_numpy(alpha).to(DEV), Ld)
            finally:
                ctx.pinsage_set_option("linear_pool", -1)
                ctx.pinsage_set_option("pool_mode", 0)
            assert_rows_close(to_f64(got), ref, dtype, f"layer linear_pool={lin} gamma={gamma}",
                              tol=6e-3 if dtype == torch.bfloat16 else 2e-5)


# ------------------------------------------------------------------ bipartite alternation (NEXT #1)
@pytest.mark.parametrize("dtype", DTYPES)
def test_bipartite_layers_compose_from_the_step_calls(ctx, dtype):
    """The paper's production graph is bipartite (pins with features, feature-less boards) and its
    layers alternate pins -> boards -> pins.  Reading A8: a board has no
    representation of its own, so its layer drops the self segment.  Composed from pinsage_dense /
    pinsage_pool (n_dst != n_src) / pinsage_combine (H = NULL), against the same composition of the
    oracle's steps."""
    n_pin, n_board, T, d0, m, d = 3000, 700, 20, 64, 128, 64
    g = torch.Generator().manual_seed(90)

    def rn(*shape, std=1.0):
        return torch.randn(shape, generator=g) * std

    X = rn(n_pin, d0).to(dtype)
    Q1, q1 = rn(m, d0, std=d0 ** -0.5).to(dtype), rn(m, std=0.01)
    W1, w1 = rn(d, m, std=m ** -0.5).to(dtype), rn(d, std=0.01)             # boards: no self segment
    Q2, q2 = rn(m, d, std=d ** -0.5).to(dtype), rn(m, std=0.01)
    W2, w2 = rn(d, d0 + m, std=(d0 + m) ** -0.5).to(dtype), rn(d, std=0.01)  # pins: self = features
    idx_b = torch.randint(0, n_pin, (n_board, T), generator=g, dtype=torch.int32)    # board <- pins
    idx_p = torch.randint(0, n_board, (n_pin, T), generator=g, dtype=torch.int32)    # pin <- boards
    a_b = O.normalize_counts(torch.randint(1, 50, (n_board, T), generator=g, dtype=torch.int32).numpy())
    a_p = O.normalize_counts(torch.randint(1, 50, (n_pin, T), generator=g, dtype=torch.int32).numpy())
    D = lambda t: t.to(DEV)
    # GPU
    P1 = ctx.pinsage_dense(D(X), D(Q1), D(q1), True)
    nb = ctx.pinsage_pool(P1, D(idx_b), D(torch.from_numpy(a_b)))
    hb = ctx.pinsage_combine(None, nb, D(W1), D(w1))
    P2 = ctx.pinsage_dense(hb, D(Q2), D(q2), True)
    np_ = ctx.pinsage_pool(P2, D(idx_p), D(torch.from_numpy(a_p)))
    hp = ctx.pinsage_combine(D(X), np_, D(W2), D(w2))
    # oracle
    f = to_f64
    oP1 = O.dense(f(X), f(Q1), f(q1), True)
    ohb = O.combine(np.zeros((n_board, 0)), O.pool(oP1, idx_b.numpy(), a_b), f(W1), f(w1))
    oP2 = O.dense(ohb, f(Q2), f(q2), True)
    ohp = O.combine(f(X), O.pool(oP2, idx_p.numpy(), a_p), f(W2), f(w2))
    assert_rows_close(to_f64(hb), ohb, dtype, "board layer", tol=6e-3 if dtype == torch.bfloat16 else 2e-5)
    assert_rows_close(to_f64(hp), ohp, dtype, "pin layer")


def test_grid_exchange_from_two_streams():
    """S3 wider than 512 columns exchanges row norms between CTA pairs of ONE launch through global
    memory: the pairs wait on each other, so the launch is cooperative (all of its CTAs get an SM before
    it starts).  Two contexts on two streams launching such GEMMs at the same time must neither block
    each other for good nor disturb each other's exchange buffers (one per stream): same bits as alone."""
    M, d_in, m, d = 30_000, 512, 512, 1024
    H = _rand((M, d_in), torch.bfloat16, 40).to(DEV)
    n = _rand((M, m), torch.bfloat16, 41).abs().to(DEV)
    W = _rand((d, d_in + m), torch.bfloat16, 42, scale=(d_in + m) ** -0.5).to(DEV)
    w = _rand((d,), torch.float32, 43, scale=0.01).to(DEV)
    s2 = torch.cuda.Stream()
    c1 = binding.Context(0)
    c2 = binding.Context(0, stream=s2.cuda_stream)
    try:
        ref = c1.pinsage_combine(H, n, W, w).clone()
        # many tiles per CTA pair (30 000 rows = 118 row tiles on 36 lanes): against the ORACLE first
        assert_rows_close(to_f64(ref), O.combine(to_f64(H), to_f64(n), to_f64(W), to_f64(w)), torch.bfloat16,
                          "d = 1024 combine, grid-wide norm exchange", tol=4e-3)
        o1, o2 = torch.empty_like(ref), torch.empty_like(ref)
        torch.cuda.synchronize()
        for _ in range(300):
            c1.pinsage_combine(H, n, W, w, out=o1)
            c2.pinsage_combine(H, n, W, w, out=o2)
        torch.cuda.synchronize()
        assert torch.equal(o1.view(torch.int16), ref.view(torch.int16))
        assert torch.equal(o2.view(torch.int16), ref.view(torch.int16))
    finally:
        c1.close()
        c2.close()
