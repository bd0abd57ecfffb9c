"""Pins for the fp64 CPU oracle (oracle/), none of which re-types its loops.

Each test fixes the oracle to something outside itself: a hand-computed worked
example, numpy / scipy library routines on special cases, closed forms,
invariants, and brute force over the K-hop computation tree.
A dropped term, wrong sign / index or transposed operand anywhere in the oracle
fails at least one of them.
"""
import os

import numpy as np
import pytest
import scipy.sparse as sp

from oracle import oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rand_layer(rng, d_in, m, d, bias=0.01):
    return {
        "Q": rng.normal(size=(m, d_in)) / np.sqrt(d_in),
        "q": rng.normal(size=m) * bias,
        "W": rng.normal(size=(d, d_in + m)) / np.sqrt(d_in + m),
        "w": rng.normal(size=d) * bias,
    }


def _rand_head(rng, d, g1, d_out):
    return {"G1": rng.normal(size=(g1, d)) / np.sqrt(d), "g": rng.normal(size=g1) * 0.01,
            "G2": rng.normal(size=(d_out, g1)) / np.sqrt(g1)}


def _rand_graph(rng, N, T, distinct=True):
    idx = np.empty((N, T), dtype=np.int32)
    for v in range(N):
        if distinct:
            cand = np.delete(np.arange(N), v)
            idx[v] = rng.choice(cand, size=T, replace=False)
        else:
            idx[v] = rng.integers(0, N, size=T)
    counts = rng.integers(1, 51, size=(N, T)).astype(np.int32)
    return idx, counts


def _adj(idx, alpha, n_src):
    N, T = idx.shape
    rows = np.repeat(np.arange(N), T)
    return sp.csr_matrix((alpha.astype(np.float64).ravel(), (rows, idx.ravel())),
                         shape=(N, n_src))


def _rownorm(Z):
    nrm = np.linalg.norm(Z, axis=1, keepdims=True)
    return np.divide(Z, nrm, out=np.zeros_like(Z), where=nrm > 0)


# --------------------------------------------------------------------------- worked example
def _read_golden(name):
    vals = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            vals[k] = np.array([float(x) for x in v])
    return vals


def test_worked_example_by_hand():
    """tests/golden/worked_example.txt: Fig.-1-shaped example, derived by hand."""
    g = _read_golden("worked_example.txt")
    X = np.array([[1., 2.], [1., 0.], [0., 1.], [2., -1.]])
    layer = {"Q": np.array([[1., -1.], [0., 2.]]), "q": np.array([0., -1.]),
             "W": np.array([[1., 0., 2., 0.], [0., 1., 0., -4.]]), "w": np.array([0.5, 0.])}
    head = {"G1": np.array([[1., 1.], [1., -4.]]), "g": np.array([0., 0.5]),
            "G2": np.array([[2., -1.]])}
    counts = np.array([[2, 1, 1]], dtype=np.int32)
    alpha = O.normalize_counts(counts)
    assert alpha.tolist() == [[0.5, 0.25, 0.25]]
    # node A alone through CONVOLVE
    hA = O.convolve_node(X[0], X[1:4], alpha[0].astype(np.float64), layer)
    np.testing.assert_allclose(hA, g["h_A_new"], rtol=0, atol=1e-15)
    # the stages of the layer-wise schedule
    P = O.dense(X, layer["Q"], layer["q"])
    np.testing.assert_array_equal(P[1:], [[1., 0.], [0., 1.], [3., 0.]])
    nA = O.pool(P, np.array([[1, 2, 3]], dtype=np.int32), alpha)
    np.testing.assert_array_equal(nA[0], g["n_A"])
    hA2 = O.combine(X[:1], nA, layer["W"], layer["w"])
    np.testing.assert_allclose(hA2[0] * np.sqrt(17.0), g["z_A"], rtol=0, atol=1e-14)
    np.testing.assert_allclose(hA2[0], g["h_A_new"], rtol=0, atol=1e-15)
    out = O.head(hA2, head)
    np.testing.assert_allclose(out[0], g["out_A"], rtol=0, atol=1e-14)
    # and through the whole-graph drivers (other nodes get arbitrary neighbourhoods)
    idx = np.array([[1, 2, 3], [0, 2, 3], [0, 1, 3], [0, 1, 2]], dtype=np.int32)
    al = np.repeat(alpha, 4, axis=0)
    for mode in ("literal", "layerwise"):
        o = O.embed_all(X, idx, al, [layer], head, mode=mode)
        np.testing.assert_allclose(o[0], g["out_A"], rtol=0, atol=1e-14)
    np.testing.assert_allclose(O.rec(0, 1, X, idx, al, [layer]), g["h_A_new"], atol=1e-15)


# --------------------------------------------------------------------------- library pins
@pytest.mark.parametrize("N,d_in,d_out", [(37, 12, 20), (5, 24, 8), (130, 16, 16)])
def test_dense_is_numpy_affine_relu(N, d_in, d_out):
    rng = np.random.default_rng(1)
    H = rng.normal(size=(N, d_in))
    M = rng.normal(size=(d_out, d_in))
    b = rng.normal(size=d_out)
    np.testing.assert_allclose(O.dense(H, M, b), np.maximum(H @ M.T + b, 0), atol=1e-13)
    np.testing.assert_allclose(O.dense(H, M, None, act=False), H @ M.T, atol=1e-13)
    np.testing.assert_allclose(O.dense(H, M, b, act=False), H @ M.T + b, atol=1e-13)


@pytest.mark.parametrize("N,T,m", [(50, 1, 8), (64, 7, 12), (200, 50, 16)])
def test_pool_is_sparse_matmul(N, T, m):
    """S2 == ELL SpMM A @ P with A[v, idx[v,t]] += alpha[v,t] (scipy fp64)."""
    rng = np.random.default_rng(2)
    P = rng.normal(size=(N, m))
    idx, counts = _rand_graph(rng, N, T, distinct=False)   # repeats and self ids are legal (A7)
    alpha = O.normalize_counts(counts)
    np.testing.assert_allclose(O.pool(P, idx, alpha), _adj(idx, alpha, N) @ P, atol=1e-14)


def test_pool_special_cases():
    rng = np.random.default_rng(3)
    N, T, m = 40, 6, 10
    P = rng.normal(size=(N, m))
    idx, counts = _rand_graph(rng, N, T)
    alpha = O.normalize_counts(counts)
    # T = 1: a plain weighted row gather
    i1 = idx[:, :1].copy()
    a1 = rng.uniform(0.5, 2.0, size=(N, 1)).astype(np.float32)
    np.testing.assert_allclose(O.pool(P, i1, a1), P[i1[:, 0]] * a1.astype(np.float64), atol=1e-15)
    # all neighbour rows equal and sum(alpha) = 1  ->  n = that row
    Pc = np.tile(rng.normal(size=(1, m)), (N, 1))
    np.testing.assert_allclose(O.pool(Pc, idx, alpha), Pc, atol=1e-6)  # alpha is fp32: sums to 1 +- T ulp
    # uniform alpha = the paper's mean-pooling variant
    au = np.full((N, T), 1.0 / T, dtype=np.float32)
    np.testing.assert_allclose(O.pool(P, idx, au), P[idx].mean(axis=1) * (np.float32(1 / T) * T),
                               atol=1e-14)
    # splitting one entry into two with weights summing to the original changes nothing
    half = (alpha[:, :1] / 2).astype(np.float32)      # exact in binary32
    idx2 = np.concatenate([idx[:, :1], idx], axis=1)
    alpha2 = np.concatenate([half, half, alpha[:, 1:]], axis=1)
    np.testing.assert_allclose(O.pool(P, idx2, alpha2), O.pool(P, idx, alpha), atol=1e-15)
    # linear in P
    P2 = rng.normal(size=(N, m))
    np.testing.assert_allclose(O.pool(P + 3 * P2, idx, alpha),
                               O.pool(P, idx, alpha) + 3 * O.pool(P2, idx, alpha), atol=1e-13)
    # destinations may be a chunk: fewer rows in idx than in P
    np.testing.assert_array_equal(O.pool(P, idx[5:9], alpha[5:9]), O.pool(P, idx, alpha)[5:9])


def test_normalize_counts():
    rng = np.random.default_rng(4)
    c = rng.integers(1, 101, size=(300, 50)).astype(np.int32)
    a = O.normalize_counts(c)
    assert a.dtype == np.float32 and (a > 0).all()
    np.testing.assert_allclose(a.astype(np.float64).sum(axis=1), 1.0, atol=50 * 2.0 ** -24)
    # bit-exact IEEE binary32 quotient (reading A2)
    ref = c.astype(np.float32) / c.sum(axis=1, keepdims=True).astype(np.float32)
    np.testing.assert_array_equal(a, ref)
    # exactly representable cases
    assert O.normalize_counts(np.array([[1, 1, 2, 4]], dtype=np.int32)).tolist() == \
        [[0.125, 0.125, 0.25, 0.5]]


def test_combine_against_numpy_and_invariants():
    rng = np.random.default_rng(5)
    N, d_in, m, d = 60, 12, 20, 8      # three different widths: a transposed read cannot pass
    H = rng.normal(size=(N, d_in))
    n = rng.normal(size=(N, m))
    W = rng.normal(size=(d, d_in + m))
    w = rng.normal(size=d)
    out = O.combine(H, n, W, w)
    Z = np.maximum(H @ W[:, :d_in].T + n @ W[:, d_in:].T + w, 0)   # two K-segments, self first
    np.testing.assert_allclose(out, _rownorm(Z), atol=1e-13)
    nrm = np.linalg.norm(out, axis=1)
    assert np.all((np.abs(nrm - 1) < 1e-14) | (nrm == 0))
    # A3: an all-negative pre-activation gives the zero row, not NaN
    out0 = O.combine(H, n, -np.abs(W) * 0, -np.ones(d))
    assert np.array_equal(out0, np.zeros((N, d)))
    # swapping the concat order is detected (self first)
    Wsw = np.concatenate([W[:, d_in:], W[:, :d_in]], axis=1)
    assert not np.allclose(O.combine(H, n[:, :d_in], W[:, :2 * d_in], w),
                           O.combine(n[:, :d_in], H, W[:, :2 * d_in], w))
    del Wsw


def test_head_against_numpy():
    rng = np.random.default_rng(6)
    N, d, g1, d_out = 33, 16, 24, 6
    H = rng.normal(size=(N, d))
    hp = _rand_head(rng, d, g1, d_out)
    ref = np.maximum(H @ hp["G1"].T + hp["g"], 0) @ hp["G2"].T    # one bias, nothing after G2 (A6)
    np.testing.assert_allclose(O.head(H, hp), ref, atol=1e-13)


# --------------------------------------------------------------------------- closed forms
def _setup(seed, N=40, T=4, d=8):
    rng = np.random.default_rng(seed)
    idx, counts = _rand_graph(rng, N, T)
    alpha = O.normalize_counts(counts)
    return rng, idx, alpha


def test_closed_form_identity_layer():
    """(i) Q=I,q=0,W=[I|0],w=0, X>=0  =>  H_1 = rownormalise(X)."""
    rng, idx, alpha = _setup(10)
    d = 8
    X = np.abs(rng.normal(size=(40, d)))
    lp = {"Q": np.eye(d), "q": np.zeros(d), "W": np.hstack([np.eye(d), np.zeros((d, d))]),
          "w": np.zeros(d)}
    for f in (O.layer_literal, O.layer_layerwise):
        np.testing.assert_allclose(f(X, idx, alpha, lp), _rownorm(X), atol=1e-15)


def test_closed_form_sparse_power_step():
    """(ii) Q=I,q=0,W=[0|I],w=0, X>=0  =>  H_k = rownormalise(A H_{k-1}) (scipy)."""
    rng, idx, alpha = _setup(11)
    d = 8
    X = np.abs(rng.normal(size=(40, d)))
    lp = {"Q": np.eye(d), "q": np.zeros(d), "W": np.hstack([np.zeros((d, d)), np.eye(d)]),
          "w": np.zeros(d)}
    A = _adj(idx, alpha, 40)
    H = X
    ref = X
    for _ in range(3):
        H = O.layer_layerwise(H, idx, alpha, lp)
        ref = _rownorm(A @ ref)
        np.testing.assert_allclose(H, ref, atol=1e-14)


def test_closed_form_self_loops_is_per_node_mlp():
    """(iii) idx[v,t] = v for all t  =>  graph-free MLP normalise(relu(W1 h + W2 relu(Q h + q) + w))."""
    rng = np.random.default_rng(12)
    N, T, d_in, m, d = 30, 5, 6, 10, 7
    X = rng.normal(size=(N, d_in))
    lp = _rand_layer(rng, d_in, m, d, bias=0.3)
    idx = np.repeat(np.arange(N, dtype=np.int32)[:, None], T, axis=1)
    alpha = O.normalize_counts(rng.integers(1, 9, size=(N, T)).astype(np.int32))
    s = alpha.astype(np.float64).sum(axis=1, keepdims=True)          # 1 +- ulp
    Pn = np.maximum(X @ lp["Q"].T + lp["q"], 0) * s
    ref = _rownorm(np.maximum(X @ lp["W"][:, :d_in].T + Pn @ lp["W"][:, d_in:].T + lp["w"], 0))
    for f in (O.layer_literal, O.layer_layerwise):
        np.testing.assert_allclose(f(X, idx, alpha, lp), ref, atol=1e-14)


def test_closed_form_positive_scale_invariance():
    """(iv) zero biases  =>  H_1(c X) = H_1(X) for c > 0."""
    rng, idx, alpha = _setup(13)
    X = rng.normal(size=(40, 8))
    lp = _rand_layer(rng, 8, 12, 10, bias=0.0)
    a = O.layer_layerwise(X, idx, alpha, lp)
    b = O.layer_layerwise(3.7 * X, idx, alpha, lp)
    np.testing.assert_allclose(a, b, atol=1e-14)
    # and the pool weights matter: a different alpha gives a different answer
    alpha2 = np.roll(alpha, 1, axis=1)
    assert np.abs(O.layer_layerwise(X, idx, alpha2, lp) - a).max() > 1e-3


# --------------------------------------------------------------------------- brute force / schedule
@pytest.mark.parametrize("K,T", [(1, 3), (2, 4), (3, 3)])
def test_recursion_equals_literal_equals_layerwise(K, T):
    """Brute force over the K-hop tree (Fig. 1) == mode A == mode B."""
    rng = np.random.default_rng(20 + K)
    N = 24
    dims = [6, 10, 8, 12][:K + 1]
    ms = [7, 5, 9][:K]
    idx, counts = _rand_graph(rng, N, T)
    alpha = O.normalize_counts(counts)
    X = rng.normal(size=(N, dims[0]))
    layers = [_rand_layer(rng, dims[k], ms[k], dims[k + 1], bias=0.05) for k in range(K)]
    hp = _rand_head(rng, dims[K], 9, 5)
    outA, hidA = O.embed_all(X, idx, alpha, layers, hp, mode="literal", return_hidden=True)
    outB, hidB = O.embed_all(X, idx, alpha, layers, hp, mode="layerwise", return_hidden=True)
    for a, b in zip(hidA + [outA], hidB + [outB]):
        np.testing.assert_array_equal(a, b)        # same arithmetic, same order: bit for bit
    for u in (0, 5, N - 1):
        np.testing.assert_allclose(O.rec(u, K, X, idx, alpha, layers), hidB[-1][u], atol=1e-15)
        np.testing.assert_allclose(O.rec(u, 0, X, idx, alpha, layers), X[u], atol=0)
    memo = O.RecMemo(lambda ids: X[ids], lambda ids: (idx[ids], alpha[ids]), layers, hp)
    rows = [3, 0, N - 1, 3]
    np.testing.assert_allclose(memo.embed(rows), outB[rows], atol=1e-15)
    np.testing.assert_allclose(memo.hidden(rows, 1), hidB[0][rows], atol=1e-15)
    nrm = np.linalg.norm(hidB[-1], axis=1)
    assert np.all((np.abs(nrm - 1) < 1e-14) | (nrm == 0))


@pytest.mark.parametrize("K,T", [(1, 5), (2, 4), (3, 3)])
def test_minibatch_algorithm2_equals_full_graph_and_brute_force(K, T):
    """Algorithm 2 on a minibatch M (K-hop sets S^(k), then CONVOLVE per
    level) gives the rows of the full-graph result and of the brute-force recursion; it is
    the sampler of the full-size GPU parity tests."""
    rng = np.random.default_rng(40 + K)
    N = 80
    dims = [6, 10, 8, 12][:K + 1]
    ms = [7, 5, 9][:K]
    idx, counts = _rand_graph(rng, N, T)
    alpha = O.normalize_counts(counts)
    X = rng.normal(size=(N, dims[0]))
    layers = [_rand_layer(rng, dims[k], ms[k], dims[k + 1], bias=0.05) for k in range(K)]
    hp = _rand_head(rng, dims[K], 9, 5)
    full, hid = O.embed_all(X, idx, alpha, layers, hp, mode="literal", return_hidden=True)
    touched = []

    def fetch_x(ids):
        touched.append(len(ids))
        return X[ids]

    M = [7, 0, N - 1, 7, 33]
    out, hM = O.minibatch_embed(M, fetch_x, lambda ids: (idx[ids], alpha[ids]), layers, hp,
                                return_hidden=True)
    np.testing.assert_allclose(out, full[M], rtol=0, atol=1e-15)
    for a, b in zip(hM, hid):
        np.testing.assert_allclose(a, b[M], rtol=0, atol=1e-15)
    for r, u in enumerate(M[:2]):
        np.testing.assert_allclose(hM[-1][r], O.rec(u, K, X, idx, alpha, layers), atol=1e-15)
    if K == 1:
        assert touched == [len(np.union1d(M, idx[M].ravel()))]   # only the closure is read
    # without a head the last hidden rows come back
    np.testing.assert_array_equal(
        O.minibatch_embed(M, fetch_x, lambda ids: (idx[ids], alpha[ids]), layers), hM[-1])


def test_neighbour_order_and_relabelling_invariance():
    """gamma is symmetric: permuting (idx, alpha) jointly within a row
    changes nothing; relabelling nodes by pi permutes the outputs by pi."""
    rng = np.random.default_rng(30)
    N, T = 32, 5
    idx, counts = _rand_graph(rng, N, T)
    alpha = O.normalize_counts(counts)
    X = rng.normal(size=(N, 6))
    layers = [_rand_layer(rng, 6, 9, 8), _rand_layer(rng, 8, 7, 8)]
    hp = _rand_head(rng, 8, 8, 4)
    base = O.embed_all(X, idx, alpha, layers, hp)
    perm = np.stack([rng.permutation(T) for _ in range(N)])
    idx_p = np.take_along_axis(idx, perm, axis=1)
    alpha_p = np.take_along_axis(alpha, perm, axis=1)
    np.testing.assert_allclose(O.embed_all(X, idx_p, alpha_p, layers, hp), base, atol=1e-14)
    pi = rng.permutation(N)              # new id of old node v is pi[v]
    inv = np.argsort(pi)
    X2 = X[inv]
    idx2 = pi[idx[inv]].astype(np.int32)
    alpha2 = alpha[inv]
    np.testing.assert_allclose(O.embed_all(X2, idx2, alpha2, layers, hp), base[inv], atol=1e-14)


def test_linearity_identity_for_w2():
    """W [h; sum a p] = W1 h + sum a (W2 p): pooling after the W2 projection is exact
    in real arithmetic -- recorded as a property of the definition."""
    rng = np.random.default_rng(31)
    N, T, d_in, m, d = 30, 4, 6, 12, 5
    idx, counts = _rand_graph(rng, N, T)
    alpha = O.normalize_counts(counts)
    X = rng.normal(size=(N, d_in))
    lp = _rand_layer(rng, d_in, m, d)
    out, P, n = O.layer_layerwise(X, idx, alpha, lp, return_parts=True)
    P2 = P @ lp["W"][:, d_in:].T
    Z = np.maximum(X @ lp["W"][:, :d_in].T + O.pool(P2, idx, alpha) + lp["w"], 0)
    np.testing.assert_allclose(_rownorm(Z), out, atol=1e-14)


def test_golden_regression_file():
    """tests/golden/tiny_rows.txt is written by tests/golden/make_golden.py, which calls
    only oracle/ -- a tripwire against silent changes of the oracle's arithmetic."""
    from tests.golden.make_golden import compute
    stored = np.loadtxt(os.path.join(GOLDEN, "tiny_rows.txt"))
    np.testing.assert_allclose(compute(), stored, rtol=0, atol=1e-15)


# --------------------------------------------------------------------------- ablation aggregators
@pytest.mark.parametrize("N,T,m", [(50, 1, 8), (64, 7, 12), (200, 50, 16)])
def test_mean_and_max_pooling_are_numpy_reductions(N, T, m):
    """gamma = mean / max == numpy mean / max over the gathered rows; mean ==
    importance pooling with uniform weights; T = 1 returns the row; order does not matter."""
    rng = np.random.default_rng(50 + T)
    P = rng.normal(size=(N + 5, m))
    idx = rng.integers(0, N + 5, size=(N, T)).astype(np.int32)
    np.testing.assert_allclose(O.pool(P, idx, gamma="mean"), P[idx].mean(axis=1), atol=1e-15)
    np.testing.assert_array_equal(O.pool(P, idx, gamma="max"), P[idx].max(axis=1))
    uniform = np.full((N, T), 1.0 / T, dtype=np.float32)
    np.testing.assert_allclose(O.pool(P, idx, gamma="mean"), O.pool(P, idx, uniform), atol=1e-6)
    if T == 1:
        np.testing.assert_array_equal(O.pool(P, idx, gamma="max"), P[idx[:, 0]])
        np.testing.assert_array_equal(O.pool(P, idx, gamma="mean"), P[idx[:, 0]])
    perm = np.stack([rng.permutation(T) for _ in range(N)])
    idx_p = np.take_along_axis(idx, perm, axis=1)
    np.testing.assert_array_equal(O.pool(P, idx_p, gamma="max"), O.pool(P, idx, gamma="max"))
    np.testing.assert_allclose(O.pool(P, idx_p, gamma="mean"), O.pool(P, idx, gamma="mean"), atol=1e-14)


def test_variant_layers_compose_the_pinned_steps():
    """A mean / max layer is dense -> variant pool -> combine; with every neighbour id equal to the
    node itself all three aggregators give the same graph-free MLP (closed form iii)."""
    rng = np.random.default_rng(60)
    N, T, d_in, m, d = 30, 4, 6, 10, 8
    X = rng.normal(size=(N, d_in))
    lp = _rand_layer(rng, d_in, m, d)
    idx = np.repeat(np.arange(N, dtype=np.int32)[:, None], T, axis=1)
    alpha = O.normalize_counts(rng.integers(1, 51, size=(N, T)).astype(np.int32))
    base = O.layer_layerwise(X, idx, alpha, lp)
    # (binary32 alpha rows sum to 1 only to ~1e-7, hence the looser match with importance pooling)
    np.testing.assert_allclose(O.layer_layerwise(X, idx, None, lp, gamma="mean"), base, atol=1e-6)
    np.testing.assert_allclose(O.layer_layerwise(X, idx, None, lp, gamma="max"),
                               O.layer_layerwise(X, idx, None, lp, gamma="mean"), atol=1e-14)
    idx2, _ = _rand_graph(rng, N, T)
    out = O.embed_all(X, idx2, None, [lp], gamma="max")
    Pm = np.maximum(X @ lp["Q"].T + lp["q"], 0)[idx2].max(axis=1)
    Z = np.maximum(X @ lp["W"][:, :d_in].T + Pm @ lp["W"][:, d_in:].T + lp["w"], 0)
    np.testing.assert_allclose(out, _rownorm(Z), atol=1e-14)


# --------------------------------------------------------------------------- importance neighbourhoods
def _csr(adj):
    row_ptr = np.zeros(len(adj) + 1, dtype=np.int64)
    row_ptr[1:] = np.cumsum([len(a) for a in adj])
    col = np.array([v for a in adj for v in a], dtype=np.int32)
    return row_ptr, col


def test_walks_on_a_directed_cycle_are_deterministic():
    """Out-degree 1 leaves nothing to chance: R walks of L steps from u visit u+1..u+L, R times
    each (readings B2-B4: ties to the smaller id, padding = (u, 0))."""
    N, R, L, T = 20, 7, 4, 6
    rp, ci = _csr([[(u + 1) % N] for u in range(N)])
    idx, cnt = O.walk_neighbourhoods(rp, ci, R, L, T, seed=3)
    for u in range(N):
        ids = sorted((u + s) % N for s in range(1, L + 1))
        assert list(idx[u]) == ids + [u] * (T - L)
        assert list(cnt[u]) == [R] * L + [0] * (T - L)
    # a cycle shorter than the walk returns to u: arrivals at u are not counted (B3)
    rp, ci = _csr([[1], [2], [0]])
    idx, cnt = O.walk_neighbourhoods(rp, ci, 5, 6, 2, seed=0)
    assert list(idx[0]) == [1, 2] and list(cnt[0]) == [10, 10]


def test_walk_visit_frequencies_match_the_markov_chain():
    """Expected visits of v != u per walk = sum_{s=1..L} (e_u P^s)_v with P the uniform
    out-neighbour transition matrix (and, as L grows, Personalized PageRank -- PAPER.md fn. 2):
    pins the uniform choice, the restart at u, the step count and the exclusion of u."""
    rng = np.random.default_rng(70)
    N, R, L = 12, 60000, 4
    adj = [list(rng.choice(np.delete(np.arange(N), u), size=rng.integers(1, 5), replace=False))
           for u in range(N)]
    adj[5] = []                                   # a dead end (B2): walks stop there
    rp, ci = _csr(adj)
    P = np.zeros((N, N))
    for u, a in enumerate(adj):
        for v in a:
            P[u, v] += 1.0 / len(a)
    idx, cnt = O.walk_neighbourhoods(rp, ci, R, L, N, seed=11)   # T = N: nothing truncated
    for u in (0, 3, 7):
        e = np.zeros(N)
        e[u] = 1.0
        expect = np.zeros(N)
        for _ in range(L):
            e = e @ P
            expect += e
        expect[u] = 0.0
        got = np.zeros(N)
        got[idx[u]] += cnt[u] / R
        np.testing.assert_allclose(got, expect, atol=5 * np.sqrt(L / R) + 1e-12)
        assert cnt[u].sum() <= R * L
    assert np.all(cnt[5] == 0) and np.all(idx[5] == 5)          # isolated start: all padding
    assert np.all(O.normalize_counts(cnt[5:6]) == 0)             # and all-zero weights, not NaN


def test_walk_neighbourhoods_ranking_and_counter_based_rng():
    rng = np.random.default_rng(71)
    N = 40
    adj = [list(rng.integers(0, N, size=rng.integers(1, 8))) for _ in range(N)]   # repeats, self loops
    rp, ci = _csr(adj)
    full_i, full_c = O.walk_neighbourhoods(rp, ci, 50, 3, N, seed=5)
    top_i, top_c = O.walk_neighbourhoods(rp, ci, 50, 3, 6, seed=5)
    np.testing.assert_array_equal(top_i, full_i[:, :6])          # top-T is a prefix of the ranking
    np.testing.assert_array_equal(top_c, full_c[:, :6])
    for u in range(N):
        keys = [(-int(c), int(i)) for i, c in zip(full_i[u], full_c[u]) if c > 0]
        assert keys == sorted(keys) and len({k[1] for k in keys}) == len(keys)   # count desc, id asc
        assert u not in {k[1] for k in keys}
        assert full_c[u].sum() <= 50 * 3
    # counter-based: a node's walks depend on (seed, u) and the graph only -- appending an
    # unreachable node changes no existing row; another seed changes the draws
    rp2, ci2 = _csr(adj + [[0]])
    np.testing.assert_array_equal(O.walk_neighbourhoods(rp2, ci2, 50, 3, 6, seed=5)[0][:N], top_i)
    assert not np.array_equal(O.walk_neighbourhoods(rp, ci, 50, 3, 6, seed=6)[1], top_c)


# --------------------------------------------------------------------------- exact top-K lookup
def test_topk_against_brute_force_and_special_cases():
    """K nearest neighbours by inner product (reading C1), ties to the smaller id."""
    rng = np.random.default_rng(80)
    Z = rng.normal(size=(37, 6))
    Q = rng.normal(size=(5, 6))
    idx, sc = O.topk(Q, Z, 7)
    for q in range(5):                                      # brute force, one pair at a time
        pairs = sorted(((-sum(Q[q, j] * Z[i, j] for j in range(6)), i) for i in range(37)))[:7]
        assert [p[1] for p in pairs] == list(idx[q])
        np.testing.assert_allclose([-p[0] for p in pairs], sc[q], atol=1e-14)
    # orthonormal candidates: the score of candidate i is the i-th coordinate of the query
    E = np.eye(6)
    q = np.array([[0.3, 0.9, -0.2, 0.9, 0.1, 0.5]])
    idx, sc = O.topk(q, E, 4)
    assert list(idx[0]) == [1, 3, 5, 0] and list(sc[0]) == [0.9, 0.9, 0.5, 0.3]   # tie 1 < 3
    assert O.topk(Q, Z, 1)[0][:, 0].tolist() == (Q @ Z.T).argmax(axis=1).tolist()
    # relabelling the candidates relabels the answer (no ties here)
    perm = rng.permutation(37)
    idx_p, sc_p = O.topk(Q, Z[perm], 7)
    np.testing.assert_array_equal(perm[idx_p], O.topk(Q, Z, 7)[0])
    # a unit-norm query among unit-norm candidates finds itself first
    U = Z / np.linalg.norm(Z, axis=1, keepdims=True)
    assert O.topk(U[[4, 9]], U, 3)[0][:, 0].tolist() == [4, 9]
