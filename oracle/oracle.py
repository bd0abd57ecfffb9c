"""ctypes front-end of the fp64 CPU oracle (oracle/pinsage_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, bench.py's cpu_baseline /
``--impl reference`` leg and ``__graft_entry__.smoke()`` may import this module.
It imports nothing from ``paper_1806_01973_b200`` and the CUDA path imports
nothing from here.

Every array crossing into C is a C-contiguous numpy array: float64 for values,
int32 for neighbour ids / counts, float32 for alpha (reading A2 in DESIGN.md:
alpha is *defined* as a binary32 quotient).  Parameters are dicts

    layer = {"Q": [m, d_in], "q": [m], "W": [d, d_in + m], "w": [d]}
    head  = {"G1": [g1, d], "g": [g1], "G2": [d_out, g1]}

in the paper's "out x in" orientation.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pinsage_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None

_f64p = ctypes.POINTER(ctypes.c_double)
_f32p = ctypes.POINTER(ctypes.c_float)
_i32p = ctypes.POINTER(ctypes.c_int32)


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-o", tmp, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    with _lock:
        if _lib is None:
            _lib = ctypes.CDLL(build())
            _lib.oracle_num_threads.restype = ctypes.c_int
        return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_f64p)


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(_i32p)


def _f(a):
    a = np.ascontiguousarray(a, dtype=np.float32)
    return a, a.ctypes.data_as(_f32p)


def normalize_counts(counts) -> np.ndarray:
    """alpha = (float)c / (float)sum(c) per row (reading A2)."""
    c, cp = _i(counts)
    N, T = c.shape
    out = np.empty((N, T), dtype=np.float32)
    lib().oracle_normalize_counts(ctypes.c_int64(N), ctypes.c_int32(T), cp,
                                  out.ctypes.data_as(_f32p))
    return out


def dense(H, M, b=None, act=True) -> np.ndarray:
    """ReLU(H M^T + b) row by row (S1 / S4 / S5)."""
    H, Hp = _d(H)
    M, Mp = _d(M)
    N, d_in = H.shape
    d_out = M.shape[0]
    assert M.shape[1] == d_in
    if b is not None:
        b, bp = _d(b)
        assert b.shape == (d_out,)
    else:
        bp = _f64p()
    out = np.empty((N, d_out), dtype=np.float64)
    lib().oracle_dense(ctypes.c_int64(N), ctypes.c_int32(d_in), ctypes.c_int32(d_out), Hp, Mp, bp,
                       ctypes.c_int32(1 if act else 0), out.ctypes.data_as(_f64p))
    return out


GAMMAS = {"importance": 0, "mean": 1, "max": 2}


def pool(P, idx, alpha=None, gamma: str = "importance") -> np.ndarray:
    """n[v] = sum_t alpha[v,t] P[idx[v,t]] (S2).
    gamma = "mean" / "max": the element-wise ablation aggregators, alpha unused.
    P may have more rows than idx (chunked destinations)."""
    P, Pp = _d(P)
    idx, ip = _i(idx)
    N, T = idx.shape
    assert idx.min(initial=0) >= 0 and idx.max(initial=0) < P.shape[0]
    m = P.shape[1]
    out = np.empty((N, m), dtype=np.float64)
    if gamma == "importance":
        alpha, ap = _f(alpha)
        assert alpha.shape == (N, T)
        lib().oracle_pool(ctypes.c_int64(N), ctypes.c_int32(T), ctypes.c_int32(m), Pp, ip, ap,
                          out.ctypes.data_as(_f64p))
    else:
        lib().oracle_pool_gamma(ctypes.c_int64(N), ctypes.c_int32(T), ctypes.c_int32(m), Pp, ip,
                                _f32p(), ctypes.c_int32(GAMMAS[gamma]), out.ctypes.data_as(_f64p))
    return out


def combine(H, n, W, w) -> np.ndarray:
    """normalise(ReLU(W [h ; n] + w)) (S3)."""
    H, Hp = _d(H)
    n, np_ = _d(n)
    W, Wp = _d(W)
    w, wp = _d(w)
    N, d_in = H.shape
    m = n.shape[1]
    d = W.shape[0]
    assert W.shape[1] == d_in + m and n.shape[0] == N and w.shape == (d,)
    out = np.empty((N, d), dtype=np.float64)
    lib().oracle_combine(ctypes.c_int64(N), ctypes.c_int32(d_in), ctypes.c_int32(m),
                         ctypes.c_int32(d), Hp, np_, Wp, wp, out.ctypes.data_as(_f64p))
    return out


def convolve_node(h_u, h_nbr, alpha, layer) -> np.ndarray:
    """Algorithm 1 for one node."""
    h_u, hp = _d(h_u)
    h_nbr, nbp = _d(h_nbr)
    a, ap = _d(alpha)
    Q, Qp = _d(layer["Q"])
    q, qp = _d(layer["q"])
    W, Wp = _d(layer["W"])
    w, wp = _d(layer["w"])
    T, d_in = h_nbr.shape
    m, d = Q.shape[0], W.shape[0]
    assert h_u.shape == (d_in,) and a.shape == (T,) and Q.shape[1] == d_in
    assert W.shape[1] == d_in + m
    out = np.empty(d, dtype=np.float64)
    scratch = np.empty(3 * m + d_in, dtype=np.float64)
    lib().oracle_convolve_node(ctypes.c_int32(T), ctypes.c_int32(d_in), ctypes.c_int32(m),
                               ctypes.c_int32(d), hp, nbp, ap, Qp, qp, Wp, wp,
                               out.ctypes.data_as(_f64p), scratch.ctypes.data_as(_f64p))
    return out


def layer_literal(H, idx, alpha, layer) -> np.ndarray:
    """Mode A: literal Algorithm 1 node by node over all nodes."""
    H, Hp = _d(H)
    idx, ip = _i(idx)
    alpha, ap = _f(alpha)
    Q, Qp = _d(layer["Q"])
    q, qp = _d(layer["q"])
    W, Wp = _d(layer["W"])
    w, wp = _d(layer["w"])
    N, d_in = H.shape
    T = idx.shape[1]
    m, d = Q.shape[0], W.shape[0]
    assert idx.shape[0] == N and alpha.shape == idx.shape
    assert Q.shape[1] == d_in and W.shape[1] == d_in + m
    assert idx.min(initial=0) >= 0 and idx.max(initial=0) < N
    out = np.empty((N, d), dtype=np.float64)
    lib().oracle_layer_literal(ctypes.c_int64(N), ctypes.c_int32(T), ctypes.c_int32(d_in),
                               ctypes.c_int32(m), ctypes.c_int32(d), Hp, ip, ap, Qp, qp, Wp, wp,
                               out.ctypes.data_as(_f64p))
    return out


def layer_layerwise(H, idx, alpha, layer, return_parts: bool = False, gamma: str = "importance"):
    """Mode B: one layer in the sec. 3.4 schedule (project once, pool, combine)."""
    if gamma != "importance":
        P = dense(H, layer["Q"], layer["q"], act=True)
        n = pool(P, idx, None, gamma)
        out = combine(H, n, layer["W"], layer["w"])
        return (out, P, n) if return_parts else out
    H, Hp = _d(H)
    idx, ip = _i(idx)
    alpha, ap = _f(alpha)
    Q, Qp = _d(layer["Q"])
    q, qp = _d(layer["q"])
    W, Wp = _d(layer["W"])
    w, wp = _d(layer["w"])
    N, d_in = H.shape
    T = idx.shape[1]
    m, d = Q.shape[0], W.shape[0]
    assert idx.shape[0] == N and alpha.shape == idx.shape
    assert Q.shape[1] == d_in and W.shape[1] == d_in + m
    assert idx.min(initial=0) >= 0 and idx.max(initial=0) < N
    out = np.empty((N, d), dtype=np.float64)
    P = np.empty((N, m), dtype=np.float64)
    n = np.empty((N, m), dtype=np.float64)
    lib().oracle_layer_layerwise(ctypes.c_int64(N), ctypes.c_int32(T), ctypes.c_int32(d_in),
                                 ctypes.c_int32(m), ctypes.c_int32(d), Hp, ip, ap, Qp, qp, Wp, wp,
                                 out.ctypes.data_as(_f64p), P.ctypes.data_as(_f64p),
                                 n.ctypes.data_as(_f64p))
    if return_parts:
        return out, P, n
    return out


def head(H, hp) -> np.ndarray:
    """G2 ReLU(G1 h + g)."""
    H, Hp = _d(H)
    G1, G1p = _d(hp["G1"])
    g, gp = _d(hp["g"])
    G2, G2p = _d(hp["G2"])
    N, d = H.shape
    g1, d_out = G1.shape[0], G2.shape[0]
    assert G1.shape[1] == d and G2.shape[1] == g1 and g.shape == (g1,)
    out = np.empty((N, d_out), dtype=np.float64)
    lib().oracle_head(ctypes.c_int64(N), ctypes.c_int32(d), ctypes.c_int32(g1),
                      ctypes.c_int32(d_out), Hp, G1p, gp, G2p, out.ctypes.data_as(_f64p))
    return out


def embed_all(X, idx, alpha, layers, head_params=None, mode: str = "layerwise",
              return_hidden: bool = False, gamma: str = "importance"):
    """K stacked layers (Alg. 2 l.8-14) + head (l.16).

    mode = "literal" (A) or "layerwise" (B).  Returns out, or (out, [H_1..H_K])."""
    H = np.ascontiguousarray(X, dtype=np.float64)
    hidden = []
    for lp in layers:
        assert gamma == "importance" or mode == "layerwise"
        H = layer_literal(H, idx, alpha, lp) if mode == "literal" else \
            layer_layerwise(H, idx, alpha, lp, gamma=gamma)
        hidden.append(H)
    out = head(H, head_params) if head_params is not None else H
    return (out, hidden) if return_hidden else out


def rec(u: int, k: int, X, idx, alpha, layers) -> np.ndarray:
    """Mode R: brute-force recursion over the K-hop tree, nothing shared."""
    X, Xp = _d(X)
    idx, ip = _i(idx)
    alpha, ap = _f(alpha)
    T = idx.shape[1]
    K = len(layers)
    assert 0 <= k <= K
    dims = np.array([X.shape[1]] + [lp["W"].shape[0] for lp in layers], dtype=np.int32)
    ms = np.array([lp["Q"].shape[0] for lp in layers], dtype=np.int32)
    keep = []
    arrs = {}
    for name in ("Q", "q", "W", "w"):
        ptrs = (_f64p * K)()
        for i, lp in enumerate(layers):
            a, p = _d(lp[name])
            keep.append(a)
            ptrs[i] = p
        arrs[name] = ptrs
    out = np.empty(int(dims[k]), dtype=np.float64)
    lib().oracle_rec(ctypes.c_int64(u), ctypes.c_int32(k), ctypes.c_int32(T),
                     dims.ctypes.data_as(_i32p), ms.ctypes.data_as(_i32p), Xp, ip, ap,
                     arrs["Q"], arrs["q"], arrs["W"], arrs["w"], out.ctypes.data_as(_f64p))
    return out


class RecMemo:
    """Mode R-memo: the same recursion, memoised on (node, layer), reading inputs
    through row fetchers so that only the K-hop closure of the sampled
    destinations is ever touched (full-size parity sampling).

    fetch_x(ids) -> [len, d_0] float64;  fetch_nbr(ids) -> (idx [len, T] int32,
    alpha [len, T] float32).
    """

    def __init__(self, fetch_x, fetch_nbr, layers, head_params=None):
        self.fetch_x = fetch_x
        self.fetch_nbr = fetch_nbr
        self.layers = layers
        self.head_params = head_params
        self.memo = {}
        self.nbr = {}

    def _need(self, nodes, k):
        """Make sure memo holds (v, k) for all v in nodes."""
        todo = sorted({int(v) for v in nodes if (int(v), k) not in self.memo})
        if not todo:
            return
        if k == 0:
            rows = np.asarray(self.fetch_x(np.asarray(todo, dtype=np.int64)), dtype=np.float64)
            for v, r in zip(todo, rows):
                self.memo[(v, 0)] = r
            return
        miss = [v for v in todo if v not in self.nbr]
        if miss:
            ii, aa = self.fetch_nbr(np.asarray(miss, dtype=np.int64))
            for v, i_row, a_row in zip(miss, np.asarray(ii), np.asarray(aa)):
                self.nbr[v] = (np.asarray(i_row, dtype=np.int64),
                               np.asarray(a_row, dtype=np.float32))
        closure = set(todo)
        for v in todo:
            closure.update(int(x) for x in self.nbr[v][0])
        self._need(closure, k - 1)
        lp = self.layers[k - 1]
        for v in todo:
            ids, a = self.nbr[v]
            h_nbr = np.stack([self.memo[(int(x), k - 1)] for x in ids])
            self.memo[(v, k)] = convolve_node(self.memo[(v, k - 1)], h_nbr,
                                              a.astype(np.float64), lp)

    def hidden(self, nodes, k) -> np.ndarray:
        self._need(nodes, k)
        return np.stack([self.memo[(int(v), k)] for v in nodes])

    def embed(self, nodes) -> np.ndarray:
        H = self.hidden(nodes, len(self.layers))
        return head(H, self.head_params) if self.head_params is not None else H


def minibatch_embed(M, fetch_x, fetch_nbr, layers, head_params=None, return_hidden: bool = False):
    """Algorithm 2 MINIBATCH for a set M of destination nodes, touching only
    their K-hop closure -- the full-size parity sampler (rows of X / the tables are read through
    fetchers, so the arrays may live anywhere).

      lines 1-7 (:147-152)  S^(K) = M;  S^(k-1) = S^(k) U N(u) for u in S^(k)
      line 8    (:155)      h^(0)_u = x_u for u in S^(0)
      lines 9-14 (:156-164) h^(k)_u = CONVOLVE^(k)(h^(k-1)_u, {h^(k-1)_v, v in N(u)}), u in S^(k)
      lines 15-17 (:165-167) z_u = G2 ReLU(G1 h^(K)_u + g), u in M

    CONVOLVE is applied to a whole set at once through the layer-wise steps dense / pool /
    combine above (each projection computed once per member of S^(k-1)).

    fetch_x(ids int64) -> [len, d_0] float64;  fetch_nbr(ids) -> (idx [len, T], alpha [len, T]).
    Returns out [len(M), d_out] in the order of M (and the list of h^(k) rows of M if asked).
    """
    M = np.asarray(M, dtype=np.int64)
    K = len(layers)
    S = [None] * (K + 1)
    nbr = [None] * (K + 1)
    S[K] = np.unique(M)
    for k in range(K, 0, -1):
        ii, aa = fetch_nbr(S[k])
        ii = np.asarray(ii, dtype=np.int64)
        nbr[k] = (ii, np.asarray(aa, dtype=np.float32))
        S[k - 1] = np.union1d(S[k], ii.ravel())
    H = np.asarray(fetch_x(S[0]), dtype=np.float64)
    at_M = []
    for k in range(1, K + 1):
        lp = layers[k - 1]
        ii, aa = nbr[k]
        P = dense(H, lp["Q"], lp["q"], act=True)                 # every member of S^(k-1), once
        local = np.searchsorted(S[k - 1], ii).astype(np.int32)   # re-indexed sub-table
        n = pool(P, local, aa)
        H = combine(H[np.searchsorted(S[k - 1], S[k])], n, lp["W"], lp["w"])
        if return_hidden:
            at_M.append(H[np.searchsorted(S[k], M)])             # M is a subset of every S^(k)
    HM = H[np.searchsorted(S[K], M)]
    out = head(HM, head_params) if head_params is not None else HM
    return (out, at_M) if return_hidden else out


def walk_neighbourhoods(row_ptr, col_idx, n_walks: int, walk_len: int, T: int, seed: int = 0):
    """Importance-based neighbourhoods by simulated random walks (readings
    B1-B5): returns (nbr_idx [N, T] int32, counts [N, T] int32), top-T by (count desc, id asc)."""
    row_ptr = np.ascontiguousarray(row_ptr, dtype=np.int64)
    col_idx = np.ascontiguousarray(col_idx, dtype=np.int32)
    N = row_ptr.shape[0] - 1
    assert row_ptr[0] == 0 and row_ptr[-1] == col_idx.shape[0] and np.all(np.diff(row_ptr) >= 0)
    assert col_idx.size == 0 or (col_idx.min() >= 0 and col_idx.max() < N)
    idx = np.empty((N, T), dtype=np.int32)
    cnt = np.empty((N, T), dtype=np.int32)
    lib().oracle_walk_neighbourhoods(
        ctypes.c_int64(N), row_ptr.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
        col_idx.ctypes.data_as(_i32p), ctypes.c_int32(n_walks), ctypes.c_int32(walk_len),
        ctypes.c_int32(T), ctypes.c_uint64(seed), idx.ctypes.data_as(_i32p),
        cnt.ctypes.data_as(_i32p))
    return idx, cnt


def topk(Q, Z, k: int):
    """Exact K-nearest-neighbour lookup in the embedding space (PAPER.md:225 sec. 3.5; :289 "top K
    nearest neighbors ... from a sample of 5 million test pins", K = 500) -- the exact form of what the
    paper serves approximately with LSH.  Reading C1: "nearest" = largest inner product
    z_q . z_i, the score the training loss ranks by (Eq. 1, :172-176); ties go to the smaller id; the
    query itself is not excluded.  Q [nq, d], Z [N, d] -> (idx [nq, k] int32, score [nq, k] float64),
    each row ordered by (score descending, id ascending).  The matmul and the sort are numpy's."""
    Q = np.asarray(Q, dtype=np.float64)
    Z = np.asarray(Z, dtype=np.float64)
    S = Q @ Z.T
    ids = np.broadcast_to(np.arange(Z.shape[0]), S.shape)
    order = np.lexsort((ids, -S), axis=1)[:, :k]           # primary key -S, secondary key id
    return order.astype(np.int32), np.take_along_axis(S, order, axis=1)
