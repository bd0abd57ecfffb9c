"""Seeded synthetic inputs for the PinSage inference path.

This module holds NONE of the method's arithmetic: it only draws features,
neighbour ids, integer visit counts and parameters with the shapes and value
laws of BASELINE.json's five configs (generator rules G1-G8, DESIGN.md
"Input recipe").  It serves both the tests' oracle side and the CUDA side, so
it imports neither.  The Pinterest graph the paper measures on
 is private; these inputs stand in for it.

Everything is a torch tensor on the requested device.  Values are produced in
fp32 and rounded (RNE) to the storage dtype; integer tables are int32.
L1-normalising the counts into alpha is the method's job (``pinsage_normalize_counts``
on the CUDA side, ``oracle.normalize_counts`` on the oracle side), not this module's.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional

import torch


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    N: int
    d0: int
    T: int
    K: int
    hidden: int          # m = d = hidden in every layer (reading A4)
    g1: int
    d_out: int
    dtype: str           # "bf16" | "f32"
    nbr_law: str         # "uniform" | "zipf_ids"
    count_law: str       # "uniform_int" | "multinomial_pool" | "multinomial_ids" | "zipf_shape"
    count_hi: int = 50   # uniform_int: counts in [1, count_hi]
    walks: int = 0       # multinomial laws: walks per node
    zipf_s: float = 0.0
    unit_rows: bool = False   # config 3: features row-L2-normalised before rounding
    seed: int = 0
    m_proj: int = 0      # projection width m when it differs from d (0: m = hidden)

    def scaled(self, N: int, name: Optional[str] = None) -> "Config":
        """The "-small" sibling: same dims, T, K and value laws, fewer nodes."""
        return dataclasses.replace(self, N=N, name=name or f"{self.name}-small")

    def layer_dims(self):
        """[(d_in, m, d)] per layer."""
        out, d_in = [], self.d0
        for _ in range(self.K):
            out.append((d_in, self.m_proj or self.hidden, self.hidden))
            d_in = self.hidden
        return out


CONFIGS: Dict[str, Config] = {
    "tiny": Config("tiny", 2_000, 64, 10, 2, 64, 64, 32, "f32", "uniform", "uniform_int", 50),
    "cfg2": Config("cfg2", 1_000_000, 256, 50, 2, 256, 256, 128, "bf16", "uniform",
                   "uniform_int", 100),
    "cfg3": Config("cfg3", 5_000_000, 2048, 50, 2, 1024, 1024, 1024, "bf16", "uniform",
                   "multinomial_pool", walks=500, zipf_s=1.1, unit_rows=True),
    "cfg4": Config("cfg4", 20_000_000, 512, 50, 2, 512, 512, 256, "bf16", "zipf_ids",
                   "multinomial_ids", walks=200, zipf_s=1.2),
    "cfg5": Config("cfg5", 50_000_000, 256, 100, 3, 256, 256, 256, "bf16", "uniform",
                   "zipf_shape"),
    # not a BASELINE config: the paper's own geometry: d0 = 4096 + 256 + 1 padded
    # to 4360, m = 2048, d = 1024, T = 50, K = 2 -- exercises m > d (the linear-pool schedule)
    "paper": Config("paper", 2_000_000, 4360, 50, 2, 1024, 1024, 1024, "bf16", "uniform",
                    "multinomial_pool", walks=500, zipf_s=1.1, unit_rows=True, m_proj=2048),
}

_TAG_X, _TAG_IDX, _TAG_CNT, _TAG_LAYER, _TAG_HEAD = 1, 2, 3, 10, 99


def torch_dtype(name: str) -> torch.dtype:
    return {"bf16": torch.bfloat16, "f32": torch.float32}[name]


def _gen(seed: int, tag: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed * (1 << 20) + tag)
    return g


def make_features(cfg: Config, device="cpu", rows: Optional[int] = None) -> torch.Tensor:
    """G1: iid N(0,1) fp32 (config 3: row / its fp32 L2 norm) -> storage dtype."""
    N = cfg.N if rows is None else rows
    g = _gen(cfg.seed, _TAG_X, device)
    out = torch.empty((N, cfg.d0), dtype=torch_dtype(cfg.dtype), device=device)
    step = max(1, (1 << 26) // cfg.d0)
    for s in range(0, N, step):
        e = min(N, s + step)
        x = torch.randn((e - s, cfg.d0), generator=g, device=device, dtype=torch.float32)
        if cfg.unit_rows:
            x = x / x.norm(dim=1, keepdim=True)
        out[s:e] = x.to(out.dtype)
    return out


def make_params(cfg: Config, device="cpu"):
    """G2: weights N(0, 1/fan_in) -> storage dtype; biases fp32 N(0, 0.01^2) (A12).
    Returns (layers, head): lists/dicts of tensors in the paper's "out x in" orientation."""
    wd = torch_dtype(cfg.dtype)
    layers: List[Dict[str, torch.Tensor]] = []
    for k, (d_in, m, d) in enumerate(cfg.layer_dims(), start=1):
        g = _gen(cfg.seed, _TAG_LAYER + k, device)

        def rn(*shape, std):
            return torch.randn(shape, generator=g, device=device, dtype=torch.float32) * std

        layers.append({
            "Q": rn(m, d_in, std=d_in ** -0.5).to(wd),
            "q": rn(m, std=0.01),
            "W": rn(d, d_in + m, std=(d_in + m) ** -0.5).to(wd),
            "w": rn(d, std=0.01),
        })
    g = _gen(cfg.seed, _TAG_HEAD, device)
    d = cfg.hidden
    head = {
        "G1": (torch.randn((cfg.g1, d), generator=g, device=device) * d ** -0.5).to(wd),
        "g": torch.randn((cfg.g1,), generator=g, device=device) * 0.01,
        "G2": (torch.randn((cfg.d_out, cfg.g1), generator=g, device=device)
               * cfg.g1 ** -0.5).to(wd),
    }
    return layers, head


def _zipf(u: torch.Tensor, R: int, s: float) -> torch.Tensor:
    """G4: continuous power law floored; u ~ U[0,1) fp64 -> rank in [0, R-1]."""
    e = 1.0 - s
    r = torch.floor((1.0 + u * ((R + 1.0) ** e - 1.0)) ** (1.0 / e)) - 1.0
    return r.clamp_(0, R - 1).to(torch.int64)


def _uniform_distinct(N: int, T: int, v0: int, rows: int, g, device) -> torch.Tensor:
    """G3: T pairwise-distinct ids uniform on {0..N-1} \\ {v}; slot order = draw order."""
    assert N - 1 >= T, "need at least T other nodes"
    v = torch.arange(v0, v0 + rows, device=device, dtype=torch.int64).unsqueeze(1)
    u = torch.randint(0, N - 1, (rows, T), generator=g, device=device, dtype=torch.int64)
    ids = u + (u >= v).to(torch.int64)
    for _ in range(1000):
        srt, order = ids.sort(dim=1, stable=True)
        dup_sorted = torch.zeros_like(srt, dtype=torch.bool)
        dup_sorted[:, 1:] = srt[:, 1:] == srt[:, :-1]
        if not bool(dup_sorted.any()):
            break
        dup = torch.zeros_like(dup_sorted)
        dup.scatter_(1, order, dup_sorted)
        n_dup = int(dup.sum())
        u2 = torch.randint(0, N - 1, (n_dup,), generator=g, device=device, dtype=torch.int64)
        vv = v.expand(rows, T)[dup]
        ids[dup] = u2 + (u2 >= vv).to(torch.int64)
    else:  # pragma: no cover
        raise RuntimeError("could not make neighbour rows distinct")
    return ids.to(torch.int32)


def _counts_multinomial_pool(cfg: Config, rows: int, g, device) -> torch.Tensor:
    """G5: 500 walks land iid on a pool of C = 4T candidates with p_j ~ (j+1)^-s;
    keep the T largest counts (ties -> smaller j), descending."""
    C = 4 * cfg.T
    p = torch.arange(1, C + 1, device=device, dtype=torch.float64) ** (-cfg.zipf_s)
    land = torch.multinomial((p / p.sum()).to(torch.float32).expand(rows, C), cfg.walks,
                             replacement=True, generator=g)
    cnt = torch.zeros((rows, C), dtype=torch.int64, device=device)
    cnt.scatter_add_(1, land, torch.ones_like(land))
    key = cnt * 1024 + (1023 - torch.arange(C, device=device, dtype=torch.int64))
    top = key.sort(dim=1, descending=True).values[:, :cfg.T]
    out = top // 1024
    # fewer than T visited candidates is vanishingly rare; pad with count 1 (never 0 rows)
    return out.clamp_(min=1).to(torch.int32)


def _zipf_ids_and_counts(cfg: Config, v0: int, rows: int, g, device):
    """G6: walks land iid on node ids by Zipf(s) (rank r = node id r, self redrawn);
    counts = multiplicities; keep top-T by (count desc, id asc); keep walking while
    fewer than T distinct ids were visited."""
    N, T = cfg.N, cfg.T
    v = torch.arange(v0, v0 + rows, device=device, dtype=torch.int64).unsqueeze(1)

    def draw(shape):
        u = torch.rand(shape, generator=g, device=device, dtype=torch.float64)
        return _zipf(u, N, cfg.zipf_s)

    def draw_noself(r, w):
        x = draw((r.shape[0], w))
        for _ in range(1000):
            bad = x == r
            nb = int(bad.sum())
            if nb == 0:
                break
            x[bad] = draw((nb,))
        return x

    land = draw_noself(v, cfg.walks)
    ids_out = torch.empty((rows, T), dtype=torch.int64, device=device)
    cnt_out = torch.empty((rows, T), dtype=torch.int64, device=device)
    todo = torch.arange(rows, device=device)
    BIG = 1 << 40
    for _ in range(1000):
        srt = land.sort(dim=1).values
        W = srt.shape[1]
        first = torch.ones_like(srt, dtype=torch.bool)
        first[:, 1:] = srt[:, 1:] != srt[:, :-1]
        pos = torch.arange(W, device=device).expand_as(srt)
        # run length = (position of next run start) - position
        nxt = torch.where(first, pos, torch.full_like(pos, W))
        nxt = torch.cat([nxt[:, 1:], torch.full_like(pos[:, :1], W)], dim=1)
        nxt = nxt.flip(1).cummin(dim=1).values.flip(1)
        run = nxt - pos
        key = torch.where(first, (W - run) * BIG + srt, torch.full_like(srt, (W + 1) * BIG))
        ksrt = key.sort(dim=1).values[:, :T]
        ok = ksrt[:, T - 1] < (W + 1) * BIG
        sel = todo[ok]
        ids_out[sel] = ksrt[ok] % BIG
        cnt_out[sel] = W - ksrt[ok] // BIG
        if bool(ok.all()):
            break
        todo = todo[~ok]
        land = torch.cat([land[~ok], draw_noself(v[todo], 50)], dim=1)
    else:  # pragma: no cover
        raise RuntimeError("zipf neighbourhoods did not reach T distinct ids")
    return ids_out.to(torch.int32), cnt_out.to(torch.int32)


def make_graph(cfg: Config, device="cpu", row_chunk: int = 1 << 20):
    """Neighbour table and integer visit counts: (nbr_idx [N,T] int32, counts [N,T] int32)."""
    N, T = cfg.N, cfg.T
    gi = _gen(cfg.seed, _TAG_IDX, device)
    gc = _gen(cfg.seed, _TAG_CNT, device)
    idx = torch.empty((N, T), dtype=torch.int32, device=device)
    cnt = torch.empty((N, T), dtype=torch.int32, device=device)
    if cfg.nbr_law == "zipf_ids":
        row_chunk = min(row_chunk, 1 << 18)
    for s in range(0, N, row_chunk):
        r = min(N, s + row_chunk) - s
        if cfg.nbr_law == "uniform":
            idx[s:s + r] = _uniform_distinct(N, T, s, r, gi, device)
        elif cfg.nbr_law == "zipf_ids":
            assert cfg.count_law == "multinomial_ids"
            i, c = _zipf_ids_and_counts(cfg, s, r, gi, device)
            idx[s:s + r], cnt[s:s + r] = i, c
            continue
        else:
            raise ValueError(cfg.nbr_law)
        if cfg.count_law == "uniform_int":      # G8
            cnt[s:s + r] = torch.randint(1, cfg.count_hi + 1, (r, T), generator=gc,
                                         device=device, dtype=torch.int32)
        elif cfg.count_law == "multinomial_pool":  # G5
            cnt[s:s + r] = _counts_multinomial_pool(cfg, r, gc, device)
        elif cfg.count_law == "zipf_shape":     # G7: ceil(100 / (t+1)), no RNG
            shape = torch.tensor([math.ceil(100 / (t + 1)) for t in range(T)],
                                 dtype=torch.int32, device=device)
            cnt[s:s + r] = shape.unsqueeze(0)
        else:
            raise ValueError(cfg.count_law)
    return idx, cnt


def make_csr(N: int, deg_lo: int, deg_hi: int, law: str = "uniform", zipf_s: float = 1.2,
             seed: int = 0, device="cpu"):
    """A synthetic directed graph in CSR form for the neighbourhood builder: out-degrees iid uniform
    on [deg_lo, deg_hi] (deg_lo = 0 gives dead ends), targets iid uniform over node ids or
    Zipf(zipf_s) over ids (hub-heavy, as in a user-curated graph -- PAPER.md:58); repeated edges
    and self loops may occur.  Returns (row_ptr [N+1] int64, col_idx [E] int32)."""
    g = _gen(seed, 4, device)
    deg = torch.randint(deg_lo, deg_hi + 1, (N,), generator=g, device=device, dtype=torch.int64)
    row_ptr = torch.zeros(N + 1, dtype=torch.int64, device=device)
    row_ptr[1:] = torch.cumsum(deg, 0)
    E = int(row_ptr[-1])
    if law == "uniform":
        col = torch.randint(0, N, (E,), generator=g, device=device, dtype=torch.int64)
    elif law == "zipf":
        col = _zipf(torch.rand((E,), generator=g, device=device, dtype=torch.float64), N, zipf_s)
    else:
        raise ValueError(law)
    return row_ptr, col.to(torch.int32)
