"""Writes tests/golden/tiny_rows.txt from the oracle ALONE (no CUDA path involved).

Run:  python tests/golden/make_golden.py
The stored rows are a regression tripwire for the oracle's arithmetic, not a pin:
the pins are in tests/test_oracle_pins.py.  Inputs come from numpy's default_rng so the
file depends on nothing but numpy and oracle/.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import oracle as O  # noqa: E402


def compute():
    rng = np.random.default_rng(1806_01973)
    N, T, d0, m, d, g1, d_out = 50, 4, 6, 10, 8, 8, 4
    X = rng.normal(size=(N, d0))
    idx = np.stack([rng.choice(np.delete(np.arange(N), v), size=T, replace=False)
                    for v in range(N)]).astype(np.int32)
    alpha = O.normalize_counts(rng.integers(1, 51, size=(N, T)).astype(np.int32))
    layers = []
    for d_in in (d0, d):
        layers.append({"Q": rng.normal(size=(m, d_in)) / np.sqrt(d_in),
                       "q": rng.normal(size=m) * 0.01,
                       "W": rng.normal(size=(d, d_in + m)) / np.sqrt(d_in + m),
                       "w": rng.normal(size=d) * 0.01})
    head = {"G1": rng.normal(size=(g1, d)) / np.sqrt(d), "g": rng.normal(size=g1) * 0.01,
            "G2": rng.normal(size=(d_out, g1)) / np.sqrt(g1)}
    out = O.embed_all(X, idx, alpha, layers, head, mode="literal")
    # four live rows and, last, node 49, whose output is legitimately all zero (its ReLUs are all dead:
    # reading A3) -- kept as the explicit zero-row case, not as a fourth of the tripwire
    rows = [0, 1, 17, 33, N - 1]
    assert all(np.abs(out[r]).max() > 1e-3 for r in rows[:-1])
    return out[rows]


if __name__ == "__main__":
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tiny_rows.txt")
    np.savetxt(path, compute(), fmt="%.17g",
               header="rows 0, 1, 17, 33, 49 of oracle.embed_all(mode=literal); "
                      "written by tests/golden/make_golden.py")
    print("wrote", path)
