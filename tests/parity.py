"""Shared helpers of the parity tests: tolerances (BASELINE.json north_star) and row metrics."""
import numpy as np
import torch

# north_star: per row, cosine >= 0.999 and relative L2 error <= 1e-2 (bf16) / 1e-4 (fp32 mode)
TOL = {torch.bfloat16: 1e-2, torch.float32: 1e-4}
COS_MIN = 0.999


def to_f64(t: torch.Tensor) -> np.ndarray:
    """Exact stored values widened to double (the oracle's input convention)."""
    return t.detach().to("cpu").to(torch.float64).numpy()


def params_f64(layers, head=None):
    L = [{k: to_f64(v) for k, v in lp.items()} for lp in layers]
    H = {k: to_f64(v) for k, v in head.items()} if head is not None else None
    return L, H


def row_errors(got: np.ndarray, ref: np.ndarray):
    """(relative L2 error per row, cosine per row); rows whose reference is exactly zero must be
    exactly zero (reading A3) and report (0, 1)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape, (got.shape, ref.shape)
    rn = np.linalg.norm(ref, axis=1)
    gn = np.linalg.norm(got, axis=1)
    zero = rn == 0
    assert np.all(gn[zero] == 0), "rows that are zero in the oracle must be zero on the GPU"
    safe = np.where(zero, 1.0, rn)
    rel = np.linalg.norm(got - ref, axis=1) / safe
    cos = np.where(zero, 1.0, (got * ref).sum(axis=1) / (safe * np.where(gn == 0, 1.0, gn)))
    return rel, cos


def assert_rows_close(got, ref, dtype, what="", tol=None):
    tol = TOL[dtype] if tol is None else tol
    assert np.isfinite(np.asarray(got, dtype=np.float64)).all(), f"{what}: non-finite output"
    rel, cos = row_errors(got, ref)
    worst = int(np.argmax(rel))
    assert rel.max() <= tol, f"{what}: max rel L2 {rel.max():.3e} > {tol} at row {worst}"
    assert cos.min() >= COS_MIN, f"{what}: min cosine {cos.min():.6f}"
    return float(rel.max()), float(cos.min())
