"""Thin ctypes binding of libpinsage.so -- same names as include/pinsage.h.

Argument marshalling only: every step of the path runs in the library's CUDA kernels.
Tensors are torch tensors used as typed device (or pinned host) memory; their
``data_ptr()`` and the current CUDA stream are what crosses the boundary.  A missing
library is a hard error (there is no CPU fallback).
"""
from __future__ import annotations

import ctypes
import os
from typing import Dict, List, Optional, Sequence

import torch

PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(PKG, "libpinsage.so")

BF16, F32 = 0, 1
STATUS = {0: "OK", 1: "INVALID_ARG", 2: "UNSUPPORTED_SHAPE", 3: "MISALIGNED", 4: "BAD_INDEX",
          5: "OOM", 6: "CUDA", 7: "ARCH"}

# every symbol include/pinsage.h declares
SYMBOLS = [
    "pinsage_create", "pinsage_destroy", "pinsage_last_error", "pinsage_version",
    "pinsage_set_option", "pinsage_launch_count", "pinsage_last_plan", "pinsage_profile_read", "pinsage_dense", "pinsage_pool",
    "pinsage_combine", "pinsage_layer", "pinsage_layer_workspace_bytes", "pinsage_head", "pinsage_head_static",
    "pinsage_embed_all", "pinsage_normalize_counts", "pinsage_validate_graph",
    "pinsage_build_neighbourhoods", "pinsage_embed_nodes", "pinsage_topk", "pinsage_calibrate",
]


class PinsageError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"pinsage: {STATUS.get(status, status)}: {message}")
        self.status = status
        self.status_name = STATUS.get(status, str(status))


class LayerParams(ctypes.Structure):
    _fields_ = [("d_in", ctypes.c_int32), ("m", ctypes.c_int32), ("d", ctypes.c_int32),
                ("Q", ctypes.c_void_p), ("q", ctypes.c_void_p),
                ("W", ctypes.c_void_p), ("w", ctypes.c_void_p)]


class HeadParams(ctypes.Structure):
    _fields_ = [("d", ctypes.c_int32), ("g1", ctypes.c_int32), ("d_out", ctypes.c_int32),
                ("G1", ctypes.c_void_p), ("g", ctypes.c_void_p), ("G2", ctypes.c_void_p)]


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libpinsage.so and declare the prototypes.  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(
            f"{LIB_PATH} is missing: build it with `python -m paper_1806_01973_b200.build` "
            "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, i32, i64, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
    lib.pinsage_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, vp]
    lib.pinsage_create.restype = ctypes.c_int
    lib.pinsage_destroy.argtypes = [vp]
    lib.pinsage_destroy.restype = None
    lib.pinsage_last_error.argtypes = [vp]
    lib.pinsage_last_error.restype = ctypes.c_char_p
    lib.pinsage_version.argtypes = []
    lib.pinsage_version.restype = ctypes.c_char_p
    lib.pinsage_set_option.argtypes = [vp, ctypes.c_char_p, i64]
    lib.pinsage_set_option.restype = ctypes.c_int
    lib.pinsage_launch_count.argtypes = [vp]
    lib.pinsage_launch_count.restype = i64
    lib.pinsage_last_plan.argtypes = [vp]
    lib.pinsage_last_plan.restype = ctypes.c_char_p
    lib.pinsage_profile_read.argtypes = [vp, i32, i32, ctypes.POINTER(ctypes.c_double),
                                         ctypes.POINTER(i64)]
    lib.pinsage_profile_read.restype = ctypes.c_int
    lib.pinsage_dense.argtypes = [vp, ctypes.c_int, i64, i32, i32, vp, vp, vp, i32, vp]
    lib.pinsage_dense.restype = ctypes.c_int
    lib.pinsage_pool.argtypes = [vp, ctypes.c_int, i64, i64, i32, i32, vp, vp, vp, vp]
    lib.pinsage_pool.restype = ctypes.c_int
    lib.pinsage_combine.argtypes = [vp, ctypes.c_int, i64, i32, i32, i32, vp, vp, vp, vp, vp]
    lib.pinsage_combine.restype = ctypes.c_int
    lib.pinsage_layer.argtypes = [vp, ctypes.c_int, i64, i32, vp, vp, vp,
                                  ctypes.POINTER(LayerParams), vp, vp, sz]
    lib.pinsage_layer.restype = ctypes.c_int
    lib.pinsage_layer_workspace_bytes.argtypes = [ctypes.c_int, i64, i32,
                                                  ctypes.POINTER(LayerParams)]
    lib.pinsage_layer_workspace_bytes.restype = sz
    lib.pinsage_head.argtypes = [vp, ctypes.c_int, i64, vp, ctypes.POINTER(HeadParams), vp]
    lib.pinsage_head.restype = ctypes.c_int
    lib.pinsage_head_static.argtypes = [vp, ctypes.c_int, i64, vp, ctypes.POINTER(HeadParams), vp]
    lib.pinsage_head_static.restype = ctypes.c_int
    lib.pinsage_embed_all.argtypes = [vp, ctypes.c_int, i64, i32, i32, vp, vp, vp,
                                      ctypes.POINTER(LayerParams), ctypes.POINTER(HeadParams),
                                      vp, i64]
    lib.pinsage_embed_all.restype = ctypes.c_int
    lib.pinsage_normalize_counts.argtypes = [vp, i64, i32, vp, vp]
    lib.pinsage_normalize_counts.restype = ctypes.c_int
    lib.pinsage_embed_nodes.argtypes = [vp, ctypes.c_int, i64, i32, i32, vp, vp, vp,
                                        ctypes.POINTER(LayerParams), ctypes.POINTER(HeadParams),
                                        i64, vp, vp]
    lib.pinsage_embed_nodes.restype = ctypes.c_int
    lib.pinsage_topk.argtypes = [vp, ctypes.c_int, i64, i64, i32, vp, vp, i32, vp, vp]
    lib.pinsage_topk.restype = ctypes.c_int
    lib.pinsage_build_neighbourhoods.argtypes = [vp, i64, vp, vp, i32, i32, i32, ctypes.c_uint64, vp, vp]
    lib.pinsage_build_neighbourhoods.restype = ctypes.c_int
    lib.pinsage_calibrate.argtypes = [vp, i32, vp, sz, i32, i64, i32, vp, sz, i32,
                                      ctypes.POINTER(ctypes.c_double)]
    lib.pinsage_calibrate.restype = ctypes.c_int
    lib.pinsage_validate_graph.argtypes = [vp, i64, i64, i32, vp, vp, ctypes.POINTER(i64)]
    lib.pinsage_validate_graph.restype = ctypes.c_int
    _lib = lib
    return lib


def pinsage_version() -> str:
    return load_library().pinsage_version().decode()


def dtype_code(t: torch.dtype) -> int:
    if t == torch.bfloat16:
        return BF16
    if t == torch.float32:
        return F32
    raise TypeError(f"unsupported dtype {t}")


def _ptr(t: Optional[torch.Tensor]):
    if t is None:
        return None
    assert t.is_contiguous(), "tensors must be contiguous (row-major)"
    return ctypes.c_void_p(t.data_ptr())


def _layer_struct(lp: Dict[str, torch.Tensor]) -> LayerParams:
    m, d_in = lp["Q"].shape
    d = lp["W"].shape[0]
    assert lp["W"].shape[1] == d_in + m, "W must be [d x (d_in+m)]"
    assert lp["q"].dtype == torch.float32 and lp["w"].dtype == torch.float32
    return LayerParams(d_in, m, d, lp["Q"].data_ptr(), lp["q"].data_ptr(), lp["W"].data_ptr(),
                       lp["w"].data_ptr())


def _head_struct(hp: Dict[str, torch.Tensor]) -> HeadParams:
    g1, d = hp["G1"].shape
    d_out = hp["G2"].shape[0]
    assert hp["G2"].shape[1] == g1 and hp["g"].dtype == torch.float32
    return HeadParams(d, g1, d_out, hp["G1"].data_ptr(), hp["g"].data_ptr(), hp["G2"].data_ptr())


class Context:
    """pinsage_ctx bound to a device and (by default) torch's current stream on it."""

    def __init__(self, device: int = 0, stream: Optional[int] = None):
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("pinsage needs a CUDA device (sm_100a); there is no CPU fallback")
        if stream is None:
            stream = torch.cuda.current_stream(device).cuda_stream
        self.device = device
        h = ctypes.c_void_p()
        st = self.lib.pinsage_create(ctypes.byref(h), device, ctypes.c_void_p(stream))
        if st != 0:
            raise PinsageError(st, self.lib.pinsage_last_error(None).decode())
        self.handle = h

    def close(self):
        if getattr(self, "handle", None):
            self.lib.pinsage_destroy(self.handle)
            self.handle = None

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _check(self, st: int):
        if st != 0:
            raise PinsageError(st, self.lib.pinsage_last_error(self.handle).decode())

    # ---- same names as include/pinsage.h -------------------------------------------------
    def pinsage_set_option(self, key: str, value: int):
        self._check(self.lib.pinsage_set_option(self.handle, key.encode(), int(value)))

    def pinsage_launch_count(self) -> int:
        return int(self.lib.pinsage_launch_count(self.handle))

    def pinsage_last_plan(self) -> str:
        return self.lib.pinsage_last_plan(self.handle).decode()

    def pinsage_profile_read(self, kind: int, layer: int = 0):
        """(total_ms, launches) of kind 0 S2 / 1 S1 / 2 S3 / 3 S4 / 4 S5 / 5 linear-pool projection in
        `layer` (0 = all layers); kind -1 resets."""
        ms, n = ctypes.c_double(0.0), ctypes.c_int64(0)
        self._check(self.lib.pinsage_profile_read(self.handle, kind, layer, ctypes.byref(ms),
                                                  ctypes.byref(n)))
        return float(ms.value), int(n.value)

    def pinsage_dense(self, A, Wt, bias, relu: bool, out=None):
        M, k = A.shape
        n_out = Wt.shape[0]
        assert Wt.shape[1] == k and Wt.dtype == A.dtype
        if out is None:
            out = torch.empty((M, n_out), dtype=A.dtype, device=A.device)
        self._check(self.lib.pinsage_dense(self.handle, dtype_code(A.dtype), M, k, n_out, _ptr(A),
                                           _ptr(Wt), _ptr(bias), int(bool(relu)), _ptr(out)))
        return out

    def pinsage_pool(self, P, nbr_idx, nbr_w, out=None):
        n_src, m = P.shape
        n_dst, T = nbr_idx.shape
        assert nbr_idx.dtype == torch.int32 and nbr_w.dtype == torch.float32
        assert nbr_w.shape == nbr_idx.shape
        if out is None:
            out = torch.empty((n_dst, m), dtype=P.dtype, device=P.device)
        self._check(self.lib.pinsage_pool(self.handle, dtype_code(P.dtype), n_dst, n_src, T, m,
                                          _ptr(P), _ptr(nbr_idx), _ptr(nbr_w), _ptr(out)))
        return out

    def pinsage_combine(self, H, n, W, w, out=None):
        """H may be None: no self segment (W is then [d x m])."""
        M, m = n.shape
        d_in = 0 if H is None else H.shape[1]
        d = W.shape[0]
        assert W.shape[1] == d_in + m and (H is None or H.shape[0] == M)
        if out is None:
            out = torch.empty((M, d), dtype=n.dtype, device=n.device)
        self._check(self.lib.pinsage_combine(self.handle, dtype_code(n.dtype), M, d_in, m, d,
                                             _ptr(H), _ptr(n), _ptr(W), _ptr(w), _ptr(out)))
        return out

    def pinsage_layer_workspace_bytes(self, dtype: torch.dtype, N: int, T: int, layer) -> int:
        ls = _layer_struct(layer)
        return int(self.lib.pinsage_layer_workspace_bytes(dtype_code(dtype), N, T,
                                                          ctypes.byref(ls)))

    def pinsage_layer(self, feats, nbr_idx, nbr_w, layer, out=None, ws=None):
        N, d_in = feats.shape
        T = nbr_idx.shape[1]
        ls = _layer_struct(layer)
        assert ls.d_in == d_in and nbr_idx.shape[0] == N and nbr_w.shape == nbr_idx.shape
        assert nbr_idx.dtype == torch.int32 and nbr_w.dtype == torch.float32
        if out is None:
            out = torch.empty((N, ls.d), dtype=feats.dtype, device=feats.device)
        self._check(self.lib.pinsage_layer(
            self.handle, dtype_code(feats.dtype), N, T, _ptr(feats), _ptr(nbr_idx), _ptr(nbr_w),
            ctypes.byref(ls), _ptr(out), _ptr(ws), 0 if ws is None else ws.numel() * ws.element_size()))
        return out

    def pinsage_head(self, h, head, out=None):
        N, d = h.shape
        hs = _head_struct(head)
        assert hs.d == d
        if out is None:
            out = torch.empty((N, hs.d_out), dtype=h.dtype, device=h.device)
        self._check(self.lib.pinsage_head(self.handle, dtype_code(h.dtype), N, _ptr(h),
                                          ctypes.byref(hs), _ptr(out)))
        return out

    def pinsage_head_static(self, h, head, out):
        """pinsage_head with the scratch in the library's static device array: allocates nothing, so `out` is
        the caller's (argument marshalling only -- no tensor is created here either)."""
        N, d = h.shape
        hs = _head_struct(head)
        assert hs.d == d and out.shape == (N, hs.d_out) and out.dtype == h.dtype
        self._check(self.lib.pinsage_head_static(self.handle, dtype_code(h.dtype), N, _ptr(h),
                                                 ctypes.byref(hs), _ptr(out)))
        return out

    def pinsage_embed_all(self, feats, nbr_idx, nbr_w, layers: Sequence[dict], head: dict,
                          out=None, chunk_nodes: int = 0):
        """feats / nbr_idx / nbr_w / out may be CUDA tensors or (pinned) host tensors."""
        N, d0 = feats.shape
        T = nbr_idx.shape[1]
        K = len(layers)
        arr = (LayerParams * K)(*[_layer_struct(lp) for lp in layers])
        hs = _head_struct(head)
        assert arr[0].d_in == d0 and nbr_idx.shape[0] == N and nbr_w.shape == nbr_idx.shape
        assert nbr_idx.dtype == torch.int32 and nbr_w.dtype == torch.float32
        if out is None:
            out = torch.empty((N, hs.d_out), dtype=feats.dtype, device=feats.device)
        self._check(self.lib.pinsage_embed_all(
            self.handle, dtype_code(feats.dtype), N, T, K, _ptr(feats), _ptr(nbr_idx),
            _ptr(nbr_w), arr, ctypes.byref(hs), _ptr(out), int(chunk_nodes)))
        return out

    def pinsage_normalize_counts(self, counts, out=None):
        N, T = counts.shape
        assert counts.dtype == torch.int32
        if out is None:
            out = torch.empty((N, T), dtype=torch.float32, device=counts.device)
        self._check(self.lib.pinsage_normalize_counts(self.handle, N, T, _ptr(counts), _ptr(out)))
        return out

    def pinsage_embed_nodes(self, feats, nbr_idx, nbr_w, layers: Sequence[dict], head: dict, targets,
                            out=None):
        """Embeddings of the nodes in `targets` (int32 CUDA tensor) only, via their K-hop closure."""
        N, d0 = feats.shape
        T = nbr_idx.shape[1]
        K = len(layers)
        arr = (LayerParams * K)(*[_layer_struct(lp) for lp in layers])
        hs = _head_struct(head)
        assert arr[0].d_in == d0 and targets.dtype == torch.int32 and targets.dim() == 1
        M = targets.shape[0]
        if out is None:
            out = torch.empty((M, hs.d_out), dtype=feats.dtype, device=feats.device)
        self._check(self.lib.pinsage_embed_nodes(
            self.handle, dtype_code(feats.dtype), N, T, K, _ptr(feats), _ptr(nbr_idx), _ptr(nbr_w), arr,
            ctypes.byref(hs), M, _ptr(targets), _ptr(out)))
        return out

    def pinsage_topk(self, Q, Z, k: int):
        """(idx [nq, k] int32, score [nq, k] fp32): the k candidates of Z with the largest Q . Z."""
        nq, d = Q.shape
        N = Z.shape[0]
        assert Z.shape[1] == d and Z.dtype == Q.dtype
        idx = torch.empty((nq, k), dtype=torch.int32, device=Q.device)
        score = torch.empty((nq, k), dtype=torch.float32, device=Q.device)
        self._check(self.lib.pinsage_topk(self.handle, dtype_code(Q.dtype), nq, N, d, _ptr(Q), _ptr(Z),
                                          int(k), _ptr(idx), _ptr(score)))
        return idx, score

    def pinsage_build_neighbourhoods(self, row_ptr, col_idx, n_walks: int, walk_len: int, T: int,
                                     seed: int = 0):
        """(nbr_idx, counts) [N, T] int32 from a CSR graph (row_ptr int64 [N+1], col_idx int32)."""
        assert row_ptr.dtype == torch.int64 and col_idx.dtype == torch.int32
        N = row_ptr.shape[0] - 1
        idx = torch.empty((N, T), dtype=torch.int32, device=row_ptr.device)
        cnt = torch.empty((N, T), dtype=torch.int32, device=row_ptr.device)
        self._check(self.lib.pinsage_build_neighbourhoods(
            self.handle, N, _ptr(row_ptr), _ptr(col_idx), int(n_walks), int(walk_len), int(T),
            ctypes.c_uint64(seed), _ptr(idx), _ptr(cnt)))
        return idx, cnt

    def pinsage_calibrate(self, kind: int, table, row_bytes: int, n_dst: int, T: int, out, reps: int = 5):
        """Milliseconds per launch of calibration kernel `kind` (0 stream, 1 random-row gather)."""
        ms = ctypes.c_double(0.0)
        self._check(self.lib.pinsage_calibrate(
            self.handle, int(kind), _ptr(table), table.numel() * table.element_size(), int(row_bytes),
            int(n_dst), int(T), _ptr(out), out.numel() * out.element_size(), int(reps), ctypes.byref(ms)))
        return float(ms.value)

    def pinsage_validate_graph(self, nbr_idx, nbr_w, n_src: int) -> int:
        """Returns -1 if the tables are valid, else raises PinsageError(BAD_INDEX)."""
        n_dst, T = nbr_idx.shape
        bad = ctypes.c_int64(-1)
        st = self.lib.pinsage_validate_graph(self.handle, n_dst, n_src, T, _ptr(nbr_idx),
                                             _ptr(nbr_w), ctypes.byref(bad))
        self.first_bad = int(bad.value)
        self._check(st)
        return int(bad.value)
