"""pytest configuration: markers and import path.

`-m "not gpu"` covers the oracle against its pins, the host logic and the C-ABI
symbol table; `-m gpu` holds the parity tests proper (CUDA path vs oracle)."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200, sm_100a)")
    # a fresh checkout has no libpinsage.so (it is git-ignored): build it once, as
    # `__graft_entry__.build()` does (nvcc cross-compiles without a GPU; no-op when it is up to date)
    try:
        from paper_1806_01973_b200 import build as _build
        _build.build()
    except Exception as e:  # pragma: no cover -- the tests that need the library then fail loudly
        print(f"conftest: could not build libpinsage.so: {e}", file=sys.stderr)


def pytest_collection_modifyitems(config, items):
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:  # pragma: no cover
        has_gpu = False
    if has_gpu:
        return
    skip = pytest.mark.skip(reason="no CUDA device")
    for item in items:
        if "gpu" in item.keywords:
            item.add_marker(skip)
