"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/pinsage.h declares.  No compute call is made without a GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1806_01973_b200 import build, binding
    build.build()
    return binding.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "pinsage.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pinsage_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    from paper_1806_01973_b200 import binding
    declared = _declared_symbols()
    assert len(declared) >= 14
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in pinsage.h but not exported"
    assert sorted(binding.SYMBOLS) == declared, "binding.SYMBOLS out of sync with pinsage.h"


def test_binding_has_the_same_names():
    from paper_1806_01973_b200 import binding
    for name in _declared_symbols():
        if name in ("pinsage_create", "pinsage_destroy", "pinsage_last_error"):
            continue  # Context.__init__ / close / PinsageError carry these
        assert hasattr(binding.Context, name) or hasattr(binding, name), name


def test_version_and_struct_layout(lib):
    from paper_1806_01973_b200 import binding
    assert "sm_100a" in binding.pinsage_version()
    # C layout of the parameter structs (int32 x3, pad, then pointers)
    assert ctypes.sizeof(binding.LayerParams) == 16 + 4 * 8
    assert ctypes.sizeof(binding.HeadParams) == 16 + 3 * 8
    assert binding.LayerParams.Q.offset == 16 and binding.HeadParams.G1.offset == 16


def test_no_silent_fallback_without_gpu(lib):
    """Without a CUDA device the library must fail loudly, never compute on the CPU."""
    import torch
    from paper_1806_01973_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = ctypes.c_void_p()
    st = lib.pinsage_create(ctypes.byref(h), 0, None)
    assert st != 0 and not h.value
    assert lib.pinsage_last_error(None)
    with pytest.raises(RuntimeError):
        binding.Context(0)
    # NULL context is rejected, not dereferenced
    assert lib.pinsage_set_option(None, b"overlap", 1) != 0
    assert lib.pinsage_launch_count(None) == 0
    lib.pinsage_destroy(None)


def test_product_does_not_import_the_oracle():
    """The CUDA path and the oracle share no code (neither imports the other)."""
    pkg = os.path.join(ROOT, "paper_1806_01973_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "pinsage_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1806_01973_b200" not in src
            assert "from paper_1806_01973_b200" not in src
            assert "pinsage.h" not in src
