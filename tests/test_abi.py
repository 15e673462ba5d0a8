"""Host-side checks that need no GPU: libgadep.so builds/loads, exports every symbol include/gadep.h declares,
and refuses to create a context without a CUDA device (no CPU fallback)."""
import ctypes
import os
import re

import pytest

import paper_2605_25963_b200 as pkg

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "gadep.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gadep_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported():
    lib = pkg.load_library()
    declared = _declared_symbols()
    assert set(declared) == set(pkg.EXPORTED_SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_library_is_in_tree_and_built_for_sm100a():
    path = pkg.library_path()
    assert os.path.exists(path) and path.startswith(ROOT)
    blob = open(path, "rb").read()
    assert b"sm_100a" in blob


def test_product_path_does_not_touch_the_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2605_25963_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f), errors="ignore").read()
                assert "import oracle" not in src and "from oracle" not in src and "gadep_oracle" not in src, f


def _has_cuda():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


@pytest.mark.skipif(_has_cuda(), reason="checks the no-GPU failure mode")
def test_create_fails_loudly_without_a_gpu():
    with pytest.raises(pkg.GadepError):
        pkg.Gadep(0)
    lib = pkg.load_library()
    h = ctypes.c_void_p()
    assert lib.gadep_create(ctypes.byref(h), 0, None) == -8 and not h.value   # GADEP_E_CUDA
    assert lib.gadep_create(None, 0, None) == -1                               # GADEP_E_NULL
    assert lib.gadep_build_bvh(None, 0) == -1
    assert lib.gadep_last_error(None) == b"null context"
