"""CPU-side checks of the boundary: libshasta.so builds, loads and exports every symbol that
include/shasta.h declares (no compute calls without a GPU), and fails loudly without a device."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1206_0919_b200 import build, shasta
    build.build()
    return shasta.load()


def test_header_symbols_are_exported(lib):
    from paper_1206_0919_b200 import shasta
    hdr = open(os.path.join(ROOT, "include", "shasta.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(shasta_[a-z_]+)\s*\(", hdr))
    assert declared == set(shasta.SYMBOLS), declared ^ set(shasta.SYMBOLS)
    for s in declared:
        assert hasattr(lib, s), s


def test_no_device_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1206_0919_b200 import shasta
    with pytest.raises(shasta.ShastaError) as ei:
        shasta.Shasta(8, 8, 8, 0.1, 0.4, 4.0 / 3.0)
    assert "no CPU fallback" in str(ei.value) or "CUDA" in str(ei.value)


def test_bad_arguments_rejected_before_cuda(lib):
    h = C.c_void_p()
    assert lib.shasta_create(C.byref(h), 0, 4, 4, 0.1, 0.4, 4.0 / 3.0) == -1
    assert lib.shasta_create(C.byref(h), 4, 4, 4, 0.1, 0.6, 4.0 / 3.0) == -1
    assert lib.shasta_create(C.byref(h), 4, 4, 4, -1.0, 0.4, 4.0 / 3.0) == -1
    assert lib.shasta_create(C.byref(h), 4, 4, 4, 0.1, 0.4, 1.0) == -1
    assert b"lambda" in lib.shasta_last_error(None) or b"gamma" in lib.shasta_last_error(None)
    assert lib.shasta_step(None, 1, None) == -1


def test_product_does_not_import_oracle():
    # the product path must not route through oracle/ (and the oracle must not import the product)
    pkg = os.path.join(ROOT, "paper_1206_0919_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("oracle tests", "").replace("the oracle", "").replace(
                    "`oracle/`", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1206_0919_b200" not in src and "from paper_1206_0919_b200" not in src
            assert "libshasta" not in src
