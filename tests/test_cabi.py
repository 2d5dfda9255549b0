"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/pb.h declares.
No compute call is made here (there is no GPU); argument validation that needs no device is checked."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1704_02745_b200 import build as pb_build
    from paper_1704_02745_b200 import load_library

    pb_build.build()
    return load_library()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "pb.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pb_[a-z_]+)\s*\(", hdr))
    assert {"pb_create", "pb_solve", "pb_destroy", "pb_apply", "pb_set_rhs"} <= declared
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in pb.h but not exported"
    from paper_1704_02745_b200.binding import EXPORTS

    assert declared == set(EXPORTS)


def test_strerror_and_version(lib):
    assert lib.pb_version() >= 100
    msgs = {lib.pb_strerror(s).decode() for s in range(8)}
    assert len(msgs) == 8 and all(msgs)
    assert lib.pb_strerror(99).decode() == "unknown status"


def test_argument_validation_needs_no_device(lib):
    h = ctypes.c_void_p()
    dummy = (ctypes.c_double * 64)()
    p = ctypes.cast(dummy, ctypes.c_void_p)
    # bad sizes / spacing / NULL eps are rejected before any CUDA call
    assert lib.pb_create(ctypes.byref(h), 0, 2, 2, 0.5, p, p, p, None, None, None, 0, None) == 1
    assert lib.pb_create(ctypes.byref(h), 2, 2, 2, -1.0, p, p, p, None, None, None, 0, None) == 1
    assert lib.pb_create(ctypes.byref(h), 2, 2, 2, 0.5, None, p, p, None, None, None, 0, None) == 1
    assert lib.pb_create(None, 2, 2, 2, 0.5, p, p, p, None, None, None, 0, None) == 1
    assert h.value is None
    assert lib.pb_destroy(None) == 0
    assert lib.pb_solve(None, 1e-5, 10, 0, 1, p, 0, None, None) == 1
    assert lib.pb_apply(None, 1, p, p, 0) == 1
    assert lib.pb_set_rhs(None, p, p, 0) == 1


def test_no_cpu_fallback_without_device(lib):
    """Without a CUDA device pb_create must fail loudly (PB_ERR_CUDA), never compute on the host."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    h = ctypes.c_void_p()
    dummy = (ctypes.c_double * 64)(*([1.0] * 64))
    p = ctypes.cast(dummy, ctypes.c_void_p)
    assert lib.pb_create(ctypes.byref(h), 2, 2, 2, 0.5, p, p, p, None, None, None, 0, None) == 3
    assert h.value is None


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1704_02745_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "pbref" not in src and "import oracle" not in src and "from oracle" not in src, f
