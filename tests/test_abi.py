"""CPU-side checks of the boundary: the library loads, exports every symbol include/linac.h declares,
and its host-only logic (status strings, argument validation that precedes any CUDA call) works."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2605_25863_b200 import build, linac
    build.build()
    return linac._lib()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "linac.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(linac_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    from paper_2605_25863_b200 import linac
    names = declared_functions()
    assert set(names) == set(linac.SYMBOLS), (names, linac.SYMBOLS)
    for n in names:
        assert getattr(lib, n) is not None


def test_status_strings_and_version(lib):
    assert lib.linac_version() >= 100
    seen = set()
    for s in range(0, 9):
        txt = lib.linac_status_string(s)
        assert txt and txt not in seen
        seen.add(txt)
    assert lib.linac_status_string(99) == b"unknown status"


def test_workspace_queries_and_options(lib):
    n = C.c_size_t(0)
    assert lib.linac_rref_u32_workspace(0, 10, C.byref(n)) == 0 and n.value == 0
    assert lib.linac_rref_u32_workspace(10000, 10000, C.byref(n)) == 0 and n.value > 0
    big = n.value
    assert lib.linac_rref_u32_workspace(100000, 100000, C.byref(n)) == 0 and n.value > big
    assert n.value < 40 * 2**30                      # workspace stays well below the 40 GB matrix itself
    assert lib.linac_rref_u32_workspace(-1, 10, C.byref(n)) == 1
    assert lib.linac_solve_f64_workspace(16384, 64, C.byref(n)) == 0
    assert lib.linac_set_option(b"no_such_option", 1) == 1
    assert lib.linac_set_option(b"gemm_path", 7) == 1
    assert lib.linac_set_option(b"gemm_path", 0) == 0
    assert lib.linac_set_workspace(None, 16) == 1


def test_argument_validation_needs_no_gpu(lib):
    rank = C.c_int64(-1)
    # bad modulus is rejected on the host before any CUDA call
    for p in (0, 1, 4, 9, 2147483649, 4294967295):
        assert lib.linac_rref_u32(None, 0, 0, 0, C.c_uint32(p), None, C.byref(rank), None) == 2
    assert lib.linac_rref_u32(None, 3, 3, 3, 7, None, C.byref(rank), None) == 1          # null matrix
    assert lib.linac_rref_u32(C.c_void_p(256), 3, 4, 3, 7, None, C.byref(rank), None) == 1  # ld < cols
    assert lib.linac_rref_u32(None, 0, 5, 5, 7, None, C.byref(rank), None) == 0 and rank.value == 0


def test_python_binding_refuses_cpu_tensors():
    import torch
    import paper_2605_25863_b200 as L
    with pytest.raises(ValueError):
        L.rref_u32(torch.zeros((4, 4), dtype=torch.int32), 7)
