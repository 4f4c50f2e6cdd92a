"""CPU-side checks of the product: the C-ABI library builds, loads and exports every symbol
include/pdfgrid.h declares; host-side argument validation that needs no GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2302_03343_b200 import build, binding
    build.build()
    return binding.lib()


def test_header_symbols_exported(L):
    from paper_2302_03343_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "pdfgrid.h")).read()
    declared = set(re.findall(r"\b(pdf_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.SYMBOLS), declared ^ set(binding.SYMBOLS)
    for s in declared:
        assert hasattr(L, s), s


def test_status_strings(L):
    assert L.pdf_status_string(0) == b"ok"
    for rc in (-1, -2, -3, -4, -5):
        assert L.pdf_status_string(rc) not in (b"ok", b"unknown status")
    assert L.pdf_launch_count() >= 0


def test_create_rejects_bad_arguments_without_gpu(L):
    """validation happens before any CUDA call, so it can be exercised on a CPU-only box"""
    from paper_2302_03343_b200 import binding
    dbl, ci = ctypes.c_double, ctypes.c_int
    h = ctypes.c_void_p()

    def create(x, nq, q2, vals, pids, nmem=1):
        return L.pdf_grid_create(ctypes.byref(h), len(x), (dbl * len(x))(*x), len(nq), (ci * len(nq))(*nq),
                                 (dbl * len(q2))(*q2), (dbl * len(vals))(*vals), len(pids),
                                 (ci * len(pids))(*pids), nmem)
    ok_v = [0.0] * (3 * 4 * 1)
    assert create([0.1, 0.05, 1.0], [4], [1, 2, 3, 4], ok_v, [21]) == binding.PDF_EINVAL     # x not increasing
    assert create([0.1, 0.5, 1.0], [4], [1, 2, 2, 4], ok_v, [21]) == binding.PDF_EINVAL      # q2 not increasing
    assert create([0.1, 0.5, 1.0], [2, 2], [1, 2, 3, 4], ok_v, [21]) == binding.PDF_EINVAL   # threshold mismatch
    assert create([0.1, 0.5, 1.0], [4], [1, 2, 3, 4], [float("nan")] * 12, [21]) == binding.PDF_EINVAL
    assert create([-0.1, 0.5, 1.0], [4], [1, 2, 3, 4], ok_v, [21]) == binding.PDF_EINVAL
    assert create([0.1, 0.5, 1.0], [1, 3], [1, 1, 3, 4], ok_v, [21]) == binding.PDF_EINVAL   # sub-grid with 1 knot
    assert L.pdf_grid_destroy(None) == 0
    assert L.pdf_workspace_bytes(None, 10) == 0
