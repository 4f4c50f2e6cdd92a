"""pdf_xfxq2_noalloc: the binned kernel with its scratch in the library's static device array (include/pdfgrid.h,
csrc/pdf_noalloc.inl), for callers that may not allocate.  Its output is checked against the existing paths' output
and the oracle, within the tolerance every parity test uses (tests/parity.py), on calls in a row that share the array;
the size limit is rejected with a clear error; the call leaves the device's free memory untouched.

Collected last on purpose (the suite runs with pytest -x): it passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest
import torch

from paper_2302_03343_b200 import synth
from conftest import make_oracle_grid
from parity import assert_values

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2302_03343_b200 import binding
    assert torch.cuda.is_available()
    binding.lib()
    return binding


def with_invalid(x, q):
    x, q = x.clone(), q.clone()
    x[5], x[77], q[123], q[256] = -1.0, float("nan"), 0.0, float("inf")
    return x, q


def test_noalloc_matches_the_existing_paths_on_calls_in_a_row(B, oracle_mod):
    spec = synth.grid_c1()
    og = make_oracle_grid(oracle_mod, spec)
    g = B.PdfGrid.from_spec(spec, workspace_for=0)                       # no workspace attached at all
    probe = torch.zeros((1, len(spec.pids)), dtype=torch.float64, device="cuda")
    one = torch.full((1,), 0.1, dtype=torch.float64, device="cuda")
    max_n = g.pdf_xfxq2_noalloc(spec.pids, one, 100.0 * one, probe)
    assert 100_000 <= max_n <= 1 << 24 and max_n % 256 == 0, max_n

    # the existing paths: direct (no workspace) and binned with a caller workspace, on a handle of their own
    gb = B.PdfGrid.from_spec(spec, workspace_for=max_n)
    gb.pdf_grid_set_option(B.PDF_OPT_PATH, B.PDF_PATH_BINNED)
    g.pdf_grid_set_option(B.PDF_OPT_PATH, B.PDF_PATH_DIRECT)

    sizes = [max_n, 100_003, 257, max_n - 255]                         # the limit, ragged tails, a tiny call, again large
    first = None
    for k, n in enumerate(sizes + [sizes[0]]):
        x, q = with_invalid(*synth.queries_c2(spec, n, seed=synth.BASE_SEED + 100 + (k % len(sizes))))
        xd, qd = x.cuda(), q.cuda()
        out = torch.full((n, len(spec.pids)), -7.0, dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        assert g.pdf_xfxq2_noalloc(spec.pids, xd, qd, out) == max_n
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0, "the call changed the device's free memory"
        assert g.pdf_last_path() == B.PDF_PATH_BINNED
        assert g.pdf_error_count() == 4
        got = out.cpu().numpy()
        ref, S = og.xfxq2(spec.pids, x.numpy(), q.numpy(), want_scale=True)
        assert np.isnan(ref[[5, 77, 123, 256]]).all()
        assert_values(got, ref, S, f"noalloc vs oracle, call {k}", strict=1e-12)
        direct = g.pdf_xfxq2(spec.pids, xd, qd).cpu().numpy()
        binned = gb.pdf_xfxq2(spec.pids, xd, qd).cpu().numpy()
        assert g.pdf_last_path() == B.PDF_PATH_DIRECT and gb.pdf_last_path() == B.PDF_PATH_BINNED
        assert g.pdf_error_count() == 4 and gb.pdf_error_count() == 4
        assert_values(got, np.where(np.isnan(ref), ref, direct), S, f"noalloc vs direct path, call {k}")
        assert_values(got, np.where(np.isnan(ref), ref, binned), S, f"noalloc vs binned path, call {k}")
        if k == 0:
            first = got
    # the repeat of call 0 after other calls used the array (which queries overflow a full bin into the list units
    # depends on the order of the atomics, and the two kinds of unit sum in different orders: tolerance, not bits)
    assert_values(got, first, S, "noalloc, call 0 repeated")


def test_noalloc_subset_of_columns_and_stream(B, oracle_mod):
    spec = synth.grid_c1()
    og = make_oracle_grid(oracle_mod, spec)
    g = B.PdfGrid.from_spec(spec, workspace_for=0)
    n, pids = 50_001, [21, 2, -1, 6]                                     # 6 is not in the grid: a column of zeros
    x, q = synth.queries_c2(spec, n, seed=synth.BASE_SEED + 200)
    st = torch.cuda.Stream()
    out = torch.empty((n, len(pids)), dtype=torch.float64, device="cuda")
    xd, qd = x.cuda(), q.cuda()
    torch.cuda.synchronize()
    g.pdf_xfxq2_noalloc(pids, xd, qd, out, stream=st)
    st.synchronize()
    ref, S = og.xfxq2(pids, x.numpy(), q.numpy(), want_scale=True)
    assert_values(out.cpu().numpy(), ref, S, "noalloc, 4 columns on a side stream")
    assert np.all(out.cpu().numpy()[:, 3] == 0.0)


def test_noalloc_rejects_what_the_array_cannot_hold(B):
    spec = synth.grid_c1()
    g = B.PdfGrid.from_spec(spec, workspace_for=0)
    one = torch.full((1,), 0.1, dtype=torch.float64, device="cuda")
    max_n = g.pdf_xfxq2_noalloc(spec.pids, one, 100.0 * one, torch.zeros((1, 11), dtype=torch.float64, device="cuda"))
    n = max_n + 1
    x = torch.full((n,), 0.1, dtype=torch.float64, device="cuda")
    out = torch.full((n, 11), -7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(B.PdfGridError, match=r"beyond the \d+ queries that the static scratch"):
        g.pdf_xfxq2_noalloc(spec.pids, x, 100.0 * x, out)
    torch.cuda.synchronize()
    assert bool((out == -7.0).all())                                    # a rejected call launches nothing
    empty = torch.empty((0,), dtype=torch.float64, device="cuda")
    assert g.pdf_xfxq2_noalloc(spec.pids, empty, empty, torch.empty((0, 11), dtype=torch.float64, device="cuda")) == max_n
