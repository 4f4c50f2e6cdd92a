"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (PDF_PATH_AUTO
with an attached workspace -> the binned persistent kernel): the CUDA path evaluates all n queries
on seeded inputs generated on the device, the oracle evaluates a random sample of them one by one.
Indices (region, sub-grid, cell) of the sample must be bit-exact, values obey tests/parity.py."""
import numpy as np
import pytest
import torch

from paper_2302_03343_b200 import synth
from conftest import make_oracle_grid
from parity import assert_values

pytestmark = pytest.mark.gpu

N_FULL = 100_000_000
N_SAMPLE = 100_000


@pytest.fixture(scope="module")
def B():
    from paper_2302_03343_b200 import binding
    assert torch.cuda.is_available()
    binding.lib()
    return binding


def _sample(n, seed):
    g = torch.Generator(device="cpu")
    g.manual_seed(seed)
    idx = torch.randint(0, n, (N_SAMPLE,), generator=g)
    idx[:64] = torch.arange(64)                      # first tile
    idx[64:128] = torch.arange(n - 64, n)            # ragged tail of the last chunk
    return idx.cuda()


def test_c2_full_size_sampled(B, oracle_mod):
    """configs[2]: 1e8 queries, 5 % extrapolated, 11 flavours, + alpha_s over the same Q2"""
    spec = synth.grid_c1()
    n = N_FULL
    g = B.PdfGrid.from_spec(spec, workspace_for=n)
    og = make_oracle_grid(oracle_mod, spec)
    x, q = synth.queries_c2(spec, n, device="cuda")
    out = g.pdf_xfxq2(spec.pids, x, q)
    assert g.pdf_error_count() == 0
    idx = _sample(n, 5)
    xs, qs = x[idx].cpu().numpy(), q[idx].cpu().numpy()
    ref, S = og.xfxq2(spec.pids, xs, qs, want_scale=True)
    assert_values(out[idx].cpu().numpy(), ref, S, "c2 full size")
    ix, iq, isub, reg = og.locate(xs, qs)
    gx, gq, gs, gr = [t.cpu().numpy() for t in g.pdf_locate(x[idx].contiguous(), q[idx].contiguous())]
    assert np.array_equal(reg, gr) and np.array_equal(isub, gs) and np.array_equal(ix, gx) and np.array_equal(iq, gq)
    assert len(np.unique(reg)) == 6                  # every class of Fig. 3.1(b) is in the sample
    del out
    a = g.pdf_alphas_q2(q)
    aref = og.alphas_q2(qs)
    assert np.max(np.abs(a[idx].cpu().numpy() - aref) / np.abs(aref)) < 1e-12


def test_c3_full_size_sampled(B, oracle_mod):
    """configs[3]: 1e8 queries over 100 member grids, one member id per query"""
    spec = synth.grid_c1(nmem=100)
    n = N_FULL
    g = B.PdfGrid.from_spec(spec, workspace_for=n)
    og = make_oracle_grid(oracle_mod, spec)
    x, q = synth.queries_inside(spec, n, synth.BASE_SEED + 1, device="cuda")
    mem = synth.members(spec, n, device="cuda")
    out = g.pdf_xfxq2(spec.pids, x, q, member=mem)
    assert g.pdf_error_count() == 0
    idx = _sample(n, 6)
    ref, S = og.xfxq2(spec.pids, x[idx].cpu().numpy(), q[idx].cpu().numpy(), member=mem[idx].cpu().numpy(), want_scale=True)
    assert_values(out[idx].cpu().numpy(), ref, S, "c3 full size")
    assert len(np.unique(mem[idx].cpu().numpy())) == 100


def test_c4_full_size_sampled(B, oracle_mod):
    """configs[4]: 1e8 events, x1, x2 log-uniform in [1e-6, 1], Q2 = x1 x2 s, weights, 11 x 11 coupling"""
    spec = synth.grid_c1()
    n = N_FULL
    g = B.PdfGrid.from_spec(spec, workspace_for=n)
    og = make_oracle_grid(oracle_mod, spec)
    x1, x2, q2, w = synth.events_c4(n, device="cuda")
    out = g.pdf_lumi(x1, x2, q2, w)
    idx = _sample(n, 7)
    ref, S = og.lumi(*[t[idx].cpu().numpy() for t in (x1, x2, q2, w)], want_scale=True)
    assert_values(out[idx].cpu().numpy(), ref, S, "c4 full size")
    assert g.pdf_error_count() == int(torch.isnan(out).sum())
