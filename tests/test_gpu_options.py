"""NEXT-4 on the GPU: the extrapolation options of PAPER.md L1720 (freeze, error) and xfxQ (L1712), both evaluation
paths, against the oracle under the same option; the luminosity and the multi-member call under 'freeze'."""
import numpy as np
import pytest
import torch

from paper_2302_03343_b200 import synth
from conftest import make_oracle_grid
from parity import assert_values
from test_gpu_parity import B, PATHS, check_locate, gpu_grid  # noqa: F401  (B is a fixture)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("mode", ["freeze", "error"])
def test_extrapolation_options_parity(B, oracle_mod, path, mode):
    spec = synth.grid_c1()
    n = 400_000
    x, q = synth.queries_c2(spec, n, seed=77)
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec, path, n)
    og.set_extrapolation({"freeze": oracle_mod.EXTRAP_FREEZE, "error": oracle_mod.EXTRAP_ERROR}[mode])
    g.pdf_grid_set_option(B.PDF_OPT_EXTRAPOLATION, {"freeze": B.PDF_EXTRAP_FREEZE, "error": B.PDF_EXTRAP_ERROR}[mode])
    ref, S = og.xfxq2(spec.pids, x.numpy(), q.numpy(), want_scale=True)
    out = g.pdf_xfxq2(spec.pids, x.cuda(), q.cuda()).cpu().numpy()
    print("\n", mode, path, assert_values(out, ref, S, f"{mode} {path}", strict=1e-12))
    n_nan = int(np.isnan(ref[:, 0]).sum())
    assert g.pdf_error_count() == n_nan
    assert (n_nan > 0.04 * n) if mode == "error" else (n_nan == 0)
    check_locate(B, og, g, x.numpy(), q.numpy())
    # back to the default option: the default numbers
    og.set_extrapolation(oracle_mod.EXTRAP_CONTINUATION)
    g.pdf_grid_set_option(B.PDF_OPT_EXTRAPOLATION, B.PDF_EXTRAP_CONTINUATION)
    ref, S = og.xfxq2(spec.pids, x.numpy()[:50_000], q.numpy()[:50_000], want_scale=True)
    assert_values(g.pdf_xfxq2(spec.pids, x[:50_000].cuda(), q[:50_000].cuda()).cpu().numpy(), ref, S, "default again")


@pytest.mark.parametrize("path", PATHS)
def test_freeze_lumi_and_members(B, oracle_mod, path):
    spec = synth.grid_c1()
    n = 200_000
    x1, x2, qq, w = synth.events_c4(n, seed=31)
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec, path, n)
    og.set_coupling(spec.coupling.numpy())
    og.set_extrapolation(oracle_mod.EXTRAP_FREEZE)
    g.pdf_grid_set_option(B.PDF_OPT_EXTRAPOLATION, B.PDF_EXTRAP_FREEZE)
    ref, S = og.lumi(x1.numpy(), x2.numpy(), qq.numpy(), w.numpy(), want_scale=True)
    out = g.pdf_lumi(x1.cuda(), x2.cuda(), qq.cuda(), w.cuda()).cpu().numpy()
    print("\nlumi freeze", path, assert_values(out, ref, S, "lumi freeze"))
    mspec = synth.grid_c1(nmem=5)
    nm = 300_000
    x, q = synth.queries_c2(mspec, nm, seed=78)
    mem = synth.members(mspec, nm)
    mog = oracle_mod.OracleGrid(mspec.x_knots.numpy(), [k.numpy() for k in mspec.q2_subgrids], mspec.values.numpy(), mspec.pids, nmem=5)
    mog.set_extrapolation(oracle_mod.EXTRAP_FREEZE)
    mg = gpu_grid(B, mspec, path, nm)
    mg.pdf_grid_set_option(B.PDF_OPT_EXTRAPOLATION, B.PDF_EXTRAP_FREEZE)
    ref, S = mog.xfxq2(mspec.pids, x.numpy(), q.numpy(), member=mem.numpy(), want_scale=True)
    out = mg.pdf_xfxq2(mspec.pids, x.cuda(), q.cuda(), member=mem.cuda()).cpu().numpy()
    print("\nmembers freeze", path, assert_values(out, ref, S, "members freeze"))


@pytest.mark.parametrize("path", PATHS)
def test_xfxq_parity(B, oracle_mod, path):
    spec = synth.grid_c1()
    n = 300_000
    x, q2 = synth.queries_c2(spec, n, seed=79)
    Q = torch.sqrt(q2)
    Q[::1000] = -Q[::1000]                      # invalid although the square is not
    Q[1::5000] = 0.0
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec, path, n)
    ref, S = og.xfxq(spec.pids, x.numpy(), Q.numpy(), want_scale=True)
    out = g.pdf_xfxq(spec.pids, x.cuda(), Q.cuda()).cpu().numpy()
    print("\nxfxq", path, assert_values(out, ref, S, f"xfxq {path}", strict=1e-12))
    assert g.pdf_error_count() == int(np.isnan(ref[:, 0]).sum()) > 0


def test_alphas_subgrids_parity(B, oracle_mod):
    """alpha_s knot line with two flavour thresholds (repeated knots, L1835): strict 1e-12 relative against the oracle,
    stored values at every knot (the upper one on a threshold), both below-range modes"""
    spec = synth.grid_c1()
    a = np.exp(np.linspace(0.0, np.log(1e10), 58))
    a = np.sort(np.concatenate([a, a[[9, 23]]]))                       # two repeated knots
    A = 1.0 / (1.0 / 0.35 + (1.0 / 0.08 - 1.0 / 0.35) * (np.arange(60) / 59.0) ** 1.1)
    dup = np.nonzero(a[1:] == a[:-1])[0] + 1
    A[dup[0]:] *= 1.004; A[dup[1]:] *= 0.997                           # a jump at each threshold
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec)
    rng = np.random.default_rng(8)
    q = np.exp(rng.uniform(np.log(0.01), np.log(1e12), 500_000))
    q[: len(a)] = a
    q[len(a): len(a) + 2] = np.nextafter(a[dup], 0.0)
    for mode_o, mode_g in ((oracle_mod.ALPHAS_FREEZE, B.PDF_ALPHAS_FREEZE), (oracle_mod.ALPHAS_LOGGRAD, B.PDF_ALPHAS_LOGGRAD)):
        og.set_alphas(a, A, mode_o)
        g.pdf_grid_set_alphas(torch.tensor(a), torch.tensor(A))
        g.pdf_grid_set_option(B.PDF_OPT_ALPHAS_MODE, mode_g)
        ref = og.alphas_q2(q)
        got = g.pdf_alphas_q2(torch.tensor(q).cuda()).cpu().numpy()
        assert np.max(np.abs(got - ref) / np.abs(ref)) < 1e-12
        exp = A.copy(); exp[dup - 1] = A[dup]
        assert np.array_equal(got[: len(a)], exp)
    with pytest.raises(B.PdfGridError):
        g.pdf_grid_set_alphas(torch.tensor([1.0, 2.0, 2.0, 2.0, 3.0]), torch.tensor([0.3, 0.25, 0.2, 0.15, 0.1]))


@pytest.mark.parametrize("mode", ["freeze", "error"])
def test_extrapolation_options_on_the_shared_point_list(B, oracle_mod, mode):
    """pdf_xfxq2_xgrid (both of its kernels) and pdf_xfxq2_noalloc under the options of L1720"""
    spec = synth.grid_c1(nmem=210)
    og = make_oracle_grid(oracle_mod, spec)
    og.set_extrapolation({"freeze": oracle_mod.EXTRAP_FREEZE, "error": oracle_mod.EXTRAP_ERROR}[mode])
    opt = {"freeze": B.PDF_EXTRAP_FREEZE, "error": B.PDF_EXTRAP_ERROR}[mode]
    npts = 2000
    x, q = synth.queries_c2(spec, npts, seed=91)
    for path, nrep in (("direct", 3), ("auto", 210)):                 # per-point kernel; (member, cell)-shared kernel
        g = gpu_grid(B, spec, path)
        g.pdf_grid_set_option(B.PDF_OPT_EXTRAPOLATION, opt)
        B.pdf_profile_enable(True)
        got = g.pdf_xfxq2_xgrid(spec.pids, x.cuda(), q.cuda(), nrep).cpu().numpy()
        names = [k for k, _ in B.pdf_profile_read(64)]
        B.pdf_profile_enable(False)
        assert names == ["k_xfxq2_xgrid" if path == "direct" else "k_xfxq2_xgrid_cell"], names
        n_bad = 0
        for r in (0, nrep // 2, nrep - 1):
            ref, S = og.xfxq2(spec.pids, x.numpy(), q.numpy(), member=np.full(npts, r, dtype=np.int32), want_scale=True)
            assert_values(got[r], ref, S, f"xgrid {mode} {path} member {r}")
            n_bad = int(np.isnan(ref[:, 0]).sum())
        assert g.pdf_error_count() == n_bad * nrep
        g.close()
    spec1 = synth.grid_c1()
    og1 = make_oracle_grid(oracle_mod, spec1)
    og1.set_extrapolation({"freeze": oracle_mod.EXTRAP_FREEZE, "error": oracle_mod.EXTRAP_ERROR}[mode])
    g = gpu_grid(B, spec1)
    g.pdf_grid_set_option(B.PDF_OPT_EXTRAPOLATION, opt)
    n = 60_000
    x, q = synth.queries_c2(spec1, n, seed=92)
    out = torch.empty((n, 11), dtype=torch.float64, device="cuda")
    g.pdf_xfxq2_noalloc(spec1.pids, x.cuda(), q.cuda(), out)
    ref, S = og1.xfxq2(spec1.pids, x.numpy(), q.numpy(), want_scale=True)
    assert_values(out.cpu().numpy(), ref, S, f"noalloc {mode}")
