"""Parity of the Monte Carlo steps around the hot path through the C ABI against
the CPU oracle (oracle/mc_oracle.c) on the same seeded uniforms.  Momenta, weights, points and jacobians element by
element (1e-12 relative; momenta to 1e-12 of sqrt s where a component cancels); bin indices and acceptance flags
bit-exact; sums within 1e-12 of the sum of magnitudes (the GPU adds in a different order)."""
import math

import numpy as np
import pytest
import torch

import oracle as O

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2302_03343_b200 import binding
    assert torch.cuda.is_available()
    binding.lib()
    O.build()
    return binding


def uniforms(shape, seed):
    g = torch.Generator().manual_seed(seed)
    return torch.rand(shape, generator=g, dtype=torch.float64).clamp_(min=1e-300)


def collinearity(u):
    """the two condition numbers of eq. 1.107 / 1.103 as functions of the uniforms: (Q0 / M)^2 for the invariant mass M,
    and 1 / sin(theta) for sin = sqrt(1 - c^2) near the poles (c * c rounds once on the CPU, not at all in an FMA)"""
    c, phi, q0 = 2 * u[..., 0] - 1, 2 * np.pi * u[..., 1], -np.log(u[..., 2] * u[..., 3])
    st = np.sqrt(1 - c * c)
    Q = np.stack([q0, q0 * st * np.cos(phi), q0 * st * np.sin(phi), q0 * c], axis=-1).sum(axis=1)
    return Q[:, 0] ** 2 / (Q[:, 0] ** 2 - (Q[:, 1:] ** 2).sum(axis=1)) + (1.0 / st).max(axis=1)


@pytest.mark.parametrize("n,masses", [(2, None), (3, None), (4, [173.0, 173.0, 0.0, 0.0]), (6, [80.4, 91.2, 0, 0, 4.7, 4.7])])
def test_rambo_parity(B, n, masses):
    nev = 200_003                                   # several CTAs and a ragged tail
    u = uniforms((nev, n, 4), 100 + n)
    rs = 200.0 + 12800.0 * uniforms((nev,), 7)
    p_ref, w_ref = O.rambo(rs.numpy(), u.numpy(), masses=masses, ptmin=30.0)
    p, w = B.pdf_rambo(rs.cuda(), u.cuda(), masses=masses, ptmin=30.0)
    p, w = p.cpu().numpy(), w.cpu().numpy()
    # a p_T within rounding of the cut may fall on either side: those events are compared without the cut
    pt = np.sqrt(p_ref[..., 1] ** 2 + p_ref[..., 2] ** 2)
    edge = (np.abs(pt - 30.0) < 1e-9).any(axis=1)
    assert edge.sum() < 5
    # Conditioning of the input, not of either implementation: nearly collinear q's cancel in the invariant mass
    # M^2 = Q0^2 - |Q|^2 of eq. 1.103, whose rounding enters every momentum as dM/M ~ eps (Q0/M)^2.  The bound is
    # 64 eps ((Q0/M)^2 + max 1/sin theta_i) of sqrt s per component (different log / sincos roundings upstream of the cancellation).
    cond = collinearity(u.numpy())
    eps = 2.0 ** -52
    bound = 64 * eps * cond
    err = np.abs(p - p_ref) / rs.numpy()[:, None, None]
    ratio = (err / bound[:, None, None]).max()
    print(f"rambo n={n}: median err {np.median(err):.2e} of sqrt s, max {err.max():.2e}, worst err/bound {ratio:.3f}, "
          f"max (Q0/M)^2 {cond.max():.2e}")
    assert np.median(err) < 1e-15 and ratio <= 1.0
    well = cond < 100.0                               # the bulk: plain 1e-12
    assert well.mean() > 0.9 and err[well].max() < 1e-12
    ok = ~edge
    assert np.array_equal(w[ok] == 0.0, w_ref[ok] == 0.0)
    nz = ok & (w_ref != 0.0)
    rel = np.abs(w[nz] / w_ref[nz] - 1)
    assert np.all(rel <= 4 * n * bound[nz]) and rel[well[nz]].max() < 1e-12
    assert (w_ref == 0).any() and (w_ref != 0).any()


def test_rambo_edge_cases(B):
    u = uniforms((5, 3, 4), 1)
    rs = torch.full((5,), 100.0, dtype=torch.float64)
    p, w = B.pdf_rambo(rs[:0].cuda(), u[:0].cuda())
    assert p.shape == (0, 3, 4) and w.numel() == 0
    with pytest.raises(B.PdfGridError):
        B.pdf_rambo(rs.cuda(), uniforms((5, 1, 4), 2).cuda())          # one final-state particle: no phase space
    with pytest.raises(B.PdfGridError):
        B.pdf_rambo(rs.cuda(), u.cuda(), masses=[1.0, -2.0, 0.0])
    p, w = B.pdf_rambo(rs.cuda(), u.cuda(), masses=[0.0, 0.0, 0.0])      # all-zero masses = the massless weight
    assert torch.allclose(w.cpu(), torch.full((5,), O.rambo_w0(3, 1e4), dtype=torch.float64), rtol=1e-14)


def test_vegas_step_parity(B):
    """one full importance-sampling iteration: map -> integrand -> accumulate -> estimate -> refine, then eq. 1.82-1.83"""
    ndim, nb, n = 4, 50, 500_009
    rng = np.random.default_rng(3)
    edges = np.sort(np.concatenate([np.zeros((ndim, 1)), rng.random((ndim, nb - 1)), np.ones((ndim, 1))], axis=1), axis=1)
    edges[2] = -3.0 + 7.0 * edges[2]
    u = uniforms((n, ndim), 11)
    x_ref, jac_ref, bin_ref = O.vegas_map(edges, u.numpy())
    ed = torch.tensor(edges).cuda()
    x, jac, bins = B.pdf_vegas_map(ed, u.cuda())
    assert np.array_equal(bins.cpu().numpy(), bin_ref)
    # x = e_k + (y - k)(e_{k+1} - e_k) cancels near x = 0 where an axis spans it: the error is eps of the edge, not of x
    emax = np.abs(edges).max(axis=1)[None, :]
    assert np.max(np.abs(x.cpu().numpy() - x_ref) / emax) < 4 * 2.0 ** -52
    assert np.max(np.abs(jac.cpu().numpy() / jac_ref - 1)) < 1e-13
    f = torch.cos(3.0 * x).prod(dim=1) + 0.1                                  # a signed integrand, computed once, used by both
    sums_ref, hist_ref = O.vegas_accumulate(nb, f.cpu().numpy(), jac.cpu().numpy(), bin_ref)
    sums, hist = B.pdf_vegas_accumulate(nb, f, jac, bins)
    mag = float((f * jac).abs().sum())
    assert abs(float(sums[0]) - sums_ref[0]) < 1e-12 * mag
    assert abs(float(sums[1]) / sums_ref[1] - 1) < 1e-12
    assert np.max(np.abs(hist.cpu().numpy() / hist_ref - 1)) < 1e-12
    res = B.pdf_vegas_estimate(n, sums).cpu().numpy()
    E_ref, var_ref = O.vegas_estimate(n, sums.cpu().numpy())
    assert abs(res[0] - E_ref) <= 1e-15 * abs(E_ref) + 1e-300 and abs(res[1] / var_ref - 1) < 1e-13
    for alpha in (1.0, 0.5):
        new_ref = O.vegas_refine(hist.cpu().numpy(), edges, alpha=alpha)
        new = B.pdf_vegas_refine(hist, ed.clone(), alpha=alpha).cpu().numpy()
        assert np.max(np.abs(new - new_ref)) < 1e-13
        assert np.all(np.diff(new, axis=1) > 0) and np.array_equal(new[:, [0, -1]], edges[:, [0, -1]])
    E = torch.tensor([10.0, 12.0, 11.0], dtype=torch.float64)
    S2 = torch.tensor([1.0, 4.0, 0.25], dtype=torch.float64)
    got = B.pdf_vegas_combine(E.cuda(), S2.cuda()).cpu().numpy()
    want = O.vegas_combine(E.numpy(), S2.numpy())
    assert np.max(np.abs(got - np.array(want))) < 1e-13


def test_vegas_loop_converges_on_the_device(B):
    """exploration + evaluation phases (L917) entirely through the C ABI: a peaked 2-D Gaussian, closed-form integral"""
    nb, n, sig = 64, 200_000, 0.04
    ed = torch.linspace(0.0, 1.0, nb + 1, dtype=torch.float64).repeat(2, 1).cuda()
    exact = (math.sqrt(2 * math.pi) * sig * math.erf(0.5 / (sig * math.sqrt(2)))) ** 2
    Es, Vs = [], []
    for it in range(8):
        x, jac, bins = B.pdf_vegas_map(ed, uniforms((n, 2), 50 + it).cuda())
        f = torch.exp(-((x - 0.5) ** 2).sum(dim=1) / (2 * sig * sig))
        sums, hist = B.pdf_vegas_accumulate(nb, f, jac, bins)
        res = B.pdf_vegas_estimate(n, sums).cpu()
        Es.append(float(res[0])); Vs.append(float(res[1]))
        if it < 4:
            B.pdf_vegas_refine(hist, ed)
    assert Vs[-1] < 0.05 * Vs[0]
    out = B.pdf_vegas_combine(torch.tensor(Es[4:], dtype=torch.float64).cuda(), torch.tensor(Vs[4:], dtype=torch.float64).cuda()).cpu()
    assert abs(float(out[0]) - exact) < 5 * math.sqrt(float(out[1])) and float(out[2]) < 5


def test_unweight_parity(B):
    n = 1_000_003
    w = uniforms((n,), 21) ** 3
    w[::7] = 0.0
    u = uniforms((n,), 22)
    wmax_ref, acc_ref, cnt_ref = O.unweight(w.numpy(), u.numpy())
    wmax, acc, cnt = B.pdf_unweight(w.cuda(), u.cuda())
    assert wmax == wmax_ref and cnt == cnt_ref and np.array_equal(acc.cpu().numpy(), acc_ref)
    wmax, acc, cnt = B.pdf_unweight(w[:0].cuda(), u[:0].cuda())
    assert cnt == 0 and wmax == 0.0


def test_mc_chain_feeds_the_luminosity(B, oracle_mod):
    """RAMBO weights x the luminosity (eq. 4.1, Fig. 4.1): VEGAS-mapped (x1, x2) -> Q2 = x1 x2 s -> pdf_lumi with the
    phase-space weight as the event weight, against the oracle chain on the same uniforms"""
    from paper_2302_03343_b200 import synth
    from conftest import make_oracle_grid
    spec = synth.grid_c1()
    og = make_oracle_grid(oracle_mod, spec)
    g = B.PdfGrid.from_spec(spec, workspace_for=100_000)
    n, nb = 100_000, 20
    edges = np.tile(np.linspace(math.log(1e-6), 0.0, nb + 1), (2, 1))
    u = uniforms((n, 2), 31)
    lx, jac, bins = B.pdf_vegas_map(torch.tensor(edges).cuda(), u.cuda())
    x12 = torch.exp(lx)
    s = 13000.0 ** 2
    q2 = (x12[:, 0] * x12[:, 1]) * s
    ur = uniforms((n, 2, 4), 32)
    p, wps = B.pdf_rambo(torch.sqrt(q2), ur.cuda(), masses=[173.0, 173.0])
    ok = torch.sqrt(q2) > 2 * 173.0 + 1.0
    wev = torch.where(ok, wps, torch.zeros_like(wps)).nan_to_num()
    lum = g.pdf_lumi(x12[:, 0].contiguous(), x12[:, 1].contiguous(), q2.contiguous(), wev.contiguous())
    lx_ref, jac_ref, _ = O.vegas_map(edges, u.numpy())
    x_ref = np.exp(lx_ref)
    q_ref = (x_ref[:, 0] * x_ref[:, 1]) * s
    okr = np.sqrt(q_ref) > 2 * 173.0 + 1.0
    assert np.array_equal(okr, ok.cpu().numpy())
    with np.errstate(invalid="ignore"):
        _, w_ref = O.rambo(np.sqrt(q_ref), ur.numpy(), masses=[173.0, 173.0])
    w_ref = np.where(okr, np.nan_to_num(w_ref), 0.0)
    ref, S = og.lumi(x_ref[:, 0].copy(), x_ref[:, 1].copy(), q_ref, w_ref, want_scale=True)
    tol = oracle_mod.tolerance(ref, S) + 1e-11 * np.abs(ref)               # + the conditioning of exp(), sqrt() and M upstream
    assert np.all(np.abs(lum.cpu().numpy() - ref) <= tol)
    assert okr.sum() > 1000
