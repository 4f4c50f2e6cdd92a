"""Pins of the Monte Carlo oracle (oracle/mc_oracle.c) against what the paper
and the mathematics fix: conservation laws, mass shells, closed phase-space volumes, the closed two-body massive
weight, exact bin volumes, equal-share refinement on closed histograms, hand-worked eq. 1.82-1.83 numbers."""
import math

import numpy as np
import pytest

import oracle as O


@pytest.fixture(scope="module", autouse=True)
def _built():
    O.build()


def minkowski2(p):
    return p[..., 0] ** 2 - (p[..., 1:] ** 2).sum(-1)


@pytest.mark.parametrize("n", [2, 3, 4, 7])
def test_rambo_massless_conservation_and_shells(n):
    """eq. 1.103-1.104, 1.107: sum p_i = P = (sqrt s, 0, 0, 0), p_i^2 = 0, p_i^0 > 0"""
    rng = np.random.default_rng(10 + n)
    u = rng.random((2000, n, 4))
    rs = rng.uniform(50.0, 13000.0, 2000)
    p, w = O.rambo(rs, u)
    tot = p.sum(axis=1)
    # (the invariant mass M of the q's cancels when they are nearly collinear: rounding is amplified by ~ Q^0 / M)
    assert np.max(np.abs(tot[:, 0] - rs) / rs) < 1e-10
    assert np.max(np.abs(tot[:, 1:]) / rs[:, None]) < 1e-10
    assert np.median(np.abs(tot[:, 0] - rs) / rs) < 1e-15
    assert np.max(np.abs(minkowski2(p)) / rs[:, None] ** 2) < 1e-10
    assert np.all(p[..., 0] > 0)
    # eq. 1.108: the weight is flat (depends on s and n only)
    w0 = np.array([O.rambo_w0(n, s * s) for s in rs])
    assert np.max(np.abs(w / w0 - 1)) < 1e-14


def test_rambo_w0_closed_volumes():
    """eq. 1.108 against the textbook massless phase-space volumes: Phi_2 = 1/(8 pi), Phi_3 = s/(256 pi^3),
    Phi_4 = s^2/(24576 pi^5)"""
    s = 1234.5 ** 2
    assert abs(O.rambo_w0(2, s) * 8 * math.pi - 1) < 1e-14
    assert abs(O.rambo_w0(3, s) / (s / (256 * math.pi ** 3)) - 1) < 1e-14
    assert abs(O.rambo_w0(4, s) / (s * s / (24576 * math.pi ** 5)) - 1) < 1e-14


def test_rambo_two_body_massive_weight_closed_form():
    """n = 2, masses m1, m2: eq. 1.109-1.110 must give the exact two-body volume sqrt(lambda(s, m1^2, m2^2)) / (8 pi s)
    for EVERY event, |k| = sqrt(lambda)/(2 sqrt s), and k_i^2 = m_i^2, sum k = P"""
    rng = np.random.default_rng(3)
    u = rng.random((500, 2, 4))
    rs, m1, m2 = 500.0, 173.0, 80.4
    p, w = O.rambo(rs, u, masses=[m1, m2])
    s = rs * rs
    lam = (s - m1 * m1 - m2 * m2) ** 2 - 4 * m1 * m1 * m2 * m2
    r = np.abs(w / (math.sqrt(lam) / (8 * math.pi * s)) - 1)
    assert np.max(r) < 1e-10 and np.median(r) < 1e-15          # (conditioning of M for nearly collinear q's)
    kabs = np.sqrt((p[..., 1:] ** 2).sum(-1))
    assert np.max(np.abs(kabs / (math.sqrt(lam) / (2 * rs)) - 1)) < 1e-10
    assert np.max(np.abs(np.sqrt(minkowski2(p)) - np.array([m1, m2]))) < 1e-7
    tot = p.sum(axis=1)
    assert np.max(np.abs(tot - np.array([rs, 0, 0, 0]))) < 1e-7


def test_rambo_massive_many_body():
    """n = 4 with two massive particles: mass shells, energy conservation (the xi constraint below eq. 1.109), the
    massless limit w_m -> 1, and the Monte Carlo mean of w against the massless volume within its error for tiny masses"""
    rng = np.random.default_rng(4)
    u = rng.random((4000, 4, 4))
    m = np.array([173.0, 173.0, 0.0, 0.0])
    rs = 1000.0
    p, w = O.rambo(rs, u, masses=m)
    assert np.max(np.abs(minkowski2(p) - m ** 2) / rs ** 2) < 1e-10
    tot = p.sum(axis=1)
    assert np.max(np.abs(tot[:, 0] - rs)) < 1e-7 and np.max(np.abs(tot[:, 1:])) < 1e-7
    assert np.all(w > 0) and np.all(w < O.rambo_w0(4, rs * rs))          # massive phase space is smaller, point by point
    p0, w0 = O.rambo(rs, u, masses=[1e-9, 1e-9, 0.0, 0.0])
    assert np.max(np.abs(w0 / O.rambo_w0(4, rs * rs) - 1)) < 1e-10
    pm, _ = O.rambo(rs, u)
    assert np.max(np.abs(p0 - pm)) < 1e-7


def test_rambo_pt_cut_and_isotropy():
    rng = np.random.default_rng(5)
    u = rng.random((20000, 3, 4))
    p, w = O.rambo(200.0, u, ptmin=30.0)
    pt = np.sqrt(p[..., 1] ** 2 + p[..., 2] ** 2)
    cut = (pt < 30.0).any(axis=1)
    assert cut.any() and (~cut).any()
    assert np.all(w[cut] == 0.0) and np.all(w[~cut] == O.rambo_w0(3, 4e4))
    # isotropic: every momentum component averages to 0 within 5 sigma
    for k in (1, 2, 3):
        v = p[:, 0, k]
        assert abs(v.mean()) < 5 * v.std() / math.sqrt(len(v))


def test_vegas_map_uniform_grid_is_identity():
    edges = np.tile(np.linspace(0.0, 1.0, 11), (3, 1))
    u = np.random.default_rng(6).random((1000, 3))
    x, jac, b = O.vegas_map(edges, u)
    assert np.max(np.abs(x - u)) < 1e-15 and np.max(np.abs(jac - 1)) < 1e-14
    assert np.array_equal(b, np.floor(u * 10).astype(np.int32))


def test_vegas_map_jacobian_is_bin_volume():
    """1/p(x) = prod_d nb * width_d(bin): the separable piecewise-constant density of eq. 1.81; its integral is 1"""
    rng = np.random.default_rng(7)
    nb, ndim = 8, 2
    edges = np.sort(np.concatenate([np.zeros((ndim, 1)), rng.random((ndim, nb - 1)), np.ones((ndim, 1))], axis=1), axis=1)
    edges[1] = 2.0 + 3.0 * edges[1]                                   # a dimension on [2, 5]
    u = rng.random((200000, ndim))
    x, jac, b = O.vegas_map(edges, u)
    for d in range(ndim):
        w = np.diff(edges[d])
        assert np.all(x[:, d] >= edges[d][b[:, d]]) and np.all(x[:, d] <= edges[d][b[:, d] + 1])
    want = nb * np.diff(edges[0])[b[:, 0]] * nb * np.diff(edges[1])[b[:, 1]]
    assert np.max(np.abs(jac / want - 1)) < 1e-14
    # E[jac] = volume of the domain (integral of 1): 1 * 3
    assert abs(jac.mean() - 3.0) < 5 * jac.std() / math.sqrt(len(jac))
    # importance sampling identity (eq. 1.73-1.74) on f = x0 * x1: integral = 1/2 * (25 - 4)/2
    sums, hist = O.vegas_accumulate(nb, x[:, 0] * x[:, 1], jac, b)
    E, var = O.vegas_estimate(len(jac), sums)
    assert abs(E - 0.5 * 10.5) < 5 * math.sqrt(var)
    assert abs(hist.sum(axis=1)[0] - hist.sum(axis=1)[1]) < 1e-9 * hist.sum()     # every point is in one bin per dimension


def test_vegas_accumulate_and_estimate_hand_worked():
    f = np.array([1.0, -2.0, 3.0, 4.0])
    jac = np.array([2.0, 1.0, 1.0, 0.5])
    bins = np.array([[0], [1], [1], [0]], dtype=np.int32)
    sums, hist = O.vegas_accumulate(2, f, jac, bins)
    assert sums.tolist() == [2.0 - 2.0 + 3.0 + 2.0, 4.0 + 4.0 + 9.0 + 4.0]
    assert hist.tolist() == [[4.0, 5.0]]
    E, var = O.vegas_estimate(4, sums)
    assert E == 1.25 and abs(var - (21.0 / 4 - 1.25 ** 2) / 3) < 1e-15


def test_vegas_refine_equal_shares():
    """a histogram concentrated in one old bin: the new edges put nb equal shares of it; a flat histogram leaves a uniform
    grid unchanged; the end points never move"""
    nb = 4
    edges = np.array([[0.0, 0.25, 0.5, 0.75, 1.0]])
    flat = O.vegas_refine(np.array([[1.0, 1.0, 1.0, 1.0]]), edges)
    assert np.max(np.abs(flat - edges)) < 1e-15
    new = O.vegas_refine(np.array([[0.0, 8.0, 0.0, 0.0]]), edges)
    assert np.allclose(new, [[0.0, 0.25 + 0.0625, 0.375, 0.4375, 1.0]], atol=1e-15)
    # shares 1:3 over two halves of [0,1]: cumulative distribution is piecewise linear, quartiles at 0.5, 2/3, 5/6
    new = O.vegas_refine(np.array([[1.0, 3.0]]), np.array([[0.0, 0.5, 1.0]]))
    assert new.shape == (1, 3) and abs(new[0, 1] - (0.5 + 0.5 / 3)) < 1e-15
    # damping: alpha = 0 ignores the histogram (equal widths of the OLD bins are kept)
    new = O.vegas_refine(np.array([[0.0, 8.0, 1.0, 1.0]]), edges, alpha=0.0)
    assert np.max(np.abs(new - edges)) < 1e-15


def test_vegas_refinement_reduces_variance():
    """exploration phase (L917): iterating map -> accumulate -> refine on a peaked integrand shrinks the variance of the
    estimate and keeps the estimate consistent with the exact integral (Gaussian peak: closed form with erf)"""
    rng = np.random.default_rng(8)
    nb, n = 50, 20000
    edges = np.tile(np.linspace(0.0, 1.0, nb + 1), (2, 1))
    sig = 0.05
    exact = (math.sqrt(2 * math.pi) * sig * math.erf(0.5 / (sig * math.sqrt(2)))) ** 2
    Es, Vs = [], []
    for it in range(6):
        x, jac, b = O.vegas_map(edges, rng.random((n, 2)))
        f = np.exp(-((x - 0.5) ** 2).sum(axis=1) / (2 * sig * sig))
        sums, hist = O.vegas_accumulate(nb, f, jac, b)
        E, var = O.vegas_estimate(n, sums)
        Es.append(E); Vs.append(var)
        edges = O.vegas_refine(hist, edges)
    assert Vs[-1] < 0.1 * Vs[0]
    Ebar, S2bar, chi2 = O.vegas_combine(Es[2:], Vs[2:])
    assert abs(Ebar - exact) < 5 * math.sqrt(S2bar) and chi2 < 5


def test_vegas_combine_hand_worked():
    """eq. 1.82-1.83 on numbers worked by hand: E = (10, 12), S^2 = (1, 4): 1/S^2 = 1.25, Ebar = 0.8 (10 + 3) = 10.4,
    chi2/dof = (0.16/1 + 2.56/4)/1 = 0.8"""
    Ebar, S2bar, chi2 = O.vegas_combine([10.0, 12.0], [1.0, 4.0])
    assert abs(S2bar - 0.8) < 1e-15 and abs(Ebar - 10.4) < 1e-14 and abs(chi2 - 0.8) < 1e-13
    Ebar, S2bar, chi2 = O.vegas_combine([3.0], [2.0])
    assert Ebar == 3.0 and S2bar == 2.0 and chi2 == 0.0


def test_unweight_rule():
    """L2028-2030: accepted iff w > u * w_max; acceptance probability w / w_max"""
    w = np.array([1.0, 4.0, 2.0, 0.0])
    u = np.array([0.3, 0.999, 0.5, 0.0])
    wmax, acc, cnt = O.unweight(w, u)
    assert wmax == 4.0 and acc.tolist() == [False, True, False, False] and cnt == 1
    rng = np.random.default_rng(9)
    w = rng.random(200000) ** 3
    wmax, acc, cnt = O.unweight(w, rng.random(w.size))
    assert abs(cnt / w.size - w.mean() / wmax) < 5 * math.sqrt(0.25 / w.size)


def test_rambo_closed_threshold():
    """reading R-6: sqrt s <= sum m has no phase space (weight 0, zero momenta); just above it the two-body weight
    sqrt(lambda)/(8 pi s) tends to 0 continuously, so the case joins on without a jump"""
    rng = np.random.default_rng(8)
    u = rng.random((64, 2, 4))
    m = [173.0, 173.0]
    rs = np.full(64, 346.0); rs[::2] = 300.0; rs[1::4] = 346.0 * (1 + 1e-9)
    p, w = O.rambo(rs, u, masses=m)
    closed = rs <= 346.0
    assert np.all(w[closed] == 0.0) and np.all(p[closed] == 0.0)
    s = rs[~closed] ** 2
    lam = (s - 4 * 173.0 ** 2) * s
    assert np.all(w[~closed] > 0) and np.allclose(w[~closed], np.sqrt(lam) / (8 * np.pi * s), rtol=1e-6)
    assert np.all(np.isfinite(p)) and w[~closed].max() < 1e-5
