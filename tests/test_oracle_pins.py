"""Pins of the CPU oracle against things OTHER than itself (no GPU needed).

Each test names the pin (P-n of DESIGN.md) and the passage of PAPER.md it fixes.
Expected values come from closed forms, hand-worked fixtures under tests/golden/,
textbook special cases, or a literal second implementation written here in numpy
in a different form (monomial coefficients, explicit slope arrays).
"""
import math
import os

import numpy as np
import pytest
import torch

from paper_2302_03343_b200 import synth
from conftest import make_oracle_grid

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------------------
# helpers: custom grids
# ---------------------------------------------------------------------------
def spec_from_function(x, subs, fun, nflav=1):
    """values[ix][iq][f] = fun(ln x, ln Q2, f, k) on every sub-grid."""
    blocks = []
    for k, q in enumerate(subs):
        U, S = np.meshgrid(np.log(x), np.log(q), indexing="ij")
        v = np.stack([fun(U, S, f, k) for f in range(nflav)], axis=-1)
        blocks.append(v.reshape(-1))
    return synth.GridSpec(torch.tensor(np.asarray(x, dtype=np.float64)),
                          [torch.tensor(np.asarray(q, dtype=np.float64)) for q in subs],
                          torch.tensor(np.concatenate(blocks)), pids=tuple(range(1, nflav + 1)))


def uniform_log_knots(lo, hi, n):
    k = np.exp(np.linspace(math.log(lo), math.log(hi), n))
    k[0], k[-1] = lo, hi
    return k


# ---------------------------------------------------------------------------
# literal second implementation (P-11): slopes -> monomial cubic -> Horner
# ---------------------------------------------------------------------------
def brute_slopes(w, v):
    m = len(w)
    s = np.empty(m)
    for c in range(m):
        if c == 0:
            s[c] = (v[1] - v[0]) / (w[1] - w[0])
        elif c == m - 1:
            s[c] = (v[m - 1] - v[m - 2]) / (w[m - 1] - w[m - 2])
        else:
            s[c] = ((v[c + 1] - v[c]) / (w[c + 1] - w[c]) + (v[c] - v[c - 1]) / (w[c] - w[c - 1])) / 2
    return s


def brute_line(w, v, wpt, c):
    """piecewise cubic through (w, v) with slopes s, in monomial form in t"""
    s = brute_slopes(w, v)
    d = w[c + 1] - w[c]
    t = (wpt - w[c]) / d
    a0 = v[c]
    a1 = d * s[c]
    a2 = 3 * (v[c + 1] - v[c]) - 2 * d * s[c] - d * s[c + 1]
    a3 = 2 * (v[c] - v[c + 1]) + d * s[c] + d * s[c + 1]
    return a0 + t * (a1 + t * (a2 + t * a3))


def brute_cell(knots, v):
    c = 0
    for i in range(len(knots) - 1):
        if knots[i] <= v:
            c = i
    return c


def brute_interior(spec, x, q2, f, mem=0):
    xk = spec.x_knots.numpy()
    k = 0
    for kk, q in enumerate(spec.q2_subgrids):
        if float(q[0]) <= q2:
            k = kk
    qk = spec.q2_subgrids[k].numpy()
    V = spec.block(mem, k).numpy()[:, :, f]
    i, j = brute_cell(xk, x), brute_cell(qk, q2)
    rows = np.array([brute_line(np.log(xk), V[:, b], math.log(x), i) for b in range(len(qk))])
    return brute_line(np.log(qk), rows, math.log(q2), j)


# ---------------------------------------------------------------------------
# P-1 node reproduction (bitwise), incl. last x knot, Q2max, thresholds (upper copy)
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("which", ["c0", "c1"])
def test_p1_nodes_bitwise(oracle_mod, which):
    spec = synth.grid_c0() if which == "c0" else synth.grid_c1()
    g = make_oracle_grid(oracle_mod, spec)
    nsub = len(spec.q2_subgrids)
    for k, qk in enumerate(spec.q2_subgrids):
        X, Q = torch.meshgrid(spec.x_knots, qk, indexing="ij")
        out = g.xfxq2(spec.pids, X.reshape(-1).numpy(), Q.reshape(-1).numpy())
        want = spec.block(0, k).numpy().reshape(-1, spec.nflav).copy()
        got = out.reshape(spec.nx, len(qk), spec.nflav)
        want = want.reshape(spec.nx, len(qk), spec.nflav)
        # the top knot of sub-grid k < K-1 is a threshold: the query belongs to the UPPER sub-grid (S-6)
        top = len(qk) - 1 if k < nsub - 1 else len(qk)
        assert np.array_equal(got[:, :top], want[:, :top])
        if k < nsub - 1:
            upper = spec.block(0, k + 1).numpy()[:, 0, :]
            assert np.array_equal(got[:, -1], upper)


def test_p1_locate_at_nodes_and_neighbours(oracle_mod):
    """C-3/C-4/S-6: knot -> cell on its right (last knot -> last cell); threshold -> upper sub-grid;
    index flips between nextafter(thr, -inf) and thr."""
    spec = synth.grid_c1()
    g = make_oracle_grid(oracle_mod, spec)
    xk = spec.x_knots.numpy()
    q_mid = np.full_like(xk, 50.0)
    ix, iq, isub, reg = g.locate(xk, q_mid)
    assert np.array_equal(ix, np.minimum(np.arange(len(xk)), len(xk) - 2))
    ix2, *_ = g.locate(np.nextafter(xk[1:], 0.0), q_mid[1:])
    assert np.array_equal(ix2, np.arange(len(xk) - 1))
    off = 0
    for k, qk in enumerate(spec.q2_subgrids):
        qk = qk.numpy()
        xs = np.full_like(qk, 1e-3)
        _, iq, isub, reg = g.locate(xs, qk)
        exp_sub = np.full(len(qk), k)
        exp_iq = np.minimum(np.arange(len(qk)), len(qk) - 2)
        if k < len(spec.q2_subgrids) - 1:
            exp_sub[-1], exp_iq[-1] = k + 1, 0
        assert np.array_equal(isub, exp_sub) and np.array_equal(iq, exp_iq)
        assert np.all(reg == 0)
        if k > 0:
            _, iqb, isubb, _ = g.locate(xs[:1], np.nextafter(qk[:1], 0.0))
            assert isubb[0] == k - 1 and iqb[0] == len(spec.q2_subgrids[k - 1]) - 2
        off += len(qk)


def test_region_classes(oracle_mod):
    spec = synth.grid_c1()
    g = make_oracle_grid(oracle_mod, spec)
    x = np.array([1e-3, 1e-10, 1e-3, 1e-3, 1e-10, 1e-10, 1.5, -1.0, 0.0, 1e-3, 1e-3, np.nan, 1.0, 1e-9])
    q = np.array([10.0, 10.0, 0.5, 1e11, 0.5, 1e11, 10.0, 10.0, 10.0, 0.0, np.inf, 10.0, 1e10, 1.0])
    ix, iq, isub, reg = g.locate(x, q)
    assert list(reg) == [0, 1, 2, 3, 4, 5, 6, 6, 6, 6, 6, 6, 0, 0]
    out = g.xfxq2(spec.pids, x, q)
    assert np.all(np.isnan(out[reg == 6])) and not np.any(np.isnan(out[reg != 6]))
    assert np.all(ix[reg == 6] == -1)
    # anchors of the extrapolation regions
    assert ix[1] == 0 and iq[2] == 0 and isub[2] == 0
    assert isub[3] == 2 and iq[3] == 38


# ---------------------------------------------------------------------------
# P-2 / P-3: constants and functions linear in (ln x, ln Q2) are reproduced
# ---------------------------------------------------------------------------
def test_p2_p3_bilinear_reproduction(oracle_mod):
    rng = np.random.default_rng(5)
    spec0 = synth.tiny_grid(11, 7, [4, 3, 6])
    x, subs = spec0.x_knots.numpy(), [q.numpy() for q in spec0.q2_subgrids]
    al, be, ga, de = 0.7, -0.31, 0.23, 0.045
    spec = spec_from_function(x, subs, lambda U, S, f, k: al + be * U + ga * S + de * U * S + 0 * f)
    g = make_oracle_grid(oracle_mod, spec)
    n = 4000
    xs = np.exp(rng.uniform(math.log(x[0]), math.log(x[-1]), n)).clip(x[0], x[-1])
    qs = np.exp(rng.uniform(math.log(subs[0][0]), math.log(subs[-1][-1]), n)).clip(subs[0][0], subs[-1][-1])
    out = g.xfxq2(spec.pids, xs, qs)[:, 0]
    want = al + be * np.log(xs) + ga * np.log(qs) + de * np.log(xs) * np.log(qs)
    assert np.max(np.abs(out - want)) < 1e-14 * np.max(np.abs(spec.values.numpy())) * 10
    const = spec_from_function(x, subs, lambda U, S, f, k: 0 * U + 3.25)
    gc = make_oracle_grid(oracle_mod, const)
    assert np.max(np.abs(gc.xfxq2(const.pids, xs, qs) - 3.25)) < 4 * 3.25 * 2.3e-16


# ---------------------------------------------------------------------------
# P-4: closed form on uniform log knots = Catmull-Rom (golden fixture, hand-worked)
# ---------------------------------------------------------------------------
def _read_weight_fixture():
    rows = []
    for line in open(os.path.join(GOLD, "hermite_uniform_weights.txt")):
        if line.startswith("#") or not line.strip():
            continue
        p = line.split()
        rows.append((p[0], float(p[1]), [float(v) for v in p[2:6]]))
    return rows


def test_p4_catmull_rom_weights_fixture(oracle_mod):
    knots = np.arange(6, dtype=np.float64) * 0.5 - 1.0
    for case, t, want in _read_weight_fixture():
        if case == "interior":
            m, c, kn = 6, 2, knots
        elif case == "left_end":
            m, c, kn = 6, 0, knots
        elif case == "right_end":
            m, c, kn = 6, 4, knots
        else:
            m, c, kn = 2, 0, knots[:2]
        w = oracle_mod.weights_1d(kn[:m], kn[c] + t * (kn[c + 1] - kn[c]), c)
        assert np.max(np.abs(w - np.array(want))) < 1e-15, (case, t, w)
        assert abs(w.sum() - 1.0) < 1e-15


def test_p4_catmull_rom_polynomial_everywhere(oracle_mod):
    knots = np.linspace(-3.0, 2.0, 11)
    for t in np.linspace(0, 1, 21):
        w = oracle_mod.weights_1d(knots, knots[4] + t * 0.5, 4)
        cr = 0.5 * np.array([-t**3 + 2 * t**2 - t, 3 * t**3 - 5 * t**2 + 2, -3 * t**3 + 4 * t**2 + t, t**3 - t**2])
        assert np.max(np.abs(w - cr)) < 1e-15


def test_p4_2d_midpoint_tensor_product(oracle_mod):
    """C0 is log-uniform on both axes: the mid-cell value is the tensor product of (-1,9,9,-1)/16."""
    spec = synth.grid_c0()
    g = make_oracle_grid(oracle_mod, spec)
    u, s = np.log(spec.x_knots.numpy()), np.log(spec.q2_subgrids[0].numpy())
    V = spec.block(0, 0).numpy()
    w = np.array([-1, 9, 9, -1]) / 16.0
    for (i, j) in [(5, 7), (20, 3), (40, 25), (1, 1), (47, 27)]:
        xm, qm = math.exp(0.5 * (u[i] + u[i + 1])), math.exp(0.5 * (s[j] + s[j + 1]))
        out = g.xfxq2(spec.pids, [xm], [qm])[0]
        want = np.einsum("a,b,abf->f", w, w, V[i - 1:i + 3, j - 1:j + 3, :])
        scale = np.einsum("a,b,abf->f", abs(w), abs(w), abs(V[i - 1:i + 3, j - 1:j + 3, :]))
        # exp/log round trip moves t by ~1e-14: tolerance on the value, relative to the stencil scale
        assert np.max(np.abs(out - want) / scale) < 2e-13


# ---------------------------------------------------------------------------
# S-2: interior slope = PLAIN average of the two secants (not spacing weighted)
# ---------------------------------------------------------------------------
def test_s2_plain_average_slope_on_nonuniform_knots(oracle_mod):
    w = np.array([0.0, 1.0, 3.0, 3.5, 6.0])
    v = w ** 2
    c, t = 1, 0.4
    # secants of w^2 are sums of neighbouring knots
    m1 = 0.5 * ((w[2] + w[1]) + (w[1] + w[0]))
    m2 = 0.5 * ((w[3] + w[2]) + (w[2] + w[1]))
    d = w[2] - w[1]
    h00, h10, h01, h11 = 2 * t**3 - 3 * t**2 + 1, t**3 - 2 * t**2 + t, -2 * t**3 + 3 * t**2, t**3 - t**2
    want = h00 * v[1] + h10 * d * m1 + h01 * v[2] + h11 * d * m2
    got = float(np.dot(oracle_mod.weights_1d(w, w[1] + t * d, c), v[0:4]))
    assert abs(got - want) < 1e-14
    # the spacing-weighted three-point rule would reproduce w^2 exactly; the plain average does not
    assert abs(got - (w[1] + t * d) ** 2) > 1e-3


# ---------------------------------------------------------------------------
# P-5: quadratics exact in interior cells of uniform knots
# ---------------------------------------------------------------------------
def test_p5_quadratic_exact_on_uniform_interior(oracle_mod):
    x = uniform_log_knots(1e-4, 1.0, 12)
    q = uniform_log_knots(2.0, 1e4, 9)
    spec = spec_from_function(x, [q], lambda U, S, f, k: U * U - 0.5 * S * S + 0.3 * U * S)
    g = make_oracle_grid(oracle_mod, spec)
    rng = np.random.default_rng(2)
    xs = np.exp(rng.uniform(math.log(x[1]), math.log(x[-2]), 2000))
    qs = np.exp(rng.uniform(math.log(q[1]), math.log(q[-2]), 2000))
    out = g.xfxq2(spec.pids, xs, qs)[:, 0]
    want = np.log(xs) ** 2 - 0.5 * np.log(qs) ** 2 + 0.3 * np.log(xs) * np.log(qs)
    assert np.max(np.abs(out - want)) < 1e-13 * 100
    # end cells are NOT exact (one-sided slope): documented behaviour
    xe = np.exp(0.5 * (math.log(x[0]) + math.log(x[1])))
    oe = g.xfxq2(spec.pids, [xe], [qs[0]])[0, 0]
    assert abs(oe - (math.log(xe) ** 2 - 0.5 * math.log(qs[0]) ** 2 + 0.3 * math.log(xe) * math.log(qs[0]))) > 1e-3


# ---------------------------------------------------------------------------
# P-6: C0 at every cell boundary, C1 at knots strictly inside a (sub-)grid
# ---------------------------------------------------------------------------
def test_p6_continuity_c0_c1(oracle_mod):
    spec = synth.tiny_grid(3, 8, [5, 6])
    g = make_oracle_grid(oracle_mod, spec)
    xk = spec.x_knots.numpy()
    qfix = float(spec.q2_subgrids[1][2]) * 1.3
    for kn in xk[1:-1]:
        lo, hi = np.nextafter(kn, 0.0), kn
        a, b = g.xfxq2(spec.pids, [lo], [qfix])[0], g.xfxq2(spec.pids, [hi], [qfix])[0]
        assert np.max(np.abs(a - b)) < 1e-13
        h = 1e-6
        dl = (g.xfxq2(spec.pids, [kn], [qfix])[0] - g.xfxq2(spec.pids, [kn * math.exp(-h)], [qfix])[0]) / h
        dr = (g.xfxq2(spec.pids, [kn * math.exp(h)], [qfix])[0] - g.xfxq2(spec.pids, [kn], [qfix])[0]) / h
        assert np.max(np.abs(dl - dr)) < 2e-5
    xfix = float(xk[3]) * 1.2
    for k, qk in enumerate(spec.q2_subgrids):
        for kn in qk.numpy()[1:-1]:
            a = g.xfxq2(spec.pids, [xfix], [np.nextafter(kn, 0.0)])[0]
            b = g.xfxq2(spec.pids, [xfix], [kn])[0]
            assert np.max(np.abs(a - b)) < 1e-13
            h = 1e-6
            dl = (b - g.xfxq2(spec.pids, [xfix], [kn * math.exp(-h)])[0]) / h
            dr = (g.xfxq2(spec.pids, [xfix], [kn * math.exp(h)])[0] - b) / h
            assert np.max(np.abs(dl - dr)) < 2e-5


# ---------------------------------------------------------------------------
# P-7: sub-grid boundaries: no leakage across a threshold, jump = stored difference
# ---------------------------------------------------------------------------
def test_p7_subgrid_threshold(oracle_mod):
    spec = synth.grid_c1()
    g = make_oracle_grid(oracle_mod, spec)
    xk = spec.x_knots.numpy()
    for k in (0, 1):
        thr = float(spec.q2_subgrids[k][-1])
        lo = np.nextafter(thr, 0.0)
        up = g.xfxq2(spec.pids, xk, np.full_like(xk, thr))
        dn = g.xfxq2(spec.pids, xk, np.full_like(xk, lo))
        top_lower = spec.block(0, k).numpy()[:, -1, :]
        bot_upper = spec.block(0, k + 1).numpy()[:, 0, :]
        assert np.array_equal(up, bot_upper)
        assert np.max(np.abs(dn - top_lower)) <= 1e-13 * np.max(np.abs(top_lower))
        jump_col = spec.pids.index(4 if k == 0 else 5)
        assert np.all(top_lower[:-1, jump_col] == 0.0) and np.all(bot_upper[:-1, jump_col] != 0.0)
        _, _, isub, _ = g.locate([0.1, 0.1], [lo, thr])
        assert list(isub) == [k, k + 1]
    # a stencil never crosses a threshold: changing the other sub-grids leaves the result unchanged
    spec2 = synth.grid_c1()
    b1 = spec2.block(0, 1)
    keep = b1.clone()
    spec2.values.mul_(3.0).add_(1.0)
    spec2.block(0, 1).copy_(keep)
    g2 = make_oracle_grid(oracle_mod, spec2)
    rng = np.random.default_rng(3)
    xs = np.exp(rng.uniform(math.log(1e-9), 0, 500)).clip(1e-9, 1.0)
    qs = np.exp(rng.uniform(math.log(synth.MC2), math.log(synth.MB2), 500)).clip(synth.MC2, np.nextafter(synth.MB2, 0))
    assert np.array_equal(g.xfxq2(spec.pids, xs, qs), g2.xfxq2(spec.pids, xs, qs))


# ---------------------------------------------------------------------------
# P-8: extrapolation closed forms (L1722): power laws continue exactly
# ---------------------------------------------------------------------------
def test_p8_lowx_highq_power_law_and_affine(oracle_mod):
    x = uniform_log_knots(1e-5, 1.0, 14)
    q = uniform_log_knots(2.0, 1e6, 10)
    A, p, gq = 0.8, -0.45, 0.21
    # V = A x^p (Q2)^g : >1e-3 everywhere  -> log branch -> exact power-law continuation
    spec = spec_from_function(x, [q], lambda U, S, f, k: A * np.exp(p * U + gq * S))
    g = make_oracle_grid(oracle_mod, spec)
    xs = np.array([1e-6, 3e-8, 1e-12, np.nextafter(1e-5, 0)])
    qs = np.array([2.0, 37.0, 1e6, 5e3])
    out = g.xfxq2(spec.pids, xs, qs)[:, 0]
    # off the Q2 nodes the anchors are interpolated values I(q) of (Q2)^g; the x continuation of
    # A X^p I(q) is still the exact power law in x: out = out(X_0, q) (x/X_0)^p
    edge = g.xfxq2(spec.pids, np.full(4, x[0]), qs)[:, 0]
    want = edge * (xs / x[0]) ** p
    assert np.max(np.abs(out / want - 1)) < 1e-12   # amplified by |theta| up to ~20
    on_nodes = [0, 2]                               # q = first / last Q2 knot: interpolation exact
    assert np.max(np.abs(out[on_nodes] / (A * xs[on_nodes] ** p * qs[on_nodes] ** gq) - 1)) < 1e-12
    # on the node row / exact node column the interpolation is exact: tighter
    out = g.xfxq2(spec.pids, [1e-7], [q[3]])[0, 0]
    assert abs(out / (A * 1e-7 ** p * q[3] ** gq) - 1) < 1e-13
    qh = np.array([1e6 * 1.0000001, 1e7, 1e9])
    out = g.xfxq2(spec.pids, np.full(3, x[4]), qh)[:, 0]
    assert np.max(np.abs(out / (A * x[4] ** p * qh ** gq) - 1)) < 1e-13
    # corner low-x & high-Q: x rule first, then Q rule (L1744): still the power law
    out = g.xfxq2(spec.pids, [1e-8], [1e8])[0, 0]
    assert abs(out / (A * 1e-8 ** p * 1e8 ** gq) - 1) < 1e-12
    # affine data that are small or negative -> linear branch in ln x / ln Q2
    spec2 = spec_from_function(x, [q], lambda U, S, f, k: -0.2 + 0.01 * U + 0.003 * S)
    g2 = make_oracle_grid(oracle_mod, spec2)
    for (xx, qq) in [(1e-7, 50.0), (1e-2, 1e8), (1e-9, 1e9)]:
        out = g2.xfxq2(spec2.pids, [xx], [qq])[0, 0]
        assert abs(out - (-0.2 + 0.01 * math.log(xx) + 0.003 * math.log(qq))) < 1e-13
    # continuity into the grid
    a = g.xfxq2(spec.pids, [np.nextafter(1e-5, 0)], [100.0])[0, 0]
    b = g.xfxq2(spec.pids, [1e-5], [100.0])[0, 0]
    assert abs(a / b - 1) < 1e-13
    a = g.xfxq2(spec.pids, [1e-3], [np.nextafter(1e6, 1e7)])[0, 0]
    b = g.xfxq2(spec.pids, [1e-3], [1e6])[0, 0]
    assert abs(a / b - 1) < 1e-13


def test_p8_switch_threshold_is_strict_and_per_flavour(oracle_mod):
    """S-9: log branch iff BOTH anchor values > 1e-3 (strict), decided per flavour."""
    x = np.array([1e-3, 1e-2, 1e-1, 1.0])
    q = np.array([2.0, 20.0, 200.0])

    def fun(U, S, f, k):
        base = np.where(np.isclose(U, math.log(1e-3)), [4e-3, 1e-3, 4e-3][f], [2e-3, 2e-3, -1.0][f])
        return base + 0 * S
    spec = spec_from_function(x, [q], fun, nflav=3)
    g = make_oracle_grid(oracle_mod, spec)
    xx = 1e-4
    theta = (math.log(xx) - math.log(1e-3)) / (math.log(1e-2) - math.log(1e-3))
    out = g.xfxq2(spec.pids, [xx], [20.0])[0]
    want0 = math.exp(math.log(4e-3) + theta * (math.log(2e-3) - math.log(4e-3)))   # log branch
    want1 = 1e-3 + theta * (2e-3 - 1e-3)                                            # 1e-3 is NOT > 1e-3
    want2 = 4e-3 + theta * (-1.0 - 4e-3)                                            # negative anchor
    assert np.allclose(out, [want0, want1, want2], rtol=1e-13, atol=0)


# ---------------------------------------------------------------------------
# P-9: low-Q continuation, eq. 3.4 / 3.5 (golden fixture, hand-worked)
# ---------------------------------------------------------------------------
def _lowq_grid(oracle_mod, gamma, fmin=2.0):
    """Values affine in ln Q2 (reproduced exactly, P-3) so that gamma is known in closed form:
    f(Q2min)=fmin, f(1.01 Q2min) = fmin (1 + 0.01 gamma)."""
    x = uniform_log_knots(1e-3, 1.0, 6)
    q = uniform_log_knots(1.0, 1e4, 8)
    beta = gamma * 0.01 * fmin / math.log(1.01)
    spec = spec_from_function(x, [q], lambda U, S, f, k: fmin + beta * S + 0 * U)
    return make_oracle_grid(oracle_mod, spec), spec


def test_p9_lowq_fixture(oracle_mod):
    for line in open(os.path.join(GOLD, "eq34_lowq_worked.txt")):
        if line.startswith("#") or not line.strip():
            continue
        gamma, r, want = [float(v) for v in line.split()]
        g, spec = _lowq_grid(oracle_mod, gamma)
        out = g.xfxq2(spec.pids, [0.05], [r * 1.0])[0, 0]
        assert abs(out / want - 1) < 2e-12, (gamma, r, out, want)


def test_p9_lowq_limits_and_guards(oracle_mod):
    g, spec = _lowq_grid(oracle_mod, 1.7)
    # eq. 3.5 first limit: Q2 -> Q2min: xf -> f_min r^gamma -> f_min ; continuity at the edge
    a = g.xfxq2(spec.pids, [0.05], [np.nextafter(1.0, 0.0)])[0, 0]
    assert abs(a / 2.0 - 1) < 1e-13
    r = 1.0 - 1e-6
    a = g.xfxq2(spec.pids, [0.05], [r])[0, 0]
    assert abs(a / (2.0 * r ** 1.7) - 1) < 1e-11
    # eq. 3.5 second limit: xf / (f_min r) -> 1
    a = g.xfxq2(spec.pids, [0.05], [1e-9])[0, 0]
    assert abs(a / (2.0 * 1e-9) - 1) < 1e-7
    # floor gamma >= -2.5 [not in paper, S-13]
    g2, spec2 = _lowq_grid(oracle_mod, -7.0)
    a = g2.xfxq2(spec2.pids, [0.05], [0.5])[0, 0]
    assert abs(a / (2.0 * 0.5 ** ((-2.5 - 1) * 0.5 + 1)) - 1) < 1e-12
    # guard f_min <= 1e-5 -> gamma = 1 [not in paper, S-13]
    g3, spec3 = _lowq_grid(oracle_mod, 3.0, fmin=1e-6)
    a = g3.xfxq2(spec3.pids, [0.05], [0.25])[0, 0]
    assert abs(a / (1e-6 * 0.25) - 1) < 1e-12
    # gamma estimated by the 1 % forward difference of a power law (Q2)^g0 (interpolation error small)
    x = uniform_log_knots(1e-3, 1.0, 6)
    q = uniform_log_knots(1.0, 1e4, 60)
    g0 = 0.8
    spec4 = spec_from_function(x, [q], lambda U, S, f, k: 1.5 * np.exp(g0 * S) + 0 * U)
    g4 = make_oracle_grid(oracle_mod, spec4)
    # the bottom cell is an END cell (S-3 A): near its end knot the interpolant's log-slope is the
    # one-sided secant (e^{g0 D} - 1)/D, D = knot spacing in ln Q2, so gamma ~ secant * ln(1.01)/0.01
    D = math.log(q[1] / q[0])
    gam = (math.exp(g0 * D) - 1) / D * math.log(1.01) / 0.01
    a = g4.xfxq2(spec4.pids, [0.05], [0.3])[0, 0]
    assert abs(a / (1.5 * 0.3 ** ((gam - 1) * 0.3 + 1)) - 1) < 2e-3
    # with knots fine enough the secant tends to g0 itself
    q = uniform_log_knots(1.0, 1e4, 4000)
    spec4 = spec_from_function(x, [q], lambda U, S, f, k: 1.5 * np.exp(g0 * S) + 0 * U)
    g4 = make_oracle_grid(oracle_mod, spec4)
    gam = (1.01 ** g0 - 1) / 0.01
    a = g4.xfxq2(spec4.pids, [0.05], [0.3])[0, 0]
    assert abs(a / (1.5 * 0.3 ** ((gam - 1) * 0.3 + 1)) - 1) < 2e-4
    # corner low-x & low-Q: x rule first (L1744): affine-in-ln-x small data, then eq. 3.4
    spec5 = spec_from_function(x, [q], lambda U, S, f, k: 2.0 * np.exp(-0.3 * U) + 0 * S)
    g5 = make_oracle_grid(oracle_mod, spec5)
    a = g5.xfxq2(spec5.pids, [1e-5], [0.5])[0, 0]
    assert abs(a / (2.0 * 1e-5 ** -0.3 * 0.5 ** ((0 - 1) * 0.5 + 1)) - 1) < 1e-12


# ---------------------------------------------------------------------------
# P-10: three evaluation orders agree
# ---------------------------------------------------------------------------
def test_p10_three_orders(oracle_mod):
    spec = synth.grid_c1()
    g = make_oracle_grid(oracle_mod, spec)
    x, q = synth.queries_inside(spec, 5000, 77)
    for f in (0, 5, 9):
        a = g.interior_order(0, f, x.numpy(), q.numpy())
        b = g.interior_order(1, f, x.numpy(), q.numpy())
        c = g.interior_order(2, f, x.numpy(), q.numpy())
        _, S = g.xfxq2([spec.pids[f]], x.numpy(), q.numpy(), want_scale=True)
        S = S[:, 0, 0] + 1e-300
        assert np.max(np.abs(a - b) / S) < 1e-14 and np.max(np.abs(a - c) / S) < 1e-14


# ---------------------------------------------------------------------------
# P-11: brute force on tiny NON-uniform grids, dense raster + nextafter neighbours of knots
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("nx,nq", [(2, [2]), (3, [3]), (4, [2, 3]), (5, [4, 2, 5]), (3, [5]), (5, [3, 3])])
def test_p11_bruteforce_tiny(oracle_mod, nx, nq):
    spec = synth.tiny_grid(100 + nx * 10 + len(nq), nx, nq, nflav=2)
    g = make_oracle_grid(oracle_mod, spec)
    xk = spec.x_knots.numpy()
    qk = np.unique(np.concatenate([q.numpy() for q in spec.q2_subgrids]))
    xs = np.concatenate([np.exp(np.linspace(math.log(xk[0]), math.log(xk[-1]), 23)).clip(xk[0], xk[-1]),
                         xk, np.nextafter(xk[1:], 0), np.nextafter(xk[:-1], 2)])
    qs = np.concatenate([np.exp(np.linspace(math.log(qk[0]), math.log(qk[-1]), 29)).clip(qk[0], qk[-1]),
                         qk, np.nextafter(qk[1:], 0), np.nextafter(qk[:-1], 1e9)])
    X, Q = np.meshgrid(xs, qs, indexing="ij")
    X, Q = X.ravel(), Q.ravel()
    out = g.xfxq2(spec.pids, X, Q)
    vmax = float(np.max(np.abs(spec.values.numpy())))
    for e in range(0, len(X)):
        for f in range(2):
            want = brute_interior(spec, float(X[e]), float(Q[e]), f)
            assert abs(out[e, f] - want) < 1e-13 * vmax * 10, (X[e], Q[e], f, out[e, f], want)


def test_p11_members_and_pids(oracle_mod):
    """P-14 + C-11: member m of a batch == single-member grid of member m's values;
    unknown pid -> 0.0; pid 0 aliases 21; column order follows the request."""
    spec = synth.tiny_grid(9, 6, [4, 5], nflav=3, nmem=4)
    g = make_oracle_grid(oracle_mod, spec)
    rng = np.random.default_rng(8)
    n = 300
    xs = np.exp(rng.uniform(math.log(1e-4), 0, n)).clip(1e-4, 1.0)
    qs = np.exp(rng.uniform(math.log(1.5), math.log(1e4), n)).clip(1.5, 1e4)
    mem = rng.integers(0, 4, n).astype(np.int32)
    out = g.xfxq2(spec.pids, xs, qs, member=mem)
    for m in range(4):
        single = synth.GridSpec(spec.x_knots, spec.q2_subgrids, spec.member_values(m).clone(), pids=spec.pids)
        gs = make_oracle_grid(oracle_mod, single)
        sel = mem == m
        assert np.array_equal(out[sel], gs.xfxq2(spec.pids, xs[sel], qs[sel]))
    o2 = g.xfxq2([3, 99, 1], xs, qs, member=mem)
    assert np.array_equal(o2[:, 0], out[:, 2]) and np.all(o2[:, 1] == 0.0) and np.array_equal(o2[:, 2], out[:, 0])
    c1 = synth.grid_c1()
    gc = make_oracle_grid(oracle_mod, c1)
    o = gc.xfxq2([0, 21], [0.01], [100.0])[0]
    assert o[0] == o[1]


def test_p14_zero_noise_members_equal_base(oracle_mod):
    base = synth.grid_c1()
    batch = synth.grid_c1(nmem=3, sigma=0.0)
    gb, gm = make_oracle_grid(oracle_mod, base), make_oracle_grid(oracle_mod, batch)
    x, q = synth.queries_c2(base, 2000, 5)
    mem = synth.members(batch, 2000).numpy()
    assert np.array_equal(gb.xfxq2(base.pids, x.numpy(), q.numpy()),
                          gm.xfxq2(base.pids, x.numpy(), q.numpy(), member=mem), equal_nan=True)


# ---------------------------------------------------------------------------
# P-12: alpha_s (L1746, L1835)
# ---------------------------------------------------------------------------
def test_p12_alphas(oracle_mod):
    spec = synth.grid_c1()
    g = make_oracle_grid(oracle_mod, spec)
    aq, av = spec.alphas_q2.numpy(), spec.alphas_val.numpy()
    assert abs(av[0] - 0.35) < 1e-15 and abs(av[-1] - 0.08) < 1e-15 and np.all(np.diff(av) < 0)
    assert np.array_equal(g.alphas_q2(aq), av)                       # nodes, bitwise
    assert np.all(g.alphas_q2([aq[-1] * 2, 1e30]) == av[-1])         # constant above Q2max (L1746)
    assert np.all(g.alphas_q2([aq[0] / 2, 1e-30]) == av[0])          # PDFFlow: constant below (L1835)
    assert np.all(np.isnan(g.alphas_q2([0.0, -1.0, np.nan])))
    qs = np.exp(np.linspace(math.log(aq[0]), math.log(aq[-1]), 5001)).clip(aq[0], aq[-1])
    out = g.alphas_q2(qs)
    assert out.max() <= av[0] * (1 + 1e-3) and out.min() >= av[-1] * (1 - 1e-3)
    # brute force (monomial form) on the 1-D line
    for e in range(0, len(qs), 7):
        c = brute_cell(aq, qs[e])
        assert abs(out[e] - brute_line(np.log(aq), av, math.log(qs[e]), c)) < 1e-14
    # linear-in-ln-Q2 data reproduced; LHAPDF log-gradient option below Q2min
    lin = 0.3 - 0.01 * np.log(aq)
    g.set_alphas(aq, lin)
    assert np.max(np.abs(g.alphas_q2(qs) - (0.3 - 0.01 * np.log(qs)))) < 1e-15
    g.set_alphas(aq, av, mode=oracle_mod.ALPHAS_LOGGRAD)
    slope = math.log(av[1] / av[0]) / math.log(aq[1] / aq[0])
    got = g.alphas_q2([aq[0] * 0.3])[0]
    assert abs(got / (av[0] * 0.3 ** slope) - 1) < 1e-14
    # C1 continuity at interior alpha_s knots
    g.set_alphas(aq, av)
    for kn in aq[1:-1:6]:
        h = 1e-6
        dl = (g.alphas_q2([kn])[0] - g.alphas_q2([kn * math.exp(-h)])[0]) / h
        dr = (g.alphas_q2([kn * math.exp(h)])[0] - g.alphas_q2([kn])[0]) / h
        assert abs(dl - dr) < 1e-6


# ---------------------------------------------------------------------------
# P-13: luminosity (eq. 3.3, eq. 4.1)
# ---------------------------------------------------------------------------
def test_p13_lumi(oracle_mod):
    spec = synth.grid_c1()
    g = make_oracle_grid(oracle_mod, spec)
    x1, x2, q2, w = [t.numpy() for t in synth.events_c4(3000)]
    out, sc = g.lumi(x1, x2, q2, w, want_scale=True)
    assert np.mean(q2 < 1.0) > 0.15          # ~20 % of events take the low-Q branch (must not be clamped)
    f1 = g.xfxq2(spec.pids, x1, q2) / x1[:, None]
    f2 = g.xfxq2(spec.pids, x2, q2) / x2[:, None]
    Cm = spec.coupling.numpy()
    want = w * np.einsum("ei,ij,ej->e", f1, Cm, f2)
    sc = sc[:, 0]
    assert np.max(np.abs(out - want) / sc) < 1e-13
    # C = e_i e_j^T isolates one product
    E = np.zeros((11, 11)); E[2, 7] = 1.0
    g.set_coupling(E)
    assert np.allclose(g.lumi(x1, x2, q2, w), w * f1[:, 2] * f2[:, 7], rtol=1e-14, atol=0)
    # swapping the partons and transposing C leaves the result unchanged
    g.set_coupling(Cm.T.copy())
    swapped = g.lumi(x2, x1, q2, w)
    assert np.max(np.abs(swapped - out) / sc) < 1e-13


# ---------------------------------------------------------------------------
# The condition numbers of the parity metric (C-12).  Every GPU parity assertion divides by
# them, so a mistake that inflates them would loosen all parity tests: pinned here against an independent
# restatement (SURVEY C-5's closed 4-weight form in the monomial basis, numerical derivatives of the
# literal interpolant above, and the first-order propagation formulas written out on pinned inputs).
# ---------------------------------------------------------------------------
def closed_weights(lk, c, t):
    """SURVEY C-5 4-weight form, monomial Hermite basis; lk = ln-knots of one (sub-)line, vectorised over queries"""
    m = len(lk)
    h00, h10 = 2 * t**3 - 3 * t**2 + 1, t**3 - 2 * t**2 + t
    h01, h11 = -2 * t**3 + 3 * t**2, t**3 - t**2
    d = lk[c + 1] - lk[c]
    left, right = c > 0, c + 2 < m
    rm = np.where(left, d / (lk[c] - lk[np.maximum(c - 1, 0)] + (~left) * 1.0), 0.0)
    rp = np.where(right, d / (lk[np.minimum(c + 2, m - 1)] - lk[c + 1] + (~right) * 1.0), 0.0)
    w = np.empty((4,) + t.shape)
    w[0] = np.where(left, -0.5 * rm * h10, 0.0)
    w[1] = np.where(left, h00 + 0.5 * (rm - 1) * h10, h00 - h10) - np.where(right, 0.5 * h11, h11)
    w[2] = h01 + np.where(left, 0.5 * h10, h10) + np.where(right, 0.5 * (1 - rp) * h11, h11)
    w[3] = np.where(right, 0.5 * rp * h11, 0.0)
    return w


def closed_stencil(spec, x, q2):
    """per query: sub-grid k, cells, the 4 x 4 node weights and node values [n][4][4][nflav] (absent nodes: weight 0)"""
    xk = spec.x_knots.numpy()
    n = len(x)
    W = np.zeros((n, 4, 4))
    V = np.zeros((n, 4, 4, spec.nflav))
    T = np.zeros((n, 4))     # t_x, t_q, du, ds
    starts = np.array([float(q[0]) for q in spec.q2_subgrids])
    ksub = np.searchsorted(starts, q2, side="right") - 1
    for k, qk_t in enumerate(spec.q2_subgrids):
        sel = np.nonzero(ksub == k)[0]
        if not sel.size:
            continue
        qk = qk_t.numpy()
        i = np.clip(np.searchsorted(xk, x[sel], side="right") - 1, 0, len(xk) - 2)
        j = np.clip(np.searchsorted(qk, q2[sel], side="right") - 1, 0, len(qk) - 2)
        lx, lq = np.log(xk), np.log(qk)
        tx = (np.log(x[sel]) - lx[i]) / (lx[i + 1] - lx[i])
        tq = (np.log(q2[sel]) - lq[j]) / (lq[j + 1] - lq[j])
        wx, wq = closed_weights(lx, i, tx), closed_weights(lq, j, tq)
        blk = spec.block(0, k).numpy()
        for a in range(4):
            ia = np.clip(i - 1 + a, 0, len(xk) - 1)
            for b in range(4):
                jb = np.clip(j - 1 + b, 0, len(qk) - 1)
                W[sel, a, b] = wx[a] * wq[b]
                V[sel, a, b, :] = blk[ia, jb, :]
        T[sel] = np.stack([tx, tq, lx[i + 1] - lx[i], lq[j + 1] - lq[j]], axis=1)
    return W, V, T


@pytest.mark.parametrize("which", ["c1", "tiny"])
def test_scale_interior_sum_part(oracle_mod, which):
    """scale[0] == sum |Wx_a Wq_b V_ab| (and the value == sum Wx_a Wq_b V_ab) on 1e5 random interior queries"""
    if which == "c1":
        spec, n = synth.grid_c1(), 100_000
    else:
        spec, n = synth.tiny_grid(321, 5, [4, 2, 5], nflav=3), 20_000
    g = make_oracle_grid(oracle_mod, spec)
    x, q = synth.queries_inside(spec, n, 1234)
    x, q = x.numpy(), q.numpy()
    ref, S = g.xfxq2(spec.pids, x, q, want_scale=True)
    W, V, _ = closed_stencil(spec, x, q)
    want_S0 = np.einsum("nab,nabf->nf", np.abs(W), np.abs(V))
    want_v = np.einsum("nab,nabf->nf", W, V)
    assert S.shape == (n, spec.nflav, 2)
    assert np.max(np.abs(S[:, :, 0] - want_S0) / (want_S0 + 1e-300)) < 1e-11     # monomial vs factored basis: ~1e-13
    assert np.max(np.abs(ref - want_v) / (want_S0 + 1e-3 * S[:, :, 1] + 1e-300)) < 1e-12   # the two t's differ by their rounding
    assert np.all(S[:, :, 0] >= np.abs(ref) * (1 - 1e-12))                       # |f| <= S always
    assert np.all(S[:, :, 1] >= 0)


def test_scale_interior_t_part(oracle_mod):
    """scale[1] == |df/dt_x| (1 + |ln x|/du) + |df/dt_q| (1 + |ln Q2|/ds), derivatives taken numerically from
    the literal second implementation (brute_interior)"""
    spec = synth.tiny_grid(322, 5, [4, 5], nflav=2)
    g = make_oracle_grid(oracle_mod, spec)
    x, q = synth.queries_inside(spec, 400, 99)
    x, q = x.numpy(), q.numpy()
    _, S = g.xfxq2(spec.pids, x, q, want_scale=True)
    _, _, T = closed_stencil(spec, x, q)
    checked = 0
    for e in range(len(x)):
        tx, tq, du, ds = T[e]
        if not (0.1 < tx < 0.9 and 0.1 < tq < 0.9):
            continue                                        # the central difference must stay inside the cell
        h = 1e-5
        for f in range(spec.nflav):
            dfx = (brute_interior(spec, x[e] * math.exp(h * du), q[e], f) - brute_interior(spec, x[e] * math.exp(-h * du), q[e], f)) / (2 * h)
            dfq = (brute_interior(spec, x[e], q[e] * math.exp(h * ds), f) - brute_interior(spec, x[e], q[e] * math.exp(-h * ds), f)) / (2 * h)
            want = abs(dfx) * (1 + abs(math.log(x[e])) / du) + abs(dfq) * (1 + abs(math.log(q[e])) / ds)
            assert abs(S[e, f, 1] - want) <= 1e-6 * (want + S[e, f, 0])
            checked += 1
    assert checked > 200


def test_scale_extrapolation_propagation(oracle_mod):
    """first-order propagation through C-7 / C-8 / C-9, written out on the (pinned) interior numbers"""
    spec = synth.grid_c1()
    g = make_oracle_grid(oracle_mod, spec)
    xk = spec.x_knots.numpy()
    qall = np.concatenate([t.numpy() for t in spec.q2_subgrids])
    q2min, q2max, qprev = qall[0], qall[-1], qall[-2]
    u0, u1 = math.log(xk[0]), math.log(xk[1])
    rng = np.random.default_rng(8)
    n = 300

    def two(f0, S0, f1, S1, theta, cond):
        v = np.where((f0 > 1e-3) & (f1 > 1e-3), np.exp(np.log(np.abs(f0) + 1e-300) + theta * (np.log(np.abs(f1) + 1e-300) - np.log(np.abs(f0) + 1e-300))),
                     f0 + theta * (f1 - f0))
        logf = (f0 > 1e-3) & (f1 > 1e-3)
        out = np.empty(S0.shape)
        for c in range(2):
            lin = np.abs(1 - theta) * S0[..., c] + np.abs(theta) * S1[..., c] + (c == 1) * cond * np.abs(f1 - f0)
            with np.errstate(divide="ignore", invalid="ignore"):
                lg = np.abs(v) * (np.abs(1 - theta) * S0[..., c] / f0 + np.abs(theta) * S1[..., c] / f1
                                  + (c == 1) * cond * np.abs(np.log(f1) - np.log(f0)))
            out[..., c] = np.where(logf, lg, lin)
        return v, out

    # C-7 low-x, Q2 inside
    x = np.exp(rng.uniform(math.log(1e-12), u0, n)); x = x[x < xk[0]]
    q = np.exp(rng.uniform(math.log(q2min), math.log(q2max), len(x)))
    ref, S = g.xfxq2(spec.pids, x, q, want_scale=True)
    f0, S0 = g.xfxq2(spec.pids, np.full(len(x), xk[0]), q, want_scale=True)
    f1, S1 = g.xfxq2(spec.pids, np.full(len(x), xk[1]), q, want_scale=True)
    theta = ((np.log(x) - u0) / (u1 - u0))[:, None]
    cond = (1 + np.abs(np.log(x)) / (u1 - u0))[:, None]
    v, want = two(f0, S0, f1, S1, theta, cond)
    assert np.max(np.abs(ref - v) / (np.abs(v) + 1e-300)) < 1e-12
    assert np.max(np.abs(S - want) / (want + 1e-300)) < 1e-10
    assert ((f0 > 1e-3) & (f1 > 1e-3)).any() and (~((f0 > 1e-3) & (f1 > 1e-3))).any()    # both forms are exercised
    # C-8 high-Q, x inside
    x = np.exp(rng.uniform(u0, 0.0, n)).clip(xk[0], xk[-1])
    q = np.exp(rng.uniform(math.log(q2max), math.log(q2max) + 4, n)); q = np.maximum(q, np.nextafter(q2max, 1e300))
    ref, S = g.xfxq2(spec.pids, x, q, want_scale=True)
    f0, S0 = g.xfxq2(spec.pids, x, np.full(n, qprev), want_scale=True)
    f1, S1 = g.xfxq2(spec.pids, x, np.full(n, q2max), want_scale=True)
    ds = math.log(q2max) - math.log(qprev)
    theta = ((np.log(q) - math.log(qprev)) / ds)[:, None]
    cond = (1 + np.abs(np.log(q)) / ds)[:, None]
    v, want = two(f0, S0, f1, S1, theta, cond)
    assert np.max(np.abs(ref - v) / (np.abs(v) + 1e-300)) < 1e-12
    assert np.max(np.abs(S - want) / (want + 1e-300)) < 1e-10
    # C-9 low-Q, x inside
    q = np.exp(rng.uniform(math.log(q2min) - 4, math.log(q2min), n)); q = np.minimum(q, np.nextafter(q2min, 0))
    ref, S = g.xfxq2(spec.pids, x, q, want_scale=True)
    fm, Sm = g.xfxq2(spec.pids, x, np.full(n, q2min), want_scale=True)
    fp, Sp = g.xfxq2(spec.pids, x, np.full(n, 1.01 * q2min), want_scale=True)
    r = (q / q2min)[:, None]
    with np.errstate(divide="ignore", invalid="ignore"):
        gfd = (fp - fm) / (0.01 * fm)
    free = (fm > 1e-5) & (gfd > -2.5)
    gamma = np.where(fm > 1e-5, np.maximum(gfd, -2.5), 1.0)
    v = fm * r ** ((gamma - 1) * r + 1)
    assert np.max(np.abs(ref - v) / (np.abs(v) + 1e-300)) < 1e-12
    for c in range(2):
        with np.errstate(divide="ignore", invalid="ignore"):
            base = np.where(fm != 0, np.abs(v / fm) * Sm[..., c], r ** ((gamma - 1) * r + 1) * Sm[..., c])
            extra = np.abs(v * np.log(r) * r) * (Sp[..., c] / (0.01 * fm) + np.abs(fp) * Sm[..., c] / (0.01 * fm * fm))
        want = base + np.where(free, extra, 0.0)
        assert np.max(np.abs(S[..., c] - want) / (want + 1e-300)) < 1e-10
    assert free.any() and (~free).any()


def test_scale_lumi_formula(oracle_mod):
    """oracle_lumi's scale == |w| sum_ij |C_ij| (S1_i |f2_j| + |f1_i| S2_j) per component (pdf_oracle.h)"""
    spec = synth.grid_c1()
    g = make_oracle_grid(oracle_mod, spec)
    x1, x2, q2, w = [t.numpy() for t in synth.events_c4(2000, seed=5)]
    _, sc = g.lumi(x1, x2, q2, w, want_scale=True)
    v1, S1 = g.xfxq2(spec.pids, x1, q2, want_scale=True)
    v2, S2 = g.xfxq2(spec.pids, x2, q2, want_scale=True)
    f1, f2 = np.abs(v1 / x1[:, None]), np.abs(v2 / x2[:, None])
    aC = np.abs(spec.coupling.numpy())
    assert sc.shape == (2000, 2)
    for c in range(2):
        s1, s2 = S1[..., c] / x1[:, None], S2[..., c] / x2[:, None]
        want = np.abs(w) * (np.einsum("ei,ij,ej->e", s1, aC, f2) + np.einsum("ei,ij,ej->e", f1, aC, s2))
        assert np.max(np.abs(sc[:, c] - want) / want) < 1e-12


def test_s3_reading_b_switch(oracle_mod):
    """SURVEY S-3: the literal reading B (pure linear end cells) exists as a compile-time switch
    of the oracle; what distinguishes it from the default reading A is C1 at the first interior knot."""
    import ctypes as C
    path = oracle_mod.build(variant="ORACLE_S3_BILINEAR")
    L = C.CDLL(path)
    dp = C.POINTER(C.c_double)
    L.oracle_weights_1d.argtypes = [C.c_int, dp, C.c_double, C.c_int, dp]
    lk = np.log(np.array([1.0, 2.0, 4.5, 9.0, 20.0]))
    for lib_, end_is_linear in ((oracle_mod.lib(), False), (L, True)):
        w = np.zeros(4)
        lib_.oracle_weights_1d(5, lk.ctypes.data_as(dp), float(lk[0] + 0.3 * (lk[1] - lk[0])), 0, w.ctypes.data_as(dp))
        assert abs(w.sum() - 1) < 1e-15
        is_lin = abs(w[1] - 0.7) < 1e-15 and abs(w[2] - 0.3) < 1e-15 and w[3] == 0
        assert is_lin == end_is_linear
        w2 = np.zeros(4)                     # interior cells are the same cubic under both readings
        lib_.oracle_weights_1d(5, lk.ctypes.data_as(dp), float(lk[1] + 0.3 * (lk[2] - lk[1])), 1, w2.ctypes.data_as(dp))
        assert abs(w2[0]) > 1e-3 and abs(w2[3]) > 1e-3


# ---------------------------------------------------------------------------
# workload sanity (DESIGN.md input recipe): region mix of configs[2], sub-grid shares of configs[1]
# ---------------------------------------------------------------------------
def test_workload_shapes(oracle_mod):
    spec = synth.grid_c1()
    assert spec.nx == 196 and spec.nq == [6, 8, 40] and spec.nflav == 11
    assert float(spec.q2_subgrids[0][-1]) == float(spec.q2_subgrids[1][0]) == synth.MC2
    assert float(spec.q2_subgrids[1][-1]) == float(spec.q2_subgrids[2][0]) == synth.MB2
    g = make_oracle_grid(oracle_mod, spec)
    x, q = synth.queries_c2(spec, 400000)
    _, _, isub, reg = g.locate(x.numpy(), q.numpy())
    share = np.bincount(reg, minlength=7) / len(reg)
    assert abs(share[0] - 0.95) < 2e-3 and abs(share[1] - 0.02) < 1e-3
    assert abs(share[2] - 0.0125) < 1e-3 and abs(share[3] - 0.0125) < 1e-3
    assert abs(share[4] - 0.0025) < 5e-4 and abs(share[5] - 0.0025) < 5e-4 and share[6] == 0
    x, q = synth.queries_inside(spec, 400000, 3)
    _, _, isub, reg = g.locate(x.numpy(), q.numpy())
    assert np.all(reg == 0)
    s = np.bincount(isub, minlength=3) / len(isub)
    assert abs(s[0] - 0.036) < 3e-3 and abs(s[1] - 0.103) < 3e-3


# ---------------------------------------------------------------------------
# NEXT-4: the other extrapolation options of LHAPDF 6 and xfxQ (L1712)
# ---------------------------------------------------------------------------
def _outside_queries(spec, n=4000, seed=5):
    """valid queries of every region class of Fig. 3.1(b), and some inside"""
    rng = np.random.default_rng(seed)
    xk = spec.x_knots.numpy()
    qk = np.concatenate([q.numpy() for q in spec.q2_subgrids])
    x = np.exp(rng.uniform(np.log(xk[0]) - 6.0, np.log(xk[-1]), n))
    q = np.exp(rng.uniform(np.log(qk[0]) - 4.0, np.log(qk[-1]) + 4.0, n))
    x[::7] = xk[0]; q[::11] = qk[0]; q[5::11] = qk[-1]            # on the range's edges
    return x, q, xk, qk


def test_freeze_returns_the_value_at_the_closest_point_of_the_range(oracle_mod):
    """L1720 "freeze the grid edges": outside the range the value does not depend on how far outside the query
    is; on a knot line of the boundary it is the STORED node value (P-1 through the option); inside nothing changes."""
    spec = synth.grid_c1()
    og = make_oracle_grid(oracle_mod, spec)
    x, q, xk, qk = _outside_queries(spec)
    base = og.xfxq2(spec.pids, x, q)
    og.set_extrapolation(oracle_mod.EXTRAP_FREEZE)
    fr = og.xfxq2(spec.pids, x, q)
    inside = (x >= xk[0]) & (q >= qk[0]) & (q <= qk[-1])
    assert inside.any() and (~inside).any()
    assert np.array_equal(fr[inside], base[inside])
    # twice as far out: the same numbers, bit for bit
    x2 = np.where(x < xk[0], x * 1e-3, x)
    q2 = np.where(q < qk[0], q * 1e-2, np.where(q > qk[-1], q * 1e2, q))
    assert np.array_equal(og.xfxq2(spec.pids, x2, q2), fr)
    # below the first x knot AND on a Q2 knot: the node value V[0][jq] itself
    nx = len(xk)
    nq0 = spec.q2_subgrids[0].numel()
    V0 = spec.values.numpy()[: nx * nq0 * 11].reshape(nx, nq0, 11)
    for jq in (1, 3):
        got = og.xfxq2(spec.pids, np.array([xk[0] * 1e-4]), np.array([spec.q2_subgrids[0].numpy()[jq]]))[0]
        assert np.array_equal(got, V0[0, jq])
    # below Q2min AND on an x knot: V[ix][0]; above Q2max: the last node row
    got = og.xfxq2(spec.pids, np.array([xk[17]]), np.array([qk[0] * 1e-3]))[0]
    assert np.array_equal(got, V0[17, 0])
    nql = spec.q2_subgrids[-1].numel()
    Vl = spec.values.numpy()[-nx * nql * 11:].reshape(nx, nql, 11)
    got = og.xfxq2(spec.pids, np.array([xk[40]]), np.array([qk[-1] * 50.0]))[0]
    assert np.array_equal(got, Vl[40, nql - 1])
    # the cell reported is the boundary cell, the region interior
    ix, iq, isub, reg = og.locate(x, q)
    assert set(np.unique(reg).tolist()) == {0}
    assert (ix[x < xk[0]] == 0).all() and (isub[q < qk[0]] == 0).all() and (iq[q < qk[0]] == 0).all()
    assert (isub[q > qk[-1]] == len(spec.q2_subgrids) - 1).all() and (iq[q > qk[-1]] == nql - 2).all()


def test_error_option_rejects_every_query_outside_the_range(oracle_mod):
    """L1720 "raise an error if a point outside the grid range is queried": NaN rows outside, nothing changes inside"""
    spec = synth.grid_c1()
    og = make_oracle_grid(oracle_mod, spec)
    x, q, xk, qk = _outside_queries(spec)
    base = og.xfxq2(spec.pids, x, q)
    og.set_extrapolation(oracle_mod.EXTRAP_ERROR)
    er = og.xfxq2(spec.pids, x, q)
    inside = (x >= xk[0]) & (q >= qk[0]) & (q <= qk[-1])
    assert np.array_equal(er[inside], base[inside])
    assert np.isnan(er[~inside]).all() and not np.isnan(base[~inside]).any()
    reg = og.locate(x, q)[3]
    assert (reg[~inside] == 6).all() and (reg[inside] == 0).all()
    og.set_extrapolation(oracle_mod.EXTRAP_CONTINUATION)
    assert np.array_equal(og.xfxq2(spec.pids, x, q), base)


def test_xfxq_is_xfxq2_at_q_squared(oracle_mod):
    """L1712: PDF::xfxQ and PDF::xfxQ2 are the same function of Q and Q2.  On a grid whose Q2 knots are exact squares
    the Q knots reproduce the node values (P-1); Q <= 0 is invalid although its square is not."""
    xk = uniform_log_knots(1e-4, 1.0, 9)
    qroot = np.array([2.0, 4.0, 8.0, 16.0, 32.0])
    spec = spec_from_function(xk, [qroot * qroot], lambda U, S, f, k: np.sin(U) + 0.1 * S * S + f, nflav=2)
    og = make_oracle_grid(oracle_mod, spec)
    V = spec.values.numpy().reshape(9, 5, 2)
    for ix in (0, 3, 8):
        for jq in (0, 2, 4):
            got = og.xfxq(spec.pids, np.array([xk[ix]]), np.array([qroot[jq]]))[0]
            assert np.array_equal(got, V[ix, jq])
    rng = np.random.default_rng(2)
    x = np.exp(rng.uniform(np.log(1e-5), 0.0, 500))
    Q = np.exp(rng.uniform(np.log(1.0), np.log(64.0), 500))
    assert np.array_equal(og.xfxq(spec.pids, x, Q), og.xfxq2(spec.pids, x, Q * Q))
    bad = og.xfxq(spec.pids, np.array([0.1, 0.1, 0.1]), np.array([-4.0, 0.0, np.inf]))
    assert np.isnan(bad).all()


def test_alphas_subgrids_split_the_knot_line(oracle_mod):
    """C-alpha / L1835 ("the sub-grids mechanism ... flavor thresholds"): a repeated knot splits the alpha_s line
    exactly as C-3 splits the Q2 line.  Pins: each sub-line equals the SAME knots given as a line of their own
    (nothing leaks across a threshold); the threshold belongs to the upper sub-line; the jump is reproduced."""
    spec = synth.grid_c0()
    og = make_oracle_grid(oracle_mod, spec)
    a = np.array([1.0, 1.7, 2.28, 2.28, 5.0, 11.0, 24.2, 24.2, 90.0, 400.0, 1e4])
    A = np.array([0.40, 0.37, 0.35, 0.352, 0.30, 0.26, 0.23, 0.2312, 0.19, 0.16, 0.12])
    og.set_alphas(a, A)
    rng = np.random.default_rng(3)
    cuts = [(0, 3), (3, 7), (7, 11)]
    for lo, hi in cuts:
        q = np.exp(rng.uniform(np.log(a[lo]), np.log(a[hi - 1]), 400))
        q = q[(q >= a[lo]) & (q < a[hi - 1])]
        whole = og.alphas_q2(q)
        og2 = make_oracle_grid(oracle_mod, spec)
        og2.set_alphas(a[lo:hi], A[lo:hi])
        assert np.array_equal(whole, og2.alphas_q2(q))
    # nodes: every knot returns a stored value; on a threshold the upper one; just below it the lower sub-line's limit
    got = og.alphas_q2(a)
    exp = A.copy(); exp[2] = A[3]; exp[6] = A[7]
    assert np.array_equal(got, exp)
    below = og.alphas_q2(np.nextafter(a[[2, 6]], 0.0))
    assert np.allclose(below, A[[2, 6]], rtol=0, atol=1e-12) and not np.array_equal(below, A[[3, 7]])
    # malformed lines are refused: a triple knot (a one-knot sub-line), a repeated first or last knot
    for bad in ([1.0, 2.0, 2.0, 2.0, 3.0], [1.0, 1.0, 2.0, 3.0], [1.0, 2.0, 3.0, 3.0]):
        with pytest.raises(ValueError):
            og.set_alphas(np.array(bad), np.linspace(0.3, 0.1, len(bad)))
