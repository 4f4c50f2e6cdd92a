"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Integer results (region, sub-grid, cell) must be bit-exact; values obey the
tolerance of tests/parity.py (C-12)."""
import math

import numpy as np
import pytest
import torch

from paper_2302_03343_b200 import synth
from conftest import make_oracle_grid
from parity import assert_values, value_errors

pytestmark = pytest.mark.gpu

PATHS = ["direct", "binned"]


@pytest.fixture(scope="module")
def B():
    from paper_2302_03343_b200 import binding
    assert torch.cuda.is_available()
    binding.lib()
    return binding


def gpu_grid(B, spec, path="direct", n=0):
    g = B.PdfGrid.from_spec(spec, workspace_for=max(n, 1) if path != "direct" else 0)
    g.pdf_grid_set_option(B.PDF_OPT_PATH, {"direct": B.PDF_PATH_DIRECT, "binned": B.PDF_PATH_BINNED,
                                           "auto": B.PDF_PATH_AUTO}[path])
    return g


def knot_neighbour_queries(spec):
    """every knot and its nextafter neighbours on both axes, crossed with a few fixed partners"""
    xk = spec.x_knots.numpy()
    qk = np.unique(np.concatenate([q.numpy() for q in spec.q2_subgrids]))
    xs = np.concatenate([xk, np.nextafter(xk[1:], 0), np.nextafter(xk[:-1], 2)])
    qs = np.concatenate([qk, np.nextafter(qk[1:], 0), np.nextafter(qk[:-1], 1e300)])
    X = np.concatenate([xs, np.full(len(qs), 0.0123), np.full(len(qs), xk[0]), np.full(len(qs), xk[-1])])
    Q = np.concatenate([np.full(len(xs), float(qk[len(qk) // 2]) * 1.01), qs, qs, qs])
    return X, Q


def check_locate(B, og, g, x, q):
    ix, iq, isub, reg = og.locate(x, q)
    gx, gq, gs, gr = [t.cpu().numpy() for t in g.pdf_locate(torch.tensor(x).cuda(), torch.tensor(q).cuda())]
    assert np.array_equal(reg, gr) and np.array_equal(isub, gs)
    assert np.array_equal(ix, gx) and np.array_equal(iq, gq)


@pytest.mark.parametrize("cfg", ["c0", "c1"])
def test_locate_bitexact(B, oracle_mod, cfg):
    spec = synth.grid_c0() if cfg == "c0" else synth.grid_c1()
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec)
    x, q = synth.queries_c2(spec, 300_001, seed=17)
    check_locate(B, og, g, x.numpy(), q.numpy())
    X, Q = knot_neighbour_queries(spec)
    check_locate(B, og, g, X, Q)
    bad_x = np.array([0.0, -1.0, 1.5, np.nan, np.inf, 0.1, 0.1, 0.1])
    bad_q = np.array([10.0, 10.0, 10.0, 10.0, 10.0, 0.0, -3.0, np.nan])
    check_locate(B, og, g, bad_x, bad_q)


def test_path_logarithm(B):
    """pdf_log, the logarithm behind every abscissa of the path (C-1, C-5), against the host's log: <= 1 ulp apart
    over the whole positive range, subnormals, the neighbourhood of 1 and exact powers of two"""
    g = torch.Generator().manual_seed(12)
    parts = [torch.exp(torch.empty(4_000_000, dtype=torch.float64).uniform_(-700.0, 700.0, generator=g)),
             1.0 + torch.empty(1_000_000, dtype=torch.float64).uniform_(-0.3, 0.45, generator=g),
             1.0 + 10.0 ** torch.empty(200_000, dtype=torch.float64).uniform_(-16.0, -1.0, generator=g),
             1.0 - 10.0 ** torch.empty(200_000, dtype=torch.float64).uniform_(-16.0, -1.0, generator=g),
             2.0 ** torch.arange(-1074, 1024, dtype=torch.float64),
             torch.tensor([5e-324, 2.2250738585072014e-308, 2.225073858507201e-308, 1.0, 0.7071067811865476, 1.4142135623730951,
                           1.7976931348623157e308], dtype=torch.float64)]
    x = torch.cat(parts)
    got = B.pdf_log_f64(x.cuda()).cpu().numpy()
    ref = np.log(x.numpy())
    ulp = np.spacing(np.abs(ref))
    d = np.abs(got - ref) / np.where(ulp > 0, ulp, 5e-324)
    assert got[x.numpy() == 1.0].tolist() == [0.0] * int((x == 1.0).sum())
    print("\npdf_log: max |gpu - glibc| =", d.max(), "ulp; differing:", float(np.mean(d > 0)))
    assert d.max() <= 1.0


@pytest.mark.parametrize("path", PATHS)
def test_c0_parity(B, oracle_mod, path):
    """configs[0]: 1e5 queries strictly inside the 50x30 single-sub-grid grid"""
    spec = synth.grid_c0()
    n = 100_000
    x, q = synth.queries_inside(spec, n, synth.BASE_SEED + 10, strict=True)
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec, path, n)
    ref, S = og.xfxq2(spec.pids, x.numpy(), q.numpy(), want_scale=True)
    out = g.pdf_xfxq2(spec.pids, x.cuda(), q.cuda()).cpu().numpy()
    st = assert_values(out, ref, S, "c0", strict=1e-12)
    print("\nc0", path, st)
    assert st["frac_within_strict"] > 0.99
    assert g.pdf_error_count() == 0


@pytest.mark.parametrize("path", PATHS)
def test_c1_parity(B, oracle_mod, path):
    """configs[1] shape (1e6-query slice of the 1e7 recipe; several tiles and a ragged tail)"""
    spec = synth.grid_c1()
    n = 1_000_003
    x, q = synth.queries_inside(spec, n, synth.BASE_SEED + 11)
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec, path, n)
    ref, S = og.xfxq2(spec.pids, x.numpy(), q.numpy(), want_scale=True)
    out = g.pdf_xfxq2(spec.pids, x.cuda(), q.cuda()).cpu().numpy()
    print("\nc1", path, assert_values(out, ref, S, "c1", strict=1e-12))
    check_locate(B, og, g, x.numpy()[:200_000], q.numpy()[:200_000])


@pytest.mark.parametrize("path", PATHS)
def test_c2_extrapolation_parity(B, oracle_mod, path):
    """configs[2]: 5 % of the queries outside the grid (all five extrapolation classes)"""
    spec = synth.grid_c1()
    n = 1_000_000
    x, q = synth.queries_c2(spec, n)
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec, path, n)
    ref, S = og.xfxq2(spec.pids, x.numpy(), q.numpy(), want_scale=True)
    out = g.pdf_xfxq2(spec.pids, x.cuda(), q.cuda()).cpu().numpy()
    _, _, _, reg = og.locate(x.numpy(), q.numpy())
    for r in range(6):
        sel = reg == r
        assert sel.sum() > 1000
        print("\nc2", path, "region", r, assert_values(out[sel], ref[sel], S[sel], f"c2 region {r}", strict=1e-12 if r == 0 else None))
    a = g.pdf_alphas_q2(q.cuda()).cpu().numpy()
    aref = og.alphas_q2(q.numpy())
    assert np.max(np.abs(a - aref) / np.abs(aref)) < 1e-12


@pytest.mark.parametrize("path", PATHS)
def test_scan_lines_and_knots(B, oracle_mod, path):
    """the thesis' accuracy-scan pattern (Fig. 3.5) + every knot and its neighbours;
    P-1 on the GPU: stored node values come back bitwise"""
    spec = synth.grid_c1()
    og = make_oracle_grid(oracle_mod, spec)
    X, Q = synth.scan_lines(spec)
    Xk, Qk = knot_neighbour_queries(spec)
    x = np.concatenate([X.numpy(), Xk])
    q = np.concatenate([Q.numpy(), Qk])
    g = gpu_grid(B, spec, path, max(len(x), 196 * 54))
    ref, S = og.xfxq2(spec.pids, x, q, want_scale=True)
    out = g.pdf_xfxq2(spec.pids, torch.tensor(x).cuda(), torch.tensor(q).cuda()).cpu().numpy()
    assert_values(out, ref, S, "scan")
    for k, qk in enumerate(spec.q2_subgrids):
        top = len(qk) - 1 if k < len(spec.q2_subgrids) - 1 else len(qk)
        XX, QQ = torch.meshgrid(spec.x_knots, qk[:top], indexing="ij")
        got = g.pdf_xfxq2(spec.pids, XX.reshape(-1).cuda(), QQ.reshape(-1).cuda()).cpu()
        want = spec.block(0, k)[:, :top, :].reshape(-1, spec.nflav)
        assert torch.equal(got, want)


@pytest.mark.parametrize("path", PATHS)
def test_c3_members_parity(B, oracle_mod, path):
    """configs[3]: replica batch, per-query member index (20 members here; the 100-member grid runs in bench).
    Queries as configs[2] (5 % extrapolated), so every class crosses the member axis; on the binned
    path they are partitioned by member first (pdf_members.cuh)"""
    spec = synth.grid_c1(nmem=20)
    n = 400_037
    x, q = synth.queries_c2(spec, n, synth.BASE_SEED + 13)
    mem = synth.members(spec, n)
    mem[:3000] = 7                       # an uneven histogram: one member's run spans two chunks below
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec, path, n)
    ref, S = og.xfxq2(spec.pids, x.numpy(), q.numpy(), member=mem.numpy(), want_scale=True)
    out = g.pdf_xfxq2(spec.pids, x.cuda(), q.cuda(), member=mem.cuda()).cpu().numpy()
    assert_values(out, ref, S, "c3")
    assert g.pdf_error_count() == 0
    # invalid member ids, invalid x, and both at once: NaN rows, each query counted once
    bad, xb = mem.clone(), x.clone()
    bad[:5] = 20
    bad[5:9] = -1
    xb[7:12] = 2.0
    m = 50_000
    out = g.pdf_xfxq2(spec.pids, xb[:m].cuda(), q[:m].cuda(), member=bad[:m].cuda()).cpu().numpy()
    assert np.all(np.isnan(out[:12])) and not np.any(np.isnan(out[12:]))
    assert g.pdf_error_count() == 12
    assert_values(out[12:], ref[12:m], S[12:m], "c3 after bad rows")
    # a pid subset with an unknown pid, padded rows; small chunks so that runs span several chunks
    if path == "binned":
        g.pdf_grid_set_option(B.PDF_OPT_CHUNK, 8192)
    pids = [21, 2, 99, -3]
    o = torch.full((m, 6), -7.0, dtype=torch.float64, device="cuda")
    g.pdf_xfxq2(pids, x[:m].cuda(), q[:m].cuda(), out=o, member=mem[:m].cuda(), ld_out=6)
    o = o.cpu().numpy()
    cols = [spec.pids.index(21), spec.pids.index(2), None, spec.pids.index(-3)]
    for k, c in enumerate(cols):
        if c is None:
            assert np.all(o[:, k] == 0.0)
        else:
            assert_values(o[:, k], ref[:m, c], S[:m, c], f"c3 pid {pids[k]}")
    assert np.all(o[:, 4:] == -7.0)


@pytest.mark.parametrize("path", PATHS)
def test_c4_lumi_parity(B, oracle_mod, path):
    """configs[4]: luminosity; ~20 % of the events take the low-Q branch"""
    spec = synth.grid_c1()
    n = 300_000
    x1, x2, q2, w = synth.events_c4(n)
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec, path, n)
    ref, S = og.lumi(x1.numpy(), x2.numpy(), q2.numpy(), w.numpy(), want_scale=True)
    out = g.pdf_lumi(x1.cuda(), x2.cuda(), q2.cuda(), w.cuda()).cpu().numpy()
    assert_values(out, ref, S, "lumi")
    # invalid events
    x1b = x1[:64].clone()
    x1b[3] = 1.5
    x1b[7] = float("nan")
    out = g.pdf_lumi(x1b.cuda(), x2[:64].cuda(), q2[:64].cuda(), w[:64].cuda()).cpu().numpy()
    assert np.isnan(out[3]) and np.isnan(out[7]) and np.isnan(out).sum() == 2
    assert g.pdf_error_count() == 2


@pytest.mark.parametrize("path", PATHS)
def test_pids_ld_and_edge_sizes(B, oracle_mod, path):
    spec = synth.grid_c1()
    og = make_oracle_grid(oracle_mod, spec)
    g = gpu_grid(B, spec, path, 5000)
    x, q = synth.queries_c2(spec, 5000, seed=3)
    pids = [21, -3, 99, 0, 5]
    ref, S = og.xfxq2(pids, x.numpy(), q.numpy(), want_scale=True)
    out = g.pdf_xfxq2(pids, x.cuda(), q.cuda()).cpu().numpy()
    assert_values(out, ref, S, "pids")
    assert np.all(out[:, 2] == 0.0) and np.array_equal(out[:, 0], out[:, 3])
    # explicit leading dimension: untouched padding
    buf = torch.full((5000, 12), -7.0, dtype=torch.float64, device="cuda")
    g.pdf_xfxq2(spec.pids, x.cuda(), q.cuda(), out=buf, ld_out=12)
    ref11, S11 = og.xfxq2(spec.pids, x.numpy(), q.numpy(), want_scale=True)
    assert_values(buf[:, :11].cpu().numpy(), ref11, S11, "ld12")
    assert torch.all(buf[:, 11] == -7.0)
    # empty and ragged sizes
    for n in (0, 1, 31, 33, 127, 129, 1025):
        o = g.pdf_xfxq2(spec.pids, x[:n].cuda(), q[:n].cuda())
        assert o.shape == (n, 11)
        if n:
            assert_values(o.cpu().numpy(), ref11[:n], S11[:n], f"n={n}")
    # invalid rows -> NaN + counter
    bx = x[:10].clone()
    bq = q[:10].clone()
    bx[0], bx[1], bq[2], bq[3], bx[4] = 0.0, 1.0000001, -1.0, float("inf"), float("nan")
    g.pdf_error_count()
    o = g.pdf_xfxq2(spec.pids, bx.cuda(), bq.cuda()).cpu().numpy()
    assert np.all(np.isnan(o[:5])) and not np.any(np.isnan(o[5:]))
    assert g.pdf_error_count() == 5 and g.pdf_error_count() == 0


def test_tiny_nonuniform_grids(B, oracle_mod):
    """degenerate shapes: 2-knot axes, 2- and 3-knot sub-grids, non-uniform knots, all regions"""
    rng = np.random.default_rng(4)
    for nx, nq in [(2, [2]), (3, [3]), (4, [2, 3]), (5, [4, 2, 5]), (3, [2, 2, 2])]:
        spec = synth.tiny_grid(200 + nx + len(nq), nx, nq, nflav=3)
        og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec)
        xmin, xmax, qmin, qmax = og.limits()
        n = 4000
        x = np.exp(rng.uniform(math.log(xmin) - 3, math.log(xmax), n)).clip(max=xmax)
        q = np.exp(rng.uniform(math.log(qmin) - 3, math.log(qmax) + 3, n))
        Xk, Qk = knot_neighbour_queries(spec)
        x, q = np.concatenate([x, Xk]), np.concatenate([q, Qk])
        check_locate(B, og, g, x, q)
        ref, S = og.xfxq2(spec.pids, x, q, want_scale=True)
        out = g.pdf_xfxq2(spec.pids, torch.tensor(x).cuda(), torch.tensor(q).cuda()).cpu().numpy()
        assert_values(out, ref, S, f"tiny {nx} {nq}")


def test_alphas_modes_and_nodes(B, oracle_mod):
    spec = synth.grid_c1()
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec)
    aq = spec.alphas_q2
    assert torch.equal(g.pdf_alphas_q2(aq.cuda()).cpu(), spec.alphas_val)
    q = torch.exp(torch.linspace(math.log(1e-3), math.log(1e13), 200_001, dtype=torch.float64))
    a = g.pdf_alphas_q2(q.cuda()).cpu().numpy()
    ref = og.alphas_q2(q.numpy())
    assert np.max(np.abs(a - ref) / ref) < 1e-12
    g.pdf_grid_set_option(B.PDF_OPT_ALPHAS_MODE, B.PDF_ALPHAS_LOGGRAD)
    og.set_alphas(spec.alphas_q2.numpy(), spec.alphas_val.numpy(), mode=oracle_mod.ALPHAS_LOGGRAD)
    a = g.pdf_alphas_q2(q.cuda()).cpu().numpy()
    ref = og.alphas_q2(q.numpy())
    assert np.max(np.abs(a - ref) / ref) < 1e-12
    bad = torch.tensor([0.0, -1.0, float("nan")], dtype=torch.float64)
    assert torch.all(torch.isnan(g.pdf_alphas_q2(bad.cuda())))


def test_host_calls_match_device_calls(B, oracle_mod):
    spec = synth.grid_c1()
    g = gpu_grid(B, spec, "auto", 1 << 22)
    n = (1 << 22) + 12345          # more than one pipeline chunk
    x, q = synth.queries_c2(spec, n, seed=21)
    out_h = torch.empty((n, 11), dtype=torch.float64).pin_memory()
    g.pdf_xfxq2_host(spec.pids, x.pin_memory(), q.pin_memory(), out_h)
    out_d = g.pdf_xfxq2(spec.pids, x.cuda(), q.cuda()).cpu()
    # same kernels either way; only the chunking differs (overflow entries may take the generic order)
    assert torch.equal(torch.isnan(out_h), torch.isnan(out_d))
    assert torch.allclose(torch.nan_to_num(out_h), torch.nan_to_num(out_d), rtol=1e-13, atol=1e-300)
    a_h = torch.empty(n, dtype=torch.float64)
    g.pdf_alphas_q2_host(q, a_h)
    assert torch.equal(a_h, g.pdf_alphas_q2(q.cuda()).cpu())
    x1, x2, q2, w = synth.events_c4(100_000)
    l_h = torch.empty(100_000, dtype=torch.float64)
    g.pdf_lumi_host(x1, x2, q2, w, l_h)
    assert torch.equal(l_h, g.pdf_lumi(x1.cuda(), x2.cuda(), q2.cuda(), w.cuda()).cpu())


def test_missing_state_and_workspace_errors(B):
    spec = synth.grid_c0()
    g = B.PdfGrid(spec.x_knots, spec.q2_subgrids, spec.values, spec.pids)
    q = torch.ones(4, dtype=torch.float64, device="cuda")
    with pytest.raises(B.PdfGridError):
        g.pdf_alphas_q2(q)
    with pytest.raises(B.PdfGridError):
        g.pdf_lumi(q, q, q, q)
    g.pdf_grid_set_option(B.PDF_OPT_PATH, B.PDF_PATH_BINNED)
    if g.pdf_workspace_bytes(4) > 0:
        with pytest.raises(B.PdfGridError):
            g.pdf_xfxq2(spec.pids, q * 0.1, q * 10)


def test_binned_ring_reuse_and_overflow(B, oracle_mod):
    """the persistent kernel's chunk ring (many small chunks) and the overflow list (queries piled
    into a handful of cells so that bins exceed their capacity)"""
    spec = synth.grid_c1()
    og = make_oracle_grid(oracle_mod, spec)
    g = B.PdfGrid.from_spec(spec)
    g.pdf_grid_set_option(B.PDF_OPT_PATH, B.PDF_PATH_BINNED)
    g.pdf_grid_set_option(B.PDF_OPT_CHUNK, 4096)
    n = 150_001                                   # 37 chunks through a ring of 3
    g.attach_workspace(n)
    x, q = synth.queries_c2(spec, n, seed=31)
    ref, S = og.xfxq2(spec.pids, x.numpy(), q.numpy(), want_scale=True)
    for _ in range(2):                            # second call: control block re-initialised
        out = g.pdf_xfxq2(spec.pids, x.cuda(), q.cuda()).cpu().numpy()
        assert_values(out, ref, S, "ring")
    # skew: everything inside 3 x-cells and 2 Q2-cells, plus one corner class
    g.pdf_grid_set_option(B.PDF_OPT_CHUNK, 1 << 16)
    n = 200_000
    g.attach_workspace(n)
    gen = torch.Generator().manual_seed(5)
    xs = torch.exp(torch.rand(n, generator=gen, dtype=torch.float64) * 0.3 + math.log(1e-3))
    qs = torch.exp(torch.rand(n, generator=gen, dtype=torch.float64) * 0.9 + math.log(100.0))
    xs[:20_000] = 1e-11
    qs[:20_000] = 0.3
    ref, S = og.xfxq2(spec.pids, xs.numpy(), qs.numpy(), want_scale=True)
    out = g.pdf_xfxq2(spec.pids, xs.cuda(), qs.cuda()).cpu().numpy()
    assert_values(out, ref, S, "skew")


@pytest.mark.parametrize("n", [262_144, 1_000_003])
def test_binned_first_calls_in_a_fresh_process(n):
    """regression: shared-memory atomics of the binned kernel were read across a barrier before they
    had landed, only when the pipeline's waits were really taken (first calls of a process)"""
    import os
    import subprocess
    import sys
    script = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cold_check.py")
    for _ in range(2):
        r = subprocess.run([sys.executable, script, str(n)], capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]


@pytest.mark.parametrize("path", ["direct", "auto"])
def test_table33_workload_parity(B, oracle_mod, path):
    """NEXT-3, the multi-member workload of Table 3.3: all 11 flavours on the fixed
    2415-point x-grid at one Q2 for every member (50 members here; bench.py times N_rep = 10 ... 400).
    Every row against the oracle, the cell indices bit-exact; all members of an x-point share one cell."""
    nrep = 50
    spec = synth.grid_c1(nmem=nrep)
    x, q, mem = synth.queries_table33(nrep)
    n = x.numel()
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec, path, n)
    ref, S = og.xfxq2(spec.pids, x.numpy(), q.numpy(), member=mem.numpy(), want_scale=True)
    out = g.pdf_xfxq2(spec.pids, x.cuda(), q.cuda(), member=mem.cuda()).cpu().numpy()
    assert out.shape == (nrep * synth.TABLE33_NX, 11)
    assert_values(out, ref, S, "table33")
    assert g.pdf_error_count() == 0
    check_locate(B, og, g, x.numpy()[: synth.TABLE33_NX], q.numpy()[: synth.TABLE33_NX])
    # members differ (lognormal noise), so a wrong member stride cannot pass: rows of two members at one x-point
    assert not np.allclose(out[: synth.TABLE33_NX], out[synth.TABLE33_NX: 2 * synth.TABLE33_NX], rtol=1e-6, atol=0)


def _xgrid_call(B, g, kernel, pids, x, q, members, reps):
    """pdf_xfxq2_xgrid with the member list repeated `reps` times (large lists reach the cell-shared kernel under
    PDF_PATH_AUTO); checks which kernel ran and that every repeat gives the same rows; returns the first copy."""
    nrep = members.numel()
    mm = members.repeat(reps)
    B.pdf_profile_enable(True)
    out = g.pdf_xfxq2_xgrid(pids, x.cuda(), q.cuda(), mm.numel(), members=mm.cuda())
    torch.cuda.synchronize()
    names = [n for n, _ in B.pdf_profile_read(64)]
    B.pdf_profile_enable(False)
    assert names == [kernel], names
    out = out.cpu()
    for k in range(1, reps):
        assert torch.equal(out[k * nrep:(k + 1) * nrep].nan_to_num(nan=-1.0), out[:nrep].nan_to_num(nan=-1.0))
    return out[:nrep]


XGRID_KERNELS = [("direct", "k_xfxq2_xgrid", 1), ("auto", "k_xfxq2_xgrid", 1), ("auto", "k_xfxq2_xgrid_cell", 0)]


@pytest.mark.parametrize("path,kernel,reps", XGRID_KERNELS)
def test_xgrid_matches_member_major_calls(B, oracle_mod, path, kernel, reps):
    """pdf_xfxq2_xgrid (NEXT-3): every member on one shared point list == pdf_xfxq2_ex on the member-major
    expansion, bit for bit against its direct path, and within tolerance of the oracle; the per-point kernel
    and the (member, cell)-shared kernel (PDF_PATH_AUTO, large member lists)."""
    nrep = 23
    spec = synth.grid_c1(nmem=nrep)
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec, path)
    xg = synth.xgrid_table33()
    npts = xg.numel()
    q = torch.full((npts,), synth.TABLE33_Q2, dtype=torch.float64)
    x, qq, mem = synth.queries_table33(nrep)
    g.pdf_grid_set_option(B.PDF_OPT_PATH, B.PDF_PATH_DIRECT)
    want = g.pdf_xfxq2(spec.pids, x.cuda(), qq.cuda(), member=mem.cuda()).cpu()
    g.pdf_grid_set_option(B.PDF_OPT_PATH, B.PDF_PATH_DIRECT if path == "direct" else B.PDF_PATH_AUTO)
    got = _xgrid_call(B, g, kernel, spec.pids, xg, q, torch.arange(nrep, dtype=torch.int32), reps or 8)
    assert got.shape == (nrep, npts, 11)
    assert torch.equal(got.reshape(-1, 11), want)
    ref, S = og.xfxq2(spec.pids, x.numpy(), qq.numpy(), member=mem.numpy(), want_scale=True)
    assert_values(got.reshape(-1, 11).numpy(), ref, S, "xgrid")
    assert g.pdf_error_count() == 0


@pytest.mark.parametrize("path,kernel,reps", XGRID_KERNELS)
def test_xgrid_edge_cases(B, oracle_mod, path, kernel, reps):
    """ragged point count, extrapolated and invalid points, a member list with repeats and a bad id, a pid
    subset with an unknown pid, padded rows; error count = invalid (point, member) pairs"""
    spec = synth.grid_c1(nmem=7)
    og, g = make_oracle_grid(oracle_mod, spec), gpu_grid(B, spec, path)
    npts = 1000 + 13
    x, q = synth.queries_c2(spec, npts, synth.BASE_SEED + 77)        # 5 % extrapolated, all classes, unsorted
    x[5] = 2.0                                                        # x > x_max: invalid
    x[600] = float("nan")
    members = torch.tensor([3, 0, 6, 3, 7, 1], dtype=torch.int32)     # 7 is out of range
    nrep = members.numel()
    reps = reps or 64

    def check(got, pids_, xs, qs, what):
        n_bad = 0
        for r, m in enumerate(members.tolist()):
            if m >= spec.nmem:
                assert np.isnan(got[r]).all()
                n_bad += xs.numel()
                continue
            ref, S = og.xfxq2(pids_, xs.numpy(), qs.numpy(), member=np.full(xs.numel(), m, dtype=np.int32), want_scale=True)
            assert_values(got[r], ref, S, f"{what} member {m}")
            n_bad += int(np.isnan(ref[:, 0]).sum())
        return n_bad

    # pid subset with an unknown pid, padded rows: always the per-point kernel
    pids = [21, 2, 99, -5]
    out = torch.full((nrep, npts, 6), -7.0, dtype=torch.float64, device="cuda")
    g.pdf_xfxq2_xgrid(pids, x.cuda(), q.cuda(), nrep, members=members.cuda(), out=out, ld_out=6)
    out = out.cpu().numpy()
    assert np.all(out[:, :, 4:] == -7.0)                              # padding untouched
    n_bad = check(out[:, :, :4], pids, x, q, "xgrid subset")
    ok_rows = ~np.isnan(out[0, :, 0])
    assert np.all(out[0, ok_rows, 2] == 0.0)                          # unknown pid -> 0.0
    assert g.pdf_error_count() == n_bad
    # all 11 flavours, contiguous rows, on the same ragged, mixed, unsorted point list (runs of one point)
    got = _xgrid_call(B, g, kernel, spec.pids, x, q, members, reps).numpy()
    n_bad = check(got, spec.pids, x, q, "xgrid full")
    assert g.pdf_error_count() == n_bad * reps
    # sorted points at two Q2 values: runs of many points, run boundaries inside and across tiles
    xs = torch.sort(x[torch.isfinite(x) & (x <= 1.0)])[0][:900]
    qs = torch.where(torch.arange(xs.numel()) % 200 < 100, torch.tensor(50.0, dtype=torch.float64),
                     torch.tensor(3.0e4, dtype=torch.float64))
    got = _xgrid_call(B, g, kernel, spec.pids, xs, qs, members, reps + 8).numpy()
    check(got, spec.pids, xs, qs, "xgrid sorted")
    g.pdf_error_count()
    # empty calls are no-ops
    g.pdf_xfxq2_xgrid(spec.pids, x[:0].cuda(), q[:0].cuda(), 3)
    g.pdf_xfxq2_xgrid(spec.pids, x.cuda(), q.cuda(), 0)
