"""Seeded synthetic workloads (grids, queries, events) shaped like the thesis' inputs.

This module holds NONE of the method's arithmetic (no interpolation, no cell
search): it only draws the inputs BASELINE.json's five configs describe, so that
the CPU oracle (tests) and the CUDA path (tests, bench) can be fed the very same
arrays.  It imports neither ``oracle`` nor the CUDA binding.

Stand-in note (Table 3.3): the thesis
measures on real LHAPDF sets (NNPDF3.1 NLO, MMHT2014 NLO).  Those files are not
available here and are not reconstructed; the grids below take only their shape
(knot counts, ranges, log spacing, sub-grid thresholds, 11 flavours, ~100
members).  Recipe: DESIGN.md, "Input recipe".

Everything is a ``torch.float64`` / ``torch.int32`` tensor created with a seeded
``torch.Generator`` on the requested device (CPU for the tests that call the
oracle; ``cuda`` for the 1e8-query bench, so inputs are born in HBM).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Optional

import torch

BASE_SEED = 23020334
PIDS = (-5, -4, -3, -2, -1, 21, 1, 2, 3, 4, 5)
MC2 = 1.51 ** 2          # 2.2801 GeV^2   (BASELINE.json configs[1])
MB2 = 4.92 ** 2          # 24.2064 GeV^2  (m_b = 4.92 GeV)
S_HADRONIC = 13000.0 ** 2


@dataclass
class GridSpec:
    """Host-side description of one PDF grid in the LHAPDF layout (L1714)."""
    x_knots: torch.Tensor                 # [nx]
    q2_subgrids: List[torch.Tensor]       # per sub-grid [nq_k]; last knot == first of next
    values: torch.Tensor                  # flat [nmem][sub-grid blocks [nx][nq_k][nflav]]
    pids: tuple = PIDS
    nmem: int = 1
    alphas_q2: Optional[torch.Tensor] = None
    alphas_val: Optional[torch.Tensor] = None
    coupling: Optional[torch.Tensor] = None
    params: dict = field(default_factory=dict)

    @property
    def nx(self):
        return int(self.x_knots.numel())

    @property
    def nq(self):
        return [int(q.numel()) for q in self.q2_subgrids]

    @property
    def nflav(self):
        return len(self.pids)

    def member_values(self, m: int) -> torch.Tensor:
        stride = self.values.numel() // self.nmem
        return self.values[m * stride:(m + 1) * stride]

    def block(self, m: int, k: int) -> torch.Tensor:
        """[nx][nq_k][nflav] view of sub-grid k of member m."""
        mv = self.member_values(m)
        off = 0
        for kk in range(k):
            off += self.nx * self.nq[kk] * self.nflav
        n = self.nx * self.nq[k] * self.nflav
        return mv[off:off + n].view(self.nx, self.nq[k], self.nflav)


def _gen(seed: int, device="cpu") -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def _uniform(g, n, lo, hi, device="cpu"):
    return lo + (hi - lo) * torch.rand(n, generator=g, dtype=torch.float64, device=device)


def _geomspace(lo: float, hi: float, n: int) -> torch.Tensor:
    t = torch.linspace(0.0, 1.0, n, dtype=torch.float64)
    k = torch.exp(math.log(lo) + t * (math.log(hi) - math.log(lo)))
    k[0], k[-1] = lo, hi                  # end knots exact (thresholds must match bitwise)
    return k


def _flavour_params(g):
    nf = len(PIDS)
    a = _uniform(g, nf, -0.3, 0.5)
    b = _uniform(g, nf, 2.0, 6.0)
    c = _uniform(g, nf, -1.0, 1.0)
    d = _uniform(g, nf, -1.0, 1.0)
    return a, b, c, d


def _node_values(x, q2, a, b, c, d):
    """x^a (1-x)^b (1 + c sqrt x)(1 + d ln Q2) on the knot mesh -> [nx][nq][nflav]."""
    X = x[:, None, None]
    Q = q2[None, :, None]
    return (X ** a) * ((1.0 - X) ** b) * (1.0 + c * torch.sqrt(X)) * (1.0 + d * torch.log(Q))


def grid_c0(seed: int = BASE_SEED + 0) -> GridSpec:
    """configs[0]: 50 x-knots in [1e-9,1], 30 Q2 knots in [2.72,1e10], one sub-grid."""
    g = _gen(seed)
    a, b, c, d = _flavour_params(g)
    x = _geomspace(1e-9, 1.0, 50)
    q = _geomspace(2.72, 1e10, 30)
    v = _node_values(x, q, a, b, c, d)
    return GridSpec(x, [q], v.reshape(-1).contiguous(), params=dict(a=a, b=b, c=c, d=d))


def grid_c1(seed: int = BASE_SEED + 1, nmem: int = 1, sigma: float = 0.05,
            q2min: float = 1.0) -> GridSpec:
    """configs[1]: 196 x-knots in [1e-9,1]; sub-grids of 6, 8, 40 Q2 knots split at
    m_c^2 and m_b^2, top 1e10; charm / bottom identically zero below their
    thresholds.  nmem > 1 gives configs[3] (lognormal member noise, sigma)."""
    g = _gen(seed)
    a, b, c, d = _flavour_params(g)
    x = _geomspace(1e-9, 1.0, 196)
    subs = [_geomspace(q2min, MC2, 6), _geomspace(MC2, MB2, 8), _geomspace(MB2, 1e10, 40)]
    blocks = []
    for k, q in enumerate(subs):
        v = _node_values(x, q, a, b, c, d)
        for col, pid in enumerate(PIDS):
            if abs(pid) == 4 and k < 1:
                v[:, :, col] = 0.0
            if abs(pid) == 5 and k < 2:
                v[:, :, col] = 0.0
        blocks.append(v.reshape(-1))
    base = torch.cat(blocks)
    if nmem == 1:
        vals = base
    else:
        noise = torch.randn(nmem, base.numel(), generator=g, dtype=torch.float64)
        vals = (base[None, :] * torch.exp(sigma * noise)).reshape(-1)
    spec = GridSpec(x, subs, vals.contiguous(), nmem=nmem, params=dict(a=a, b=b, c=c, d=d))
    # coupling (configs[4]) and alpha_s knots (configs[2]) are drawn after the member noise
    spec.coupling = _uniform(g, len(PIDS) ** 2, 0.0, 1.0).view(len(PIDS), len(PIDS)).contiguous()
    eta = float(_uniform(g, 1, 0.8, 1.2))
    aq = _geomspace(q2min, 1e10, 60)
    frac = (torch.arange(60, dtype=torch.float64) / 59.0) ** eta
    spec.alphas_q2 = aq
    spec.alphas_val = 1.0 / (1.0 / 0.35 + (1.0 / 0.08 - 1.0 / 0.35) * frac)
    return spec


def tiny_grid(seed: int, nx: int, nq: List[int], nflav: int = 2, nmem: int = 1,
              jitter: float = 0.35) -> GridSpec:
    """Deliberately NON-uniform tiny grid with random values (brute-force pins)."""
    g = _gen(seed)

    def knots(lo, hi, n):
        t = torch.linspace(0.0, 1.0, n, dtype=torch.float64)
        if n > 2:
            t[1:-1] += jitter / (n - 1) * (2.0 * torch.rand(n - 2, generator=g, dtype=torch.float64) - 1.0)
        k = torch.exp(math.log(lo) + t * (math.log(hi) - math.log(lo)))
        k[0], k[-1] = lo, hi
        return k

    x = knots(1e-4, 1.0, nx)
    edges = torch.exp(torch.linspace(math.log(1.5), math.log(1e4), len(nq) + 1, dtype=torch.float64))
    subs = [knots(float(edges[k]), float(edges[k + 1]), n) for k, n in enumerate(nq)]
    tot = nx * sum(nq) * nflav * nmem
    vals = 2.0 * torch.rand(tot, generator=g, dtype=torch.float64) - 0.5
    pids = tuple(range(1, nflav + 1))
    return GridSpec(x, subs, vals, pids=pids, nmem=nmem)


# ---------------------------------------------------------------------------
# queries
# ---------------------------------------------------------------------------
def queries_inside(spec: GridSpec, n: int, seed: int, device="cpu", strict: bool = False):
    """ln x ~ U(ln xmin, ln xmax), ln Q2 ~ U(ln Q2min, ln Q2max) (configs[0], [1])."""
    g = _gen(seed, device)
    xmin, xmax = float(spec.x_knots[0]), float(spec.x_knots[-1])
    qmin, qmax = float(spec.q2_subgrids[0][0]), float(spec.q2_subgrids[-1][-1])
    x = torch.exp(_uniform(g, n, math.log(xmin), math.log(xmax), device))
    q = torch.exp(_uniform(g, n, math.log(qmin), math.log(qmax), device))
    if strict:
        x.clamp_(math.nextafter(xmin, 2.0), math.nextafter(xmax, 0.0))
        q.clamp_(math.nextafter(qmin, 1e300), math.nextafter(qmax, 0.0))
    else:
        x.clamp_(xmin, xmax)
        q.clamp_(qmin, qmax)
    return x, q


def queries_c2(spec: GridSpec, n: int, seed: int = BASE_SEED + 2, device="cpu"):
    """configs[2]: 95 % inside; 2 % low-x; 1.25 % low-Q; 1.25 % high-Q; 0.25 % each corner."""
    g = _gen(seed, device)
    xmin, xmax = float(spec.x_knots[0]), float(spec.x_knots[-1])
    qmin, qmax = float(spec.q2_subgrids[0][0]), float(spec.q2_subgrids[-1][-1])
    lx = _uniform(g, n, math.log(xmin), math.log(xmax), device)
    lq = _uniform(g, n, math.log(qmin), math.log(qmax), device)
    sel = torch.rand(n, generator=g, dtype=torch.float64, device=device)
    lx_low = _uniform(g, n, math.log(xmin) - math.log(1e3), math.log(xmin), device)
    lq_low = _uniform(g, n, math.log(qmin) - math.log(100.0), math.log(qmin), device)
    lq_high = _uniform(g, n, math.log(qmax), math.log(qmax) + math.log(100.0), device)
    lowx = ((sel >= 0.95) & (sel < 0.97)) | (sel >= 0.995)
    lowq = ((sel >= 0.97) & (sel < 0.9825)) | ((sel >= 0.995) & (sel < 0.9975))
    highq = ((sel >= 0.9825) & (sel < 0.995)) | (sel >= 0.9975)
    x = torch.exp(torch.where(lowx, lx_low, lx))
    q = torch.exp(torch.where(lowq, lq_low, torch.where(highq, lq_high, lq)))
    x.clamp_(max=xmax)
    return x, q


def members(spec: GridSpec, n: int, seed: int = BASE_SEED + 3, device="cpu"):
    g = _gen(seed + 7919, device)
    return torch.randint(0, spec.nmem, (n,), generator=g, device=device, dtype=torch.int32)


def events_c4(n: int, seed: int = BASE_SEED + 4, device="cpu"):
    """configs[4]: x1, x2 log-uniform in [1e-6,1], Q2 = fl(fl(x1 x2) s), w ~ U(0,1)."""
    g = _gen(seed, device)
    x1 = torch.exp(_uniform(g, n, math.log(1e-6), 0.0, device)).clamp_(max=1.0)
    x2 = torch.exp(_uniform(g, n, math.log(1e-6), 0.0, device)).clamp_(max=1.0)
    q2 = (x1 * x2) * S_HADRONIC
    w = torch.rand(n, generator=g, dtype=torch.float64, device=device)
    return x1, x2, q2, w


# ---- NEXT-3: the multi-member workload of Table 3.3 ---------------------------
TABLE33_NX = 2415                 # "a grid of 2415 points in x" (Table 3.3 caption)
TABLE33_NREP = (10, 50, 100, 200, 300, 400)
TABLE33_Q2 = 1.65 ** 2            # the thesis gives no scale: FastKernel tables take the PDFs at the fit's
                                  # initial scale, Q0 = 1.65 GeV for NNPDF3.1 (reading)


def xgrid_table33() -> torch.Tensor:
    """2415 fixed x-points shaped like a FastKernel x-grid: log-spaced in [1e-7, 0.1), then
    linear in [0.1, 1).  Deterministic (no seed): the workload is structured, not sampled."""
    nlog = TABLE33_NX // 2
    nlin = TABLE33_NX - nlog
    lo = _geomspace(1e-7, 0.1, nlog + 1)[:-1]
    hi = torch.linspace(0.1, 1.0, nlin + 1, dtype=torch.float64)[:-1]
    return torch.cat([lo, hi]).contiguous()


def queries_table33(nrep: int, device="cpu"):
    """member-major (member, x-point) queries: every member is evaluated on the same x-grid at
    one fixed Q2 (all 11 flavours are requested by the caller).  Returns x, q2, member."""
    xg = xgrid_table33().to(device)
    x = xg.repeat(nrep)
    q2 = torch.full((nrep * TABLE33_NX,), TABLE33_Q2, dtype=torch.float64, device=device)
    mem = torch.arange(nrep, dtype=torch.int32, device=device).repeat_interleave(TABLE33_NX)
    return x.contiguous(), q2, mem.contiguous()


def scan_lines(spec: GridSpec, npts: int = 400):
    """The thesis' accuracy-scan pattern (Fig. 3.5 caption, L1846): vary x at
    several fixed Q, and Q at several fixed x."""
    xmin, xmax = float(spec.x_knots[0]), float(spec.x_knots[-1])
    qmin, qmax = float(spec.q2_subgrids[0][0]), float(spec.q2_subgrids[-1][-1])
    xs = torch.exp(torch.linspace(math.log(xmin), math.log(xmax), npts, dtype=torch.float64)).clamp_(xmin, xmax)
    qs = torch.exp(torch.linspace(math.log(qmin), math.log(qmax), npts, dtype=torch.float64)).clamp_(qmin, qmax)
    X, Q = [], []
    for qfix in (qmin * 1.7, 10.0 ** 2, 100.0 ** 2, 1e4 ** 2):
        if qmin <= qfix <= qmax:
            X.append(xs)
            Q.append(torch.full_like(xs, qfix))
    for xfix in (1e-7, 1e-4, 1e-2, 0.3, 0.9):
        X.append(torch.full_like(qs, xfix))
        Q.append(qs)
    return torch.cat(X), torch.cat(Q)
