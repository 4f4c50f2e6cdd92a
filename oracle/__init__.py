"""TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes binding of the plain CPU fp64 oracle in ``oracle/pdf_oracle.c`` (written
from PAPER.md section 3.2; see the C header for the citations).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import this package.  It imports nothing from
``paper_2302_03343_b200`` and shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pdf_oracle.c")
_HDR = os.path.join(_HERE, "pdf_oracle.h")
_SRC_MC = os.path.join(_HERE, "mc_oracle.c")
_HDR_MC = os.path.join(_HERE, "mc_oracle.h")
_LIB = os.path.join(_HERE, "libpdf_oracle.so")

REGION_INTERIOR, REGION_LOWX, REGION_LOWQ, REGION_HIGHQ = 0, 1, 2, 3
REGION_LOWX_LOWQ, REGION_LOWX_HIGHQ, REGION_INVALID = 4, 5, 6
ALPHAS_FREEZE, ALPHAS_LOGGRAD = 0, 1
EXTRAP_CONTINUATION, EXTRAP_FREEZE, EXTRAP_ERROR = 0, 1, 2


# Parity metric C-12: |gpu - ref| <= REL |ref| + FLOOR_S S[...,0] + FLOOR_T S[...,1].
# REL is north_star's 1e-12.  FLOOR_S multiplies sum |Wx Wq V| (rounding of the 16-term stencil sum: each
# side loses up to 16 x 2^-53 of it in the worst case, ~4e-16 typically); FLOOR_T multiplies the
# t-sensitivity (each side's t carries a few 2^-52 (1 + |ln v|/delta) of rounding).  The values are the
# tightest that the measured errors allow with a margin (C-12 lists the measured worst ratios).
REL = 1e-12
FLOOR_S = 1e-15
FLOOR_T = 2 * 2.0 ** -52


def tolerance(ref, scale):
    """element-wise parity tolerance from the oracle's value and its two condition numbers"""
    ref, scale = np.asarray(ref), np.asarray(scale)
    return REL * np.abs(ref) + FLOOR_S * scale[..., 0] + FLOOR_T * scale[..., 1]


def build(force: bool = False, variant: str = "") -> str:
    """Compile the oracle with gcc (-O2, OpenMP, no FMA contraction).  `variant` = a compile-time
    switch of pdf_oracle.c (e.g. "ORACLE_S3_BILINEAR"), built beside the default library."""
    out = _LIB if not variant else os.path.join(_HERE, f"libpdf_oracle_{variant.lower()}.so")
    stale = (not os.path.exists(out)) or any(
        os.path.getmtime(p) > os.path.getmtime(out) for p in (_SRC, _HDR, _SRC_MC, _HDR_MC))
    if force or stale:
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp",
               "-ffp-contract=off", "-Wall", "-Wextra", *( [f"-D{variant}"] if variant else []),
               "-o", out + ".tmp", _SRC, _SRC_MC, "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
        os.replace(out + ".tmp", out)
    return out


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p
        ll = C.c_longlong
        L.oracle_grid_create.argtypes = [C.POINTER(vp), C.c_int, dp, C.c_int, ip, dp, dp, C.c_int, ip, C.c_int]
        L.oracle_grid_set_alphas.argtypes = [vp, C.c_int, dp, dp]
        L.oracle_grid_set_alphas_mode.argtypes = [vp, C.c_int]
        L.oracle_grid_set_extrapolation.argtypes = [vp, C.c_int]
        L.oracle_grid_set_coupling.argtypes = [vp, dp]
        L.oracle_grid_limits.argtypes = [vp, dp, dp, dp, dp]
        L.oracle_grid_destroy.argtypes = [vp]
        L.oracle_locate.argtypes = [vp, ll, dp, dp, ip, ip, ip, ip]
        L.oracle_xfxq2.argtypes = [vp, ip, C.c_int, ll, dp, dp, ip, dp, dp]
        L.oracle_alphas_q2.argtypes = [vp, ll, dp, dp]
        L.oracle_lumi.argtypes = [vp, ll, dp, dp, dp, dp, dp, dp]
        L.oracle_interior_order.argtypes = [vp, C.c_int, C.c_int, C.c_int, ll, dp, dp, dp]
        L.oracle_weights_1d.argtypes = [C.c_int, dp, C.c_double, C.c_int, dp]
        L.oracle_num_threads.restype = C.c_int
        L.oracle_rambo_w0.argtypes = [C.c_int, C.c_double]
        L.oracle_rambo_w0.restype = C.c_double
        L.oracle_rambo.argtypes = [ll, C.c_int, dp, dp, dp, C.c_double, dp, dp]
        L.oracle_vegas_map.argtypes = [C.c_int, C.c_int, dp, ll, dp, dp, dp, ip]
        L.oracle_vegas_accumulate.argtypes = [C.c_int, C.c_int, ll, dp, dp, ip, dp, dp]
        L.oracle_vegas_estimate.argtypes = [ll, dp, dp, dp]
        L.oracle_vegas_refine.argtypes = [C.c_int, C.c_int, dp, C.c_double, dp]
        L.oracle_vegas_combine.argtypes = [C.c_int, dp, dp, dp, dp, dp]
        L.oracle_unweight.argtypes = [ll, dp, dp, dp, C.POINTER(C.c_ubyte), C.POINTER(ll)]
        _lib = L
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(C.POINTER(C.c_int))


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def weights_1d(knots_log, wlog: float, cell: int) -> np.ndarray:
    k, kp = _d(knots_log)
    w = np.zeros(4)
    rc = lib().oracle_weights_1d(len(k), kp, float(wlog), int(cell), w.ctypes.data_as(C.POINTER(C.c_double)))
    if rc:
        raise ValueError(f"oracle_weights_1d: {rc}")
    return w


class OracleGrid:
    """Handle on an oracle grid.  ``values`` is [nmem] lists of per-sub-grid
    arrays [nx][nq_k][nflav], or the flat concatenation the C call takes."""

    def __init__(self, x_knots, q2_subgrids, values, pids, nmem: int = 1):
        self._h = C.c_void_p()
        x, xp = _d(x_knots)
        nq = [len(q) for q in q2_subgrids]
        q2, qp = _d(np.concatenate([np.asarray(q, dtype=np.float64) for q in q2_subgrids]))
        nqa, nqp = _i(nq)
        v, vp = _d(np.asarray(values, dtype=np.float64).ravel())
        pid, pp = _i(pids)
        expect = len(x) * sum(nq) * len(pid) * nmem
        if v.size != expect:
            raise ValueError(f"values has {v.size} entries, expected {expect}")
        rc = lib().oracle_grid_create(C.byref(self._h), len(x), xp, len(nq), nqp, qp, vp, len(pid), pp, nmem)
        if rc:
            raise ValueError(f"oracle_grid_create failed: {rc}")
        self.nflav, self.nmem = len(pid), nmem

    def close(self):
        if self._h:
            lib().oracle_grid_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_alphas(self, q2_knots, values, mode: int = ALPHAS_FREEZE):
        q, qp = _d(q2_knots)
        v, vp = _d(values)
        if lib().oracle_grid_set_alphas(self._h, len(q), qp, vp):
            raise ValueError("oracle_grid_set_alphas failed")
        if lib().oracle_grid_set_alphas_mode(self._h, mode):
            raise ValueError("oracle_grid_set_alphas_mode failed")

    def set_coupling(self, Cmat):
        c, cp = _d(Cmat)
        if c.size != self.nflav ** 2 or lib().oracle_grid_set_coupling(self._h, cp):
            raise ValueError("oracle_grid_set_coupling failed")

    def limits(self):
        a = [C.c_double() for _ in range(4)]
        lib().oracle_grid_limits(self._h, *[C.byref(t) for t in a])
        return tuple(t.value for t in a)

    def set_extrapolation(self, mode: int):
        """EXTRAP_CONTINUATION (default), EXTRAP_FREEZE, EXTRAP_ERROR"""
        if lib().oracle_grid_set_extrapolation(self._h, mode):
            raise ValueError("oracle_grid_set_extrapolation failed")

    def xfxq(self, pids, x, q, member=None, want_scale: bool = False):
        """xfxQ (the interface takes Q or Q2): by definition xfxQ2 at Q2 = Q * Q; Q <= 0 is invalid"""
        q = np.asarray(q, dtype=np.float64)
        with np.errstate(over="ignore", invalid="ignore"):
            q2 = np.where(q > 0, q * q, np.nan)
        return self.xfxq2(pids, x, q2, member=member, want_scale=want_scale)

    def locate(self, x, q2):
        x, xp = _d(x)
        q, qp = _d(q2)
        n = x.size
        outs = [np.empty(n, dtype=np.int32) for _ in range(4)]
        rc = lib().oracle_locate(self._h, n, xp, qp, *[o.ctypes.data_as(C.POINTER(C.c_int)) for o in outs])
        if rc:
            raise ValueError(f"oracle_locate: {rc}")
        return tuple(outs)  # ix, iq, isub, region

    def xfxq2(self, pids, x, q2, member=None, want_scale: bool = False):
        x, xp = _d(x)
        q, qp = _d(q2)
        pid, pp = _i(pids)
        n = x.size
        out = np.empty((n, len(pid)))
        sc = np.empty((n, len(pid), 2)) if want_scale else None
        mp = None
        if member is not None:
            member, mp = _i(member)
        rc = lib().oracle_xfxq2(self._h, pp, len(pid), n, xp, qp, mp,
                                out.ctypes.data_as(C.POINTER(C.c_double)),
                                sc.ctypes.data_as(C.POINTER(C.c_double)) if want_scale else None)
        if rc:
            raise ValueError(f"oracle_xfxq2: {rc}")
        return (out, sc) if want_scale else out

    def alphas_q2(self, q2):
        q, qp = _d(q2)
        out = np.empty(q.size)
        rc = lib().oracle_alphas_q2(self._h, q.size, qp, out.ctypes.data_as(C.POINTER(C.c_double)))
        if rc:
            raise ValueError(f"oracle_alphas_q2: {rc}")
        return out

    def lumi(self, x1, x2, q2, weights, want_scale: bool = False):
        a, ap = _d(x1)
        b, bp = _d(x2)
        q, qp = _d(q2)
        w, wp = _d(weights)
        out = np.empty(a.size)
        sc = np.empty((a.size, 2)) if want_scale else None
        rc = lib().oracle_lumi(self._h, a.size, ap, bp, qp, wp,
                               out.ctypes.data_as(C.POINTER(C.c_double)),
                               sc.ctypes.data_as(C.POINTER(C.c_double)) if want_scale else None)
        if rc:
            raise ValueError(f"oracle_lumi: {rc}")
        return (out, sc) if want_scale else out

    def interior_order(self, order: int, flavour_col: int, x, q2, member: int = 0):
        x, xp = _d(x)
        q, qp = _d(q2)
        out = np.empty(x.size)
        rc = lib().oracle_interior_order(self._h, order, flavour_col, member, x.size, xp, qp,
                                         out.ctypes.data_as(C.POINTER(C.c_double)))
        if rc:
            raise ValueError(f"oracle_interior_order: {rc}")
        return out


# ---- Monte Carlo steps around the hot path (mc_oracle.c) -------------
def rambo_w0(n: int, s: float) -> float:
    return float(lib().oracle_rambo_w0(int(n), float(s)))


def rambo(sqrt_s, u, masses=None, ptmin: float = 0.0):
    """u[nev][n][4] uniforms -> (p[nev][n][4] = (E, px, py, pz), w[nev])"""
    u, up = _d(u)
    nev, n = u.shape[0], u.shape[1]
    rs, rp = _d(np.broadcast_to(np.asarray(sqrt_s, dtype=np.float64), (nev,)))
    mp = None
    if masses is not None:
        masses, mp = _d(masses)
    p, w = np.empty((nev, n, 4)), np.empty(nev)
    rc = lib().oracle_rambo(nev, n, rp, mp, up, float(ptmin), p.ctypes.data_as(C.POINTER(C.c_double)),
                            w.ctypes.data_as(C.POINTER(C.c_double)))
    if rc:
        raise ValueError(f"oracle_rambo: {rc}")
    return p, w


def vegas_map(edges, u):
    e, ep = _d(edges)
    u, up = _d(u)
    n, ndim = u.shape
    nb = e.shape[1] - 1
    x, jac, bins = np.empty((n, ndim)), np.empty(n), np.empty((n, ndim), dtype=np.int32)
    rc = lib().oracle_vegas_map(ndim, nb, ep, n, up, x.ctypes.data_as(C.POINTER(C.c_double)),
                                jac.ctypes.data_as(C.POINTER(C.c_double)), bins.ctypes.data_as(C.POINTER(C.c_int)))
    if rc:
        raise ValueError(f"oracle_vegas_map: {rc}")
    return x, jac, bins


def vegas_accumulate(nb: int, f, jac, bins):
    f, fp = _d(f)
    j, jp = _d(jac)
    b, bp = _i(bins)
    ndim = b.shape[1]
    sums, hist = np.empty(2), np.empty((ndim, nb))
    rc = lib().oracle_vegas_accumulate(ndim, nb, f.size, fp, jp, bp, sums.ctypes.data_as(C.POINTER(C.c_double)),
                                       hist.ctypes.data_as(C.POINTER(C.c_double)))
    if rc:
        raise ValueError(f"oracle_vegas_accumulate: {rc}")
    return sums, hist


def vegas_estimate(n: int, sums):
    s, sp = _d(sums)
    E, var = C.c_double(), C.c_double()
    if lib().oracle_vegas_estimate(int(n), sp, C.byref(E), C.byref(var)):
        raise ValueError("oracle_vegas_estimate")
    return E.value, var.value


def vegas_refine(hist, edges, alpha: float = 1.0):
    h, hp = _d(hist)
    e = np.array(edges, dtype=np.float64, order="C")
    ndim, nb = h.shape
    if lib().oracle_vegas_refine(ndim, nb, hp, float(alpha), e.ctypes.data_as(C.POINTER(C.c_double))):
        raise ValueError("oracle_vegas_refine")
    return e


def vegas_combine(E, S2):
    E, Ep = _d(E)
    S, Sp = _d(S2)
    a, b, c = C.c_double(), C.c_double(), C.c_double()
    if lib().oracle_vegas_combine(E.size, Ep, Sp, C.byref(a), C.byref(b), C.byref(c)):
        raise ValueError("oracle_vegas_combine")
    return a.value, b.value, c.value


def unweight(w, u):
    w, wp = _d(w)
    u, up = _d(u)
    acc = np.empty(w.size, dtype=np.uint8)
    wmax, cnt = C.c_double(), C.c_longlong()
    if lib().oracle_unweight(w.size, wp, up, C.byref(wmax), acc.ctypes.data_as(C.POINTER(C.c_ubyte)), C.byref(cnt)):
        raise ValueError("oracle_unweight")
    return wmax.value, acc.astype(bool), int(cnt.value)
