"""Thin ctypes binding of ``libpdfgrid.so`` (C ABI: ``include/pdfgrid.h``).

Argument marshalling only: every step of the path runs in the CUDA kernels.  The
function names mirror the C calls (``pdf_grid_create`` ... ``pdf_lumi``).  PyTorch is
used for device memory and streams (``tensor.data_ptr()``, the current CUDA stream).

There is NO CPU fallback: if the shared library is missing or cannot be loaded,
importing a symbol raises ``PdfGridError``.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import torch


_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpdfgrid.so")

PDF_OK, PDF_EINVAL, PDF_ENOMEM, PDF_ECUDA, PDF_EWORKSPACE, PDF_ESTATE, PDF_ELIMIT = 0, -1, -2, -3, -4, -5, -6
PDF_PATH_AUTO, PDF_PATH_DIRECT, PDF_PATH_BINNED = 0, 1, 2
PDF_OPT_PATH, PDF_OPT_ALPHAS_MODE, PDF_OPT_CHUNK, PDF_OPT_EXTRAPOLATION = 1, 2, 3, 4
PDF_EXTRAP_CONTINUATION, PDF_EXTRAP_FREEZE, PDF_EXTRAP_ERROR = 0, 1, 2
PDF_ALPHAS_FREEZE, PDF_ALPHAS_LOGGRAD = 0, 1

# every symbol include/pdfgrid.h declares (tests check the library exports all of them)
SYMBOLS = (
    "pdf_grid_create", "pdf_grid_destroy", "pdf_grid_set_alphas", "pdf_grid_set_coupling",
    "pdf_grid_set_workspace", "pdf_workspace_bytes", "pdf_grid_set_option", "pdf_grid_limits",
    "pdf_xfxq2", "pdf_xfxq2_ex", "pdf_xfxq2_xgrid", "pdf_alphas_q2", "pdf_lumi", "pdf_locate", "pdf_error_count",
    "pdf_xfxq2_host", "pdf_alphas_q2_host", "pdf_lumi_host", "pdf_status_string",
    "pdf_last_cuda_error", "pdf_launch_count", "pdf_profile_enable", "pdf_profile_read",
    "pdf_measure_fp64_tflops", "pdf_last_path", "pdf_log_f64",
    "pdf_rambo", "pdf_vegas_map", "pdf_vegas_accumulate", "pdf_vegas_estimate", "pdf_vegas_refine", "pdf_vegas_combine",
    "pdf_unweight", "pdf_xfxq2_noalloc", "pdf_xfxq",
)


class PdfGridError(RuntimeError):
    pass


_lib = None


def lib():
    """Load libpdfgrid.so (never builds at import time on the GPU box; fails loudly if absent)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise PdfGridError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                           "(nvcc, sm_100a). There is no CPU fallback.")
    L = C.CDLL(LIB_PATH)
    vp, ip, dp, ll = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double), C.c_longlong
    L.pdf_grid_create.argtypes = [C.POINTER(vp), C.c_int, dp, C.c_int, ip, dp, dp, C.c_int, ip, C.c_int]
    L.pdf_grid_destroy.argtypes = [vp]
    L.pdf_grid_set_alphas.argtypes = [vp, C.c_int, dp, dp]
    L.pdf_grid_set_coupling.argtypes = [vp, dp]
    L.pdf_grid_set_workspace.argtypes = [vp, vp, C.c_size_t]
    L.pdf_workspace_bytes.argtypes = [vp, ll]
    L.pdf_workspace_bytes.restype = C.c_size_t
    L.pdf_grid_set_option.argtypes = [vp, C.c_int, ll]
    L.pdf_grid_limits.argtypes = [vp, dp, dp, dp, dp]
    L.pdf_xfxq2.argtypes = [vp, ip, C.c_int, ll, vp, vp, vp, vp]
    L.pdf_xfxq.argtypes = [vp, ip, C.c_int, ll, vp, vp, vp, vp]
    L.pdf_xfxq2_noalloc.argtypes = [vp, ip, C.c_int, ll, vp, vp, vp, C.POINTER(ll), vp]
    L.pdf_xfxq2_ex.argtypes = [vp, ip, C.c_int, ll, vp, vp, vp, vp, ll, vp]
    L.pdf_xfxq2_xgrid.argtypes = [vp, ip, C.c_int, ll, vp, vp, C.c_int, vp, vp, ll, vp]
    L.pdf_alphas_q2.argtypes = [vp, ll, vp, vp, vp]
    L.pdf_lumi.argtypes = [vp, ll, vp, vp, vp, vp, vp, vp]
    L.pdf_locate.argtypes = [vp, ll, vp, vp, vp, vp, vp, vp, vp]
    L.pdf_error_count.argtypes = [vp, C.POINTER(ll), vp]
    L.pdf_xfxq2_host.argtypes = [vp, ip, C.c_int, ll, vp, vp, vp]
    L.pdf_alphas_q2_host.argtypes = [vp, ll, vp, vp]
    L.pdf_lumi_host.argtypes = [vp, ll, vp, vp, vp, vp, vp]
    L.pdf_status_string.argtypes = [C.c_int]
    L.pdf_status_string.restype = C.c_char_p
    L.pdf_last_cuda_error.restype = C.c_char_p
    L.pdf_launch_count.restype = ll
    L.pdf_profile_enable.argtypes = [C.c_int]
    L.pdf_profile_read.argtypes = [C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_float)]
    L.pdf_measure_fp64_tflops.argtypes = [dp, vp]
    L.pdf_last_path.argtypes = [vp]
    L.pdf_log_f64.argtypes = [ll, vp, vp, vp]
    L.pdf_rambo.argtypes = [ll, C.c_int, vp, dp, vp, C.c_double, vp, vp, vp]
    L.pdf_vegas_map.argtypes = [C.c_int, C.c_int, vp, ll, vp, vp, vp, vp, vp]
    L.pdf_vegas_accumulate.argtypes = [C.c_int, C.c_int, ll, vp, vp, vp, vp, vp, vp]
    L.pdf_vegas_estimate.argtypes = [ll, vp, vp, vp]
    L.pdf_vegas_refine.argtypes = [C.c_int, C.c_int, vp, C.c_double, vp, vp, vp]
    L.pdf_vegas_combine.argtypes = [C.c_int, vp, vp, vp, vp]
    L.pdf_unweight.argtypes = [ll, vp, vp, vp, vp, dp, C.POINTER(ll), vp]
    _lib = L
    return L


def _check(rc: int, what: str):
    if rc != PDF_OK:
        L = lib()
        msg = L.pdf_status_string(rc).decode()
        if rc == PDF_ECUDA or rc == PDF_ENOMEM:
            msg += " [" + L.pdf_last_cuda_error().decode() + "]"
        raise PdfGridError(f"{what}: {msg} ({rc})")


def _hd(t) -> torch.Tensor:
    return torch.as_tensor(t, dtype=torch.float64, device="cpu").contiguous()


def _hi(t) -> torch.Tensor:
    return torch.as_tensor(t, dtype=torch.int32, device="cpu").contiguous()


def _dptr(t: torch.Tensor):
    return C.cast(t.data_ptr(), C.POINTER(C.c_double))


def _iptr(t: torch.Tensor):
    return C.cast(t.data_ptr(), C.POINTER(C.c_int))


def _stream_ptr(stream: Optional[torch.cuda.Stream]):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _dev(t: torch.Tensor, dtype, what: str, numel: Optional[int] = None, at_least: bool = False):
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise PdfGridError(f"{what} must be a contiguous CUDA tensor of dtype {dtype}")
    if numel is not None and (t.numel() < numel if at_least else t.numel() != numel):
        raise PdfGridError(f"{what} has {t.numel()} elements, expected {'>= ' if at_least else ''}{numel}")
    return C.c_void_p(t.data_ptr())


def _host(t: torch.Tensor, what: str, numel: int, at_least: bool = False):
    if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous():
        raise PdfGridError(f"{what} must be a contiguous CPU float64 tensor")
    if t.numel() < numel if at_least else t.numel() != numel:
        raise PdfGridError(f"{what} has {t.numel()} elements, expected {'>= ' if at_least else ''}{numel}")
    return C.c_void_p(t.data_ptr())


def pdf_launch_count() -> int:
    return int(lib().pdf_launch_count())


def pdf_profile_enable(on: bool):
    lib().pdf_profile_enable(1 if on else 0)


def pdf_profile_read(max_entries: int = 4096):
    names = (C.c_char_p * max_entries)()
    ms = (C.c_float * max_entries)()
    n = lib().pdf_profile_read(max_entries, names, ms)
    return [(names[i].decode(), float(ms[i])) for i in range(n)]


def pdf_measure_fp64_tflops(stream=None) -> float:
    v = C.c_double()
    _check(lib().pdf_measure_fp64_tflops(C.byref(v), _stream_ptr(stream)), "pdf_measure_fp64_tflops")
    return v.value


def pdf_log_f64(x: torch.Tensor, stream=None) -> torch.Tensor:
    out = torch.empty_like(x)
    _check(lib().pdf_log_f64(x.numel(), _dev(x, torch.float64, "x"), _dev(out, torch.float64, "out"), _stream_ptr(stream)), "pdf_log_f64")
    return out


# ---- Monte Carlo steps around the hot path (argument marshalling only) -------------------------------------
def pdf_rambo(sqrt_s: torch.Tensor, u: torch.Tensor, masses=None, ptmin: float = 0.0, stream=None):
    """u [nev][npart][4] uniforms -> (p [nev][npart][4], w [nev])"""
    nev, npart = u.shape[0], u.shape[1]
    f = torch.float64
    p = torch.empty((nev, npart, 4), dtype=f, device=u.device)
    w = torch.empty(nev, dtype=f, device=u.device)
    m = _hd(masses) if masses is not None else None
    if m is not None and m.numel() != npart:
        raise PdfGridError("masses must have npart entries")
    _check(lib().pdf_rambo(nev, npart, _dev(sqrt_s, f, "sqrt_s", nev), _dptr(m) if m is not None else None,
                           _dev(u, f, "u", nev * npart * 4), float(ptmin), _dev(p, f, "p"), _dev(w, f, "w"), _stream_ptr(stream)),
           "pdf_rambo")
    return p, w


def pdf_vegas_map(edges: torch.Tensor, u: torch.Tensor, stream=None):
    ndim, nb = edges.shape[0], edges.shape[1] - 1
    n = u.shape[0]
    f = torch.float64
    x = torch.empty((n, ndim), dtype=f, device=u.device)
    jac = torch.empty(n, dtype=f, device=u.device)
    bins = torch.empty((n, ndim), dtype=torch.int32, device=u.device)
    _check(lib().pdf_vegas_map(ndim, nb, _dev(edges, f, "edges"), n, _dev(u, f, "u", n * ndim), _dev(x, f, "x"), _dev(jac, f, "jac"),
                               _dev(bins, torch.int32, "bin"), _stream_ptr(stream)), "pdf_vegas_map")
    return x, jac, bins


def pdf_vegas_accumulate(nb: int, fvals: torch.Tensor, jac: torch.Tensor, bins: torch.Tensor, stream=None):
    n, ndim = bins.shape
    f = torch.float64
    sums = torch.empty(2, dtype=f, device=jac.device)
    hist = torch.empty((ndim, nb), dtype=f, device=jac.device)
    _check(lib().pdf_vegas_accumulate(ndim, nb, n, _dev(fvals, f, "f", n), _dev(jac, f, "jac", n), _dev(bins, torch.int32, "bin"),
                                      _dev(sums, f, "sums"), _dev(hist, f, "hist"), _stream_ptr(stream)), "pdf_vegas_accumulate")
    return sums, hist


def pdf_vegas_estimate(n: int, sums: torch.Tensor, stream=None):
    res = torch.empty(2, dtype=torch.float64, device=sums.device)
    _check(lib().pdf_vegas_estimate(n, _dev(sums, torch.float64, "sums", 2), _dev(res, torch.float64, "res"), _stream_ptr(stream)),
           "pdf_vegas_estimate")
    return res


def pdf_vegas_refine(hist: torch.Tensor, edges: torch.Tensor, alpha: float = 1.0, stream=None):
    """refines `edges` in place"""
    ndim, nb = hist.shape
    scratch = torch.empty((ndim, 2 * nb + 1), dtype=torch.float64, device=hist.device)
    _check(lib().pdf_vegas_refine(ndim, nb, _dev(hist, torch.float64, "hist"), float(alpha), _dev(edges, torch.float64, "edges", ndim * (nb + 1)),
                                  _dev(scratch, torch.float64, "scratch"), _stream_ptr(stream)), "pdf_vegas_refine")
    return edges


def pdf_vegas_combine(E: torch.Tensor, S2: torch.Tensor, stream=None):
    res = torch.empty(3, dtype=torch.float64, device=E.device)
    _check(lib().pdf_vegas_combine(E.numel(), _dev(E, torch.float64, "E"), _dev(S2, torch.float64, "S2", E.numel()),
                                   _dev(res, torch.float64, "res"), _stream_ptr(stream)), "pdf_vegas_combine")
    return res


def pdf_unweight(w: torch.Tensor, u: torch.Tensor, stream=None):
    n = w.numel()
    acc = torch.empty(n, dtype=torch.uint8, device=w.device)
    scratch = torch.empty(16, dtype=torch.uint8, device=w.device)
    wmax, cnt = C.c_double(), C.c_longlong()
    _check(lib().pdf_unweight(n, _dev(w, torch.float64, "w"), _dev(u, torch.float64, "u", n), _dev(acc, torch.uint8, "accept"),
                              _dev(scratch, torch.uint8, "scratch"), C.byref(wmax), C.byref(cnt), _stream_ptr(stream)), "pdf_unweight")
    return wmax.value, acc.bool(), int(cnt.value)


class PdfGrid:
    """Owner of a ``pdf_grid*`` handle.  Methods are 1:1 with the C calls."""

    def __init__(self, x_knots, q2_subgrids: Sequence, values, pids: Sequence[int], nmem: int = 1):
        L = lib()
        x = _hd(x_knots)
        nq = _hi([len(q) for q in q2_subgrids])
        q2 = _hd(torch.cat([_hd(q) for q in q2_subgrids]))
        v = _hd(values).reshape(-1)
        pid = _hi(list(pids))
        expect = x.numel() * int(nq.sum()) * pid.numel() * nmem
        if v.numel() != expect:
            raise PdfGridError(f"values has {v.numel()} entries, expected {expect}")
        self._h = C.c_void_p()
        _check(L.pdf_grid_create(C.byref(self._h), x.numel(), _dptr(x), nq.numel(), _iptr(nq), _dptr(q2),
                                 _dptr(v), pid.numel(), _iptr(pid), nmem), "pdf_grid_create")
        self.nflav, self.nmem, self.pids = pid.numel(), nmem, tuple(int(p) for p in pids)
        self._ws = None

    @classmethod
    def from_spec(cls, spec, workspace_for: int = 0):
        g = cls(spec.x_knots, spec.q2_subgrids, spec.values, spec.pids, nmem=spec.nmem)
        if spec.alphas_q2 is not None:
            g.pdf_grid_set_alphas(spec.alphas_q2, spec.alphas_val)
        if spec.coupling is not None:
            g.pdf_grid_set_coupling(spec.coupling)
        if workspace_for:
            g.attach_workspace(workspace_for)
        return g

    def close(self):
        if getattr(self, "_h", None):
            lib().pdf_grid_destroy(self._h)
            self._h = C.c_void_p()
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- configuration -------------------------------------------------------------------
    def pdf_grid_set_alphas(self, q2_knots, values):
        q, v = _hd(q2_knots), _hd(values)
        _check(lib().pdf_grid_set_alphas(self._h, q.numel(), _dptr(q), _dptr(v)), "pdf_grid_set_alphas")

    def pdf_grid_set_coupling(self, Cmat):
        c = _hd(Cmat).reshape(-1)
        if c.numel() != self.nflav ** 2:
            raise PdfGridError("coupling must be [nflav][nflav]")
        _check(lib().pdf_grid_set_coupling(self._h, _dptr(c)), "pdf_grid_set_coupling")

    def pdf_grid_set_option(self, option: int, value: int):
        _check(lib().pdf_grid_set_option(self._h, option, value), "pdf_grid_set_option")

    def pdf_workspace_bytes(self, n: int) -> int:
        return int(lib().pdf_workspace_bytes(self._h, n))

    def pdf_grid_set_workspace(self, ws: Optional[torch.Tensor]):
        if ws is None:
            _check(lib().pdf_grid_set_workspace(self._h, None, 0), "pdf_grid_set_workspace")
        else:
            _check(lib().pdf_grid_set_workspace(self._h, C.c_void_p(ws.data_ptr()), ws.numel() * ws.element_size()),
                   "pdf_grid_set_workspace")
        self._ws = ws

    def attach_workspace(self, n: int, device="cuda"):
        """Allocate (torch) and attach the scratch the binned path needs for calls of up to n queries."""
        nbytes = self.pdf_workspace_bytes(n)
        if nbytes:
            self.pdf_grid_set_workspace(torch.empty(nbytes, dtype=torch.uint8, device=device))
        return nbytes

    def pdf_grid_limits(self):
        a = [C.c_double() for _ in range(4)]
        _check(lib().pdf_grid_limits(self._h, *[C.byref(t) for t in a]), "pdf_grid_limits")
        return tuple(t.value for t in a)

    # ---- evaluation (device tensors) -----------------------------------------------------
    def pdf_xfxq2(self, pids, x: torch.Tensor, q2: torch.Tensor, out: Optional[torch.Tensor] = None,
                  member: Optional[torch.Tensor] = None, ld_out: Optional[int] = None, stream=None):
        pid = _hi(list(pids))
        n = x.numel()
        ld = ld_out or pid.numel()
        if out is None:
            out = torch.empty((n, ld), dtype=torch.float64, device=x.device)
        xp, qp, op = _dev(x, torch.float64, "x"), _dev(q2, torch.float64, "q2"), _dev(out, torch.float64, "out")
        if q2.numel() != n or out.numel() < n * ld:
            raise PdfGridError("size mismatch")
        if member is None and ld == pid.numel():
            rc = lib().pdf_xfxq2(self._h, _iptr(pid), pid.numel(), n, xp, qp, op, _stream_ptr(stream))
        else:
            mp = _dev(member, torch.int32, "member") if member is not None else None
            rc = lib().pdf_xfxq2_ex(self._h, _iptr(pid), pid.numel(), n, xp, qp, mp, op, ld, _stream_ptr(stream))
        _check(rc, "pdf_xfxq2")
        return out

    def pdf_xfxq(self, pids, x: torch.Tensor, q: torch.Tensor, out: Optional[torch.Tensor] = None, stream=None):
        """xfxQ: `q` holds Q (GeV), not Q2"""
        pid = _hi(list(pids))
        n = x.numel()
        if out is None:
            out = torch.empty((n, pid.numel()), dtype=torch.float64, device=x.device)
        xp, qp = _dev(x, torch.float64, "x", n), _dev(q, torch.float64, "q", n)
        op = _dev(out, torch.float64, "out", n * pid.numel(), at_least=True)
        _check(lib().pdf_xfxq(self._h, _iptr(pid), pid.numel(), n, xp, qp, op, _stream_ptr(stream)), "pdf_xfxq")
        return out

    def pdf_xfxq2_noalloc(self, pids, x: torch.Tensor, q2: torch.Tensor, out: torch.Tensor, stream=None) -> int:
        """pdf_xfxq2 through the library's static scratch array: no workspace, no allocation in the call (the caller
        passes `out`).  Returns the largest n the grid allows; raises PdfGridError (PDF_ELIMIT) beyond it."""
        pid = _hi(list(pids))
        n = x.numel()
        xp, qp = _dev(x, torch.float64, "x", n), _dev(q2, torch.float64, "q2", n)
        op = _dev(out, torch.float64, "out", n * pid.numel(), at_least=True)
        max_n = C.c_longlong(0)
        rc = lib().pdf_xfxq2_noalloc(self._h, _iptr(pid), pid.numel(), n, xp, qp, op, C.byref(max_n), _stream_ptr(stream))
        if rc == PDF_ELIMIT:
            raise PdfGridError(f"pdf_xfxq2_noalloc: n = {n} is beyond the {max_n.value} queries that the static scratch "
                               f"array holds for this grid ({lib().pdf_status_string(rc).decode()}) ({rc})")
        _check(rc, "pdf_xfxq2_noalloc")
        return int(max_n.value)

    def pdf_xfxq2_xgrid(self, pids, x: torch.Tensor, q2: torch.Tensor, nrep: int,
                        members: Optional[torch.Tensor] = None, out: Optional[torch.Tensor] = None,
                        ld_out: Optional[int] = None, stream=None):
        """out[r, p, k] = xf_{pids[k]}(member members[r] (default r); x[p], q2[p]): every member on one shared point list"""
        pid = _hi(list(pids))
        npts = x.numel()
        ld = ld_out or pid.numel()
        if out is None:
            out = torch.empty((nrep, npts, ld), dtype=torch.float64, device=x.device)
        xp, qp, op = _dev(x, torch.float64, "x"), _dev(q2, torch.float64, "q2"), _dev(out, torch.float64, "out")
        if q2.numel() != npts or out.numel() < nrep * npts * ld or (members is not None and members.numel() != nrep):
            raise PdfGridError("size mismatch")
        mp = _dev(members, torch.int32, "members") if members is not None else None
        _check(lib().pdf_xfxq2_xgrid(self._h, _iptr(pid), pid.numel(), npts, xp, qp, nrep, mp, op, ld, _stream_ptr(stream)),
               "pdf_xfxq2_xgrid")
        return out

    def pdf_alphas_q2(self, q2: torch.Tensor, out: Optional[torch.Tensor] = None, stream=None):
        if out is None:
            out = torch.empty_like(q2)
        n = q2.numel()
        _check(lib().pdf_alphas_q2(self._h, n, _dev(q2, torch.float64, "q2"),
                                   _dev(out, torch.float64, "out", n, at_least=True), _stream_ptr(stream)), "pdf_alphas_q2")
        return out

    def pdf_lumi(self, x1, x2, q2, weights, out: Optional[torch.Tensor] = None, stream=None):
        if out is None:
            out = torch.empty_like(x1)
        f, n = torch.float64, x1.numel()
        _check(lib().pdf_lumi(self._h, n, _dev(x1, f, "x1"), _dev(x2, f, "x2", n), _dev(q2, f, "q2", n),
                              _dev(weights, f, "weights", n), _dev(out, f, "out", n, at_least=True), _stream_ptr(stream)), "pdf_lumi")
        return out

    def pdf_locate(self, x: torch.Tensor, q2: torch.Tensor, stream=None):
        n = x.numel()
        outs = [torch.empty(n, dtype=torch.int32, device=x.device) for _ in range(4)]
        _check(lib().pdf_locate(self._h, n, _dev(x, torch.float64, "x"), _dev(q2, torch.float64, "q2", n),
                                *[C.c_void_p(o.data_ptr()) for o in outs], _stream_ptr(stream)), "pdf_locate")
        return tuple(outs)  # ix, iq, isub, region

    def pdf_last_path(self) -> int:
        """PDF_PATH_DIRECT or PDF_PATH_BINNED: which kernels the last evaluation call on this handle ran"""
        return int(lib().pdf_last_path(self._h))

    def pdf_error_count(self, stream=None) -> int:
        v = C.c_longlong()
        _check(lib().pdf_error_count(self._h, C.byref(v), _stream_ptr(stream)), "pdf_error_count")
        return int(v.value)

    # ---- evaluation (host tensors; the e2e path) -------------------------------------------
    def pdf_xfxq2_host(self, pids, x: torch.Tensor, q2: torch.Tensor, out: torch.Tensor):
        pid = _hi(list(pids))
        n = x.numel()
        _check(lib().pdf_xfxq2_host(self._h, _iptr(pid), pid.numel(), n, _host(x, "x", n), _host(q2, "q2", n),
                                    _host(out, "out", n * pid.numel(), at_least=True)), "pdf_xfxq2_host")
        return out

    def pdf_alphas_q2_host(self, q2: torch.Tensor, out: torch.Tensor):
        n = q2.numel()
        _check(lib().pdf_alphas_q2_host(self._h, n, _host(q2, "q2", n), _host(out, "out", n, at_least=True)), "pdf_alphas_q2_host")
        return out

    def pdf_lumi_host(self, x1, x2, q2, weights, out):
        n = x1.numel()
        _check(lib().pdf_lumi_host(self._h, n, _host(x1, "x1", n), _host(x2, "x2", n), _host(q2, "q2", n),
                                   _host(weights, "weights", n), _host(out, "out", n, at_least=True)), "pdf_lumi_host")
        return out
