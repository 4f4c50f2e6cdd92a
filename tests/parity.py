"""Parity metric GPU <-> oracle (C-12).

pass  <=>  |gpu - ref| <= REL |ref| + FLOOR_S S[...,0] + FLOOR_T S[...,1]   for every output element
(``oracle.tolerance``; REL = 1e-12 is north_star's tolerance).  The two floor terms are the eq.-3.6 epsilon
 made condition-aware; the oracle returns both condition numbers, pinned by
tests/test_oracle_pins.py::test_scale_*:
  * S[...,0] = sum |Wx_a Wq_b V_ab|: a few ulp of it are lost to the rounding of the 16-term stencil sum by ANY
    evaluation order (the oracle's included; its own three orders differ at that level, P-10);
  * S[...,1] = |df/dt| (1 + |ln v|/delta): t = (ln v - ln knot)/delta is only known to a few 2^-52 of that
    factor (glibc's and CUDA's log may differ in the last bit); same for the extrapolation abscissa theta.
Where the result cancels (|ref| << S: sign changes in Q2, x -> 1 where every flavour vanishes like 1 - t,
flavours switched off below threshold) no evaluation can hold a strict relative bound.  The strict relative
maximum over |ref| > STRICT_CUT * S[...,0] is reported and asserted by the C0/C1/C2 tests.
NaN rows must match as NaN.
"""
import numpy as np

import oracle

REL = oracle.REL
STRICT_CUT = 1e-3          # SURVEY C-12: "report also the strict maximum over points with |ref| > 1e-3 S"


def value_errors(gpu, ref, S):
    gpu, ref, S = np.asarray(gpu), np.asarray(ref), np.asarray(S)
    nan_ref, nan_gpu = np.isnan(ref), np.isnan(gpu)
    assert np.array_equal(nan_ref, nan_gpu), "NaN pattern differs"
    ok = ~nan_ref
    err = np.abs(gpu[ok] - ref[ok])
    tol = oracle.tolerance(ref[ok], S[ok])
    exact = err == 0
    ratio = np.where(exact, 0.0, err / np.where(tol > 0, tol, 1e-300))
    strict_sel = np.abs(ref[ok]) > STRICT_CUT * S[ok][..., 0]
    strict = float(np.max(err[strict_sel] / np.abs(ref[ok][strict_sel]))) if strict_sel.any() else 0.0
    # the same errors against tighter floors (what the floors could be lowered to): worst ratio per candidate
    probe = {}
    for fs in (1e-15, 5e-16):
        for ft in (2 * 2.0 ** -52, 2.0 ** -52):
            t2 = REL * np.abs(ref[ok]) + fs * S[ok][..., 0] + ft * S[ok][..., 1]
            probe[f"S{fs:g}_T{ft / 2.0 ** -52:g}ulp"] = float(np.max(np.where(exact, 0.0, err / np.where(t2 > 0, t2, 1e-300)))) if err.size else 0.0
    return dict(worst=float(ratio.max()) if ratio.size else 0.0, strict_rel_max=strict,
                frac_within_strict=float(np.mean(err <= REL * np.abs(ref[ok]))) if err.size else 1.0, probe=probe)


def assert_values(gpu, ref, S, what="", strict=None):
    """strict: if given, also assert the strict relative maximum (|ref| > STRICT_CUT S) <= strict"""
    st = value_errors(gpu, ref, S)
    assert st["worst"] <= 1.0, (what, st)
    if strict is not None:
        assert st["strict_rel_max"] <= strict, (what, st)
    return st
