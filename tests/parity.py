"""Parity metric GPU <-> oracle (C-12).

pass  <=>  |gpu - ref| <= REL * |ref| + FLOOR * S   for every output element,
with S the oracle's condition scale (sum of |weight * node value| propagated through the
extrapolation).  REL = 1e-12 is north_star's tolerance; the FLOOR term is the eq.-3.6 epsilon
made condition-aware: t = (ln x - u_i)/du carries an absolute rounding error of up to
2 ulp(ln x)/du ~ 3e-14 (|ln x| <= 32, du ~ 0.1) that differs between glibc's and CUDA's log, and
the 16-term sum rounds at ~1e-15 S; where the result cancels (|ref| << S: sign changes in Q2,
x -> 1, flavours switched off) no reordering of the sum can hold a strict relative bound.
NaN rows must match as NaN.
"""
import numpy as np

REL = 1e-12
FLOOR = 1e-13


def value_errors(gpu, ref, S):
    gpu, ref, S = np.asarray(gpu), np.asarray(ref), np.asarray(S)
    nan_ref, nan_gpu = np.isnan(ref), np.isnan(gpu)
    assert np.array_equal(nan_ref, nan_gpu), "NaN pattern differs"
    ok = ~nan_ref
    err = np.abs(gpu[ok] - ref[ok])
    tol = REL * np.abs(ref[ok]) + FLOOR * S[ok]
    exact = err == 0
    ratio = np.where(exact, 0.0, err / np.where(tol > 0, tol, 1e-300))
    strict_sel = np.abs(ref[ok]) > 1e-2 * S[ok]
    strict = float(np.max(err[strict_sel] / np.abs(ref[ok][strict_sel]))) if strict_sel.any() else 0.0
    return dict(worst=float(ratio.max()) if ratio.size else 0.0, strict_rel_max=strict,
                frac_within_strict=float(np.mean(err <= REL * np.abs(ref[ok]))) if err.size else 1.0)


def assert_values(gpu, ref, S, what=""):
    st = value_errors(gpu, ref, S)
    assert st["worst"] <= 1.0, (what, st)
    return st
