"""Parity metric GPU <-> oracle (C-12).

pass  <=>  |gpu - ref| <= REL * |ref| + FLOOR * scale   for every output element.
REL = 1e-12 is north_star's tolerance.  The FLOOR term is the eq.-3.6 epsilon
made condition-aware; `scale` is returned by the oracle and is a first-order bound, in units of
1e-14, of what rounding alone does to ANY evaluation of the definition (the oracle's included):
  * the 16-term stencil sum:  sum |Wx_a Wq_b V_ab|   (a few ulp of it are lost to rounding);
  * t = (ln x - u_i)/du is only known to 2^-52 (2 + 2 |ln x|/du) (one ulp each of ln x and u_i,
    divided by du ~ 0.1, and glibc's and CUDA's log may differ in the last bit), which moves the
    value by |df/dt| times that; same for t_q and for the extrapolation abscissa theta.
Where the result cancels (|ref| << scale: sign changes in Q2, x -> 1 where every flavour
vanishes like 1 - t, flavours switched off below threshold) no evaluation order can hold a
strict relative bound -- the oracle itself is uncertain there at that level.
NaN rows must match as NaN.
"""
import numpy as np

REL = 1e-12
FLOOR = 1e-14


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
