// pdf_common.cuh -- device-side data layout and the per-query arithmetic shared by all kernels.
//
// Method: PAPER.md section 3.2 (L1714-1746) in the readings of DESIGN.md (C-1 ... C-L).
// This file is part of the CUDA product path; it shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pdfg {

constexpr int kAlphaLutMax = 2048;  // search-table buckets of the alpha_s knot line (indexed by exponent and top mantissa bits)
constexpr int kMaxLumiFlav = 16;   // generic pdf_lumi keeps both flavour vectors in registers/local
constexpr int kExtrapContinuation = 0, kExtrapFreeze = 1, kExtrapError = 2;
constexpr int kRegionInterior = 0, kRegionLowX = 1, kRegionLowQ = 2, kRegionHighQ = 3,
              kRegionLowXLowQ = 4, kRegionLowXHighQ = 5, kRegionInvalid = 6;

// Per-cell constants of the 1-D Hermite operator in its 4-node-weight form (C-5):
//   W[-1] = -bL h10;  W[0] = h00 + (bL-aL) h10 - aR h11;  W[+1] = h01 + aL h10 + (aR-bR) h11;
//   W[+2] = bR h11,   with (aL,bL) = (1/2, rho_-/2) if the left neighbour exists else (1,0),
//   (aR,bR) likewise on the right (one-sided secant at a grid / sub-grid end, L1833).
struct CellTab {
    double lo_log;   // ln of the cell's lower knot
    double inv_d;    // 1 / (ln upper - ln lower)
    double aL, bL, aR, bR;
};

// Device view of one grid (a-1).  Values are re-laid as V[mem][jg][ix][nfp]: one node = one
// padded flavour row, the 4 x-neighbours of a Q2 row contiguous, jg = global Q2 knot index over
// the concatenated sub-grids (a threshold appears twice, once per sub-grid, L1714).
struct GridDev {
    int nx, nsub, nflav, nfp, nmem, nqtot;
    const double *xk, *qk;        // raw knots [nx], [nqtot]
    const double *uk, *sk;        // ln knots (device log: the same routine the queries go through)
    const int *sub_of;            // [nqtot] sub-grid of global knot jg
    const int *qoff;              // [nsub+1]
    const int *cell_adj;          // [nqtot] 1 on the last knot of a sub-grid (it belongs to the cell below), else 0
    const CellTab *cx;            // [nx-1]
    const CellTab *cq;            // [nqtot], entry jg valid when jg is not the last knot of its sub-grid
    const double *V;
    size_t memstride;             // nqtot*nx*nfp
    double q2plus;                // 1.01 * Q2min (C-9)
    // alpha_s (a-6)
    int extrap;                   // kExtrap*
    int na, alphas_mode;
    const double *ak, *alk, *av;  // raw knots, ln knots, values
    const CellTab *ca;            // [na-1]
    const double *acell;          // [na-1][6] per-cell cubic: ln lower knot, 1/dln, c0..c3 (alpha_s = c0 + t(c1 + t(c2 + t c3)))
    const unsigned short *alut;   // [nalut] cell at the lower edge of bucket (high word of Q2 >> ashift) - abase
    int ashift, abase, nalut;
    // luminosity coupling [nflav][nflav]
    const double *C;
    unsigned long long *err_count;
};

struct Point1D {      // a cell, its 4 clamped node indices and node weights
    int idx[4];
    double w[4];
};

// ln v for finite v > 0: the logarithm behind every abscissa of the path (t_x, t_q, theta: C-1, C-5, C-7, C-8) and
// behind the ln-knot tables, so that t == 0 exactly on a knot on every path.  The library routine is ~85
// instructions per call with its special cases (5 of the 42 warp instructions per query of the binned kernel,
// profile r2k); this one is 38 and inlines.  v = m 2^e, m in [sqrt(1/2), sqrt 2), f = m - 1 (exact),
// s = f / (2 + f), z = s^2:
//   ln m = 2 atanh(s) = f - f^2/2 + s (f^2/2 + R),   R = z (2/3 + z (2/5 + z (2/7 + ...))),   z <= 0.0295,
// summed in the order that keeps the exact f for last, with ln 2 split so that e ln2_hi is exact.
// Measured against glibc on the GPU box (tests/test_gpu_parity.py::test_path_logarithm): <= 1 ulp.
__device__ __forceinline__ double pdf_log(double v)
{
    int hi = __double2hiint(v), lo = __double2loint(v);
    int e = -1023;
    if (hi < 0x00100000) {                               // subnormal: scale by 2^54
        v *= 18014398509481984.0;
        hi = __double2hiint(v); lo = __double2loint(v);
        e -= 54;
    }
    e += hi >> 20;
    hi = (hi & 0x000fffff) | 0x3ff00000;                 // m in [1, 2)
    if (hi >= 0x3ff6a09f) { hi -= 0x00100000; ++e; }     // m in [sqrt(1/2), sqrt 2)
    const double f = __hiloint2double(hi, lo) - 1.0;
    const double d = 2.0 + f;
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    r = fma(fma(-d, r, 1.0), r, r);
    r = fma(fma(-d, r, 1.0), r, r);
    double s = f * r;
    s = fma(fma(-d, s, f), r, s);                        // s = f / d to the last bit or two
    const double z = s * s;
    double R = 2.0 / 21.0;
    R = fma(R, z, 2.0 / 19.0); R = fma(R, z, 2.0 / 17.0); R = fma(R, z, 2.0 / 15.0); R = fma(R, z, 2.0 / 13.0);
    R = fma(R, z, 2.0 / 11.0); R = fma(R, z, 2.0 / 9.0);  R = fma(R, z, 2.0 / 7.0);  R = fma(R, z, 2.0 / 5.0);
    R = fma(R, z, 2.0 / 3.0);
    R *= z;
    const double hfsq = 0.5 * f * f, de = (double)e;
    // ln 2 = ln2_hi + ln2_lo, the low 21 bits of ln2_hi are zero: e ln2_hi is exact for |e| < 2^11
    return fma(de, 0x1.62e42fee00000p-1, -((hfsq - fma(s, hfsq + R, de * 0x1.a39ef35793c76p-33)) - f));
}

__device__ __forceinline__ bool finite_pos(double v) { return v > 0.0 && v < __longlong_as_double(0x7ff0000000000000LL); }

// largest c in [0, m-2] with k[c] <= v (0 if none): C-4, comparisons on RAW values
__device__ __forceinline__ int find_cell(const double *__restrict__ k, int m, double v)
{
    int lo = 0, hi = m - 1;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (k[mid] <= v) lo = mid; else hi = mid;
    }
    return lo;
}

// largest jg in [0, m-1] with k[jg] <= v (0 if none); duplicates (thresholds) resolve to the
// later copy, i.e. the UPPER sub-grid (C-3, S-6)
__device__ __forceinline__ int find_last_le(const double *__restrict__ k, int m, double v)
{
    int lo = 0, hi = m;
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (k[mid] <= v) lo = mid; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ void hermite_weights(double t, const CellTab &c, double w[4])
{
    // Hermite basis cubics in factored form: relative accuracy kept where they vanish (t -> 0, 1)
    double omt = 1.0 - t, omt2 = omt * omt, t2 = t * t;
    double h00 = fma(2.0, t, 1.0) * omt2;
    double h10 = t * omt2;
    double h01 = t2 * fma(-2.0, t, 3.0);
    double h11 = -(t2 * omt);
    w[0] = -c.bL * h10;
    w[1] = h00 + (c.bL - c.aL) * h10 - c.aR * h11;
    w[2] = h01 + c.aL * h10 + (c.aR - c.bR) * h11;
    w[3] = c.bR * h11;
}

__device__ __forceinline__ int classify(const GridDev &G, double x, double q2)
{
    if (!(finite_pos(x) && finite_pos(q2)) || x > G.xk[G.nx - 1]) return kRegionInvalid;
    bool lowx = x < G.xk[0], lowq = q2 < G.qk[0], highq = q2 > G.qk[G.nqtot - 1];
    if (lowx) return lowq ? kRegionLowXLowQ : highq ? kRegionLowXHighQ : kRegionLowX;
    return lowq ? kRegionLowQ : highq ? kRegionHighQ : kRegionInterior;
}

// PAPER.md L1720, the other extrapolation options of LHAPDF 6, applied to a query before anything else looks at it:
// freeze = the point moved to the closest point of the grid's range (a coordinate inside its range is not touched),
// error = a valid query outside the range becomes an invalid one (C-10).  Warp-uniform branch on the option.
__device__ __forceinline__ void apply_extrapolation(const GridDev &G, double &x, double &q2)
{
    if (G.extrap == kExtrapContinuation) return;
    const double x0 = G.xk[0], q0 = G.qk[0], q1 = G.qk[G.nqtot - 1];
    if (!(finite_pos(x) && finite_pos(q2)) || x > G.xk[G.nx - 1]) return;          // invalid stays invalid
    if (G.extrap == kExtrapFreeze) { x = x < x0 ? x0 : x; q2 = q2 < q0 ? q0 : (q2 > q1 ? q1 : q2); }
    else if (x < x0 || q2 < q0 || q2 > q1) x = __longlong_as_double(0x7ff8000000000000LL);
}
// xfxQ: Q -> Q2; Q <= 0 is invalid although its square is not
__device__ __forceinline__ double q_to_q2(double q) { return q > 0.0 ? q * q : __longlong_as_double(0x7ff8000000000000LL); }

// x-axis point inside the knot range: cell i, t = (ln x - u_i)/(u_{i+1}-u_i)
__device__ __forceinline__ void x_point_cell(const GridDev &G, int i, double t, Point1D &p)
{
    CellTab c = G.cx[i];
    hermite_weights(t, c, p.w);
    p.idx[0] = i > 0 ? i - 1 : i;
    p.idx[1] = i;
    p.idx[2] = i + 1;
    p.idx[3] = i + 2 < G.nx ? i + 2 : i + 1;
}

__device__ __forceinline__ int x_point(const GridDev &G, double x, Point1D &p)
{
    int i = find_cell(G.xk, G.nx, x);
    // t = 1 exactly on the last knot (the only knot that belongs to the cell on its left, C-4)
    double t = (x == G.xk[i + 1]) ? 1.0 : (pdf_log(x) - G.cx[i].lo_log) * G.cx[i].inv_d;
    x_point_cell(G, i, t, p);
    return i;
}

// Q2-axis point: jg = global index of the cell's lower knot
__device__ __forceinline__ void q_point_cell(const GridDev &G, int jg, double t, Point1D &p)
{
    CellTab c = G.cq[jg];
    hermite_weights(t, c, p.w);
    p.idx[0] = (c.aL == 1.0) ? jg : jg - 1;     // no left neighbour inside the sub-grid
    p.idx[1] = jg;
    p.idx[2] = jg + 1;
    p.idx[3] = (c.aR == 1.0) ? jg + 1 : jg + 2;
}

// in-range Q2: returns sub-grid k; writes local cell j
__device__ __forceinline__ int q_locate(const GridDev &G, double q2, int &j, int &jg)
{
    int g = find_last_le(G.qk, G.nqtot, q2);
    int k = G.sub_of[g];
    int nqk = G.qoff[k + 1] - G.qoff[k];
    j = g - G.qoff[k];
    if (j > nqk - 2) j = nqk - 2;               // only Q2 == Q2max lands on a last knot
    jg = G.qoff[k] + j;
    return k;
}

__device__ __forceinline__ void q_point(const GridDev &G, double q2, Point1D &p)
{
    int j, jg;
    q_locate(G, q2, j, jg);
    double t = (q2 == G.qk[jg + 1]) ? 1.0 : (pdf_log(q2) - G.cq[jg].lo_log) * G.cq[jg].inv_d;
    q_point_cell(G, jg, t, p);
}

// x-axis descriptor: in range -> one point; below X_0 -> the two anchor points + theta (C-7)
struct XDesc { bool low; Point1D p0, p1; double theta; };
// Q2-axis descriptor for Q2 >= Q2min: in range -> one point; above -> two anchors + theta (C-8)
struct QDesc { bool high; Point1D p0, p1; double theta; };

__device__ __forceinline__ void make_xdesc(const GridDev &G, double x, XDesc &d)
{
    d.low = x < G.xk[0];
    if (!d.low) { x_point(G, x, d.p0); return; }
    x_point_cell(G, 0, 0.0, d.p0);
    if (G.nx >= 3) x_point_cell(G, 1, 0.0, d.p1); else x_point_cell(G, 0, 1.0, d.p1);
    d.theta = (pdf_log(x) - G.uk[0]) / (G.uk[1] - G.uk[0]);
}

__device__ __forceinline__ void make_qdesc(const GridDev &G, double q2, QDesc &d)
{
    int last = G.nqtot - 1;
    d.high = q2 > G.qk[last];
    if (!d.high) { q_point(G, q2, d.p0); return; }
    q_point_cell(G, last - 1, 0.0, d.p0);
    q_point_cell(G, last - 1, 1.0, d.p1);
    d.theta = (pdf_log(q2) - G.sk[last - 1]) / (G.sk[last] - G.sk[last - 1]);
}

// C-7 / C-8 switch (L1722): log form iff both anchors exceed 1e-3, per flavour
__device__ __forceinline__ double continue_two(double f0, double f1, double theta)
{
    if (f0 > 1e-3 && f1 > 1e-3) {
        double l0 = pdf_log(f0), l1 = pdf_log(f1);       // the path's own logarithm (<= 1 ulp, 38 instructions against ~85)
        return exp(l0 + theta * (l1 - l0));
    }
    return f0 + theta * (f1 - f0);
}

// C-9, eq. 3.4 with the limits of eq. 3.5
__device__ __forceinline__ double lowq_continue(double fmin, double fplus, double r)
{
    double gamma = 1.0;
    if (fmin > 1e-5) gamma = fmax(-2.5, (fplus - fmin) / (0.01 * fmin));
    return fmin * pow(r, (gamma - 1.0) * r + 1.0);
}

// the same with ln r shared by the 11 flavours of a query: r^e = exp(e ln r) (binned path)
__device__ __forceinline__ double lowq_continue_ln(double fmin, double fplus, double r, double lnr)
{
    double gamma = 1.0;
    if (fmin > 1e-5) gamma = fmax(-2.5, (fplus - fmin) / (0.01 * fmin));
    return fmin * exp(((gamma - 1.0) * r + 1.0) * lnr);
}

// C-6 as a 16-term tensor sum for one flavour column
__device__ __forceinline__ double stencil_col(const GridDev &G, const double *__restrict__ Vm,
                                              const Point1D &xp, const Point1D &qp, int col)
{
    double acc = 0.0;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
        const double *row = Vm + (size_t)qp.idx[b] * G.nx * G.nfp + col;
        double rb = 0.0;
#pragma unroll
        for (int a = 0; a < 4; ++a) rb = fma(xp.w[a], __ldg(row + (size_t)xp.idx[a] * G.nfp), rb);
        acc = fma(qp.w[b], rb, acc);
    }
    return acc;
}

__device__ __forceinline__ double value_inq(const GridDev &G, const double *Vm, const XDesc &X,
                                            const Point1D &qp, int col)
{
    if (!X.low) return stencil_col(G, Vm, X.p0, qp, col);
    return continue_two(stencil_col(G, Vm, X.p0, qp, col), stencil_col(G, Vm, X.p1, qp, col), X.theta);
}

__device__ __forceinline__ double value_geq(const GridDev &G, const double *Vm, const XDesc &X,
                                            const QDesc &Q, int col)
{
    if (!Q.high) return value_inq(G, Vm, X, Q.p0, col);
    return continue_two(value_inq(G, Vm, X, Q.p0, col), value_inq(G, Vm, X, Q.p1, col), Q.theta);
}

// everything a thread needs to evaluate any flavour column of one valid query
struct QueryPlan {
    XDesc X;
    QDesc Q;        // for q2 (in range / high) or for Q2min when lowq
    QDesc Qplus;    // for 1.01*Q2min, only when lowq
    bool lowq;
    double r;       // q2 / Q2min when lowq
};

__device__ __forceinline__ void make_plan(const GridDev &G, double x, double q2, QueryPlan &P)
{
    make_xdesc(G, x, P.X);
    P.lowq = q2 < G.qk[0];
    if (!P.lowq) { make_qdesc(G, q2, P.Q); return; }
    make_qdesc(G, G.qk[0], P.Q);
    make_qdesc(G, G.q2plus, P.Qplus);
    P.r = q2 / G.qk[0];
}

__device__ __forceinline__ double plan_value(const GridDev &G, const double *Vm, const QueryPlan &P, int col)
{
    if (!P.lowq) return value_geq(G, Vm, P.X, P.Q, col);
    return lowq_continue(value_geq(G, Vm, P.X, P.Q, col), value_geq(G, Vm, P.X, P.Qplus, col), P.r);
}

__device__ __forceinline__ double qnan() { return __longlong_as_double(0x7ff8000000000000LL); }

}  // namespace pdfg
