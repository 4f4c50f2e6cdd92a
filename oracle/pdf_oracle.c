/*
 * pdf_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see pdf_oracle.h).
 *
 * Plain CPU fp64 statement of LHAPDF-style log-bicubic PDF interpolation with
 * the default (MSTW / LHAPDF5 "continuation") extrapolation, the cubic
 * alpha_s(Q2) interpolation and the two-parton luminosity sum, following
 * PAPER.md section 3.2 (L1712-L1746), section 3.3.2 (L1831-L1835), eq. 3.3
 * (L1699) and eq. 4.1 (L1949) in the readings listed in DESIGN.md.
 *
 * Style: the definition written out.  Knot searches are linear scans, the
 * Hermite cubic is evaluated from knot values and finite-difference knot
 * slopes (not from precomputed weights), the 2-D value is "x first, then Q2".
 * No blocking, no fusion, no tables.  OpenMP only splits the query loop.
 */
#include "pdf_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

struct oracle_grid {
    int nx, nsub, nflav, nmem;
    double *x;      /* [nx] knots                                  */
    double *u;      /* [nx] ln x (C-1)                             */
    int *nq;        /* [nsub]                                      */
    int *qoff;      /* [nsub] offset of sub-grid k in q2 / s       */
    int nqtot;
    double *q2;     /* concatenated Q2 knots                       */
    double *s;      /* ln Q2                                       */
    size_t *suboff; /* [nsub] offset of block k inside one member  */
    size_t memstride;
    double *values;
    int *pids;
    int na;         /* alpha_s knots                               */
    double *aq2, *as, *aval;
    int alphas_mode;
    int extrap;                 /* ORACLE_EXTRAP_* (L1720) */
    double *C;      /* [nflav][nflav] or NULL                      */
};

static int finite_pos(double v) { return isfinite(v) && v > 0.0; }

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------ */
/* grid handle                                                          */
/* ------------------------------------------------------------------ */
int oracle_grid_create(oracle_grid **out, int nx, const double *x_knots,
                       int nsub, const int *nq, const double *q2_knots,
                       const double *values, int nflav,
                       const int *flavour_pids, int nmem)
{
    if (!out || !x_knots || !nq || !q2_knots || !values || !flavour_pids)
        return -1;
    if (nx < 2 || nsub < 1 || nflav < 1 || nmem < 1) return -1;
    for (int i = 0; i < nx; ++i) {
        if (!finite_pos(x_knots[i])) return -1;
        if (i && !(x_knots[i] > x_knots[i - 1])) return -1;
    }
    int tot = 0;
    for (int k = 0; k < nsub; ++k) {
        if (nq[k] < 2) return -1;
        for (int j = 0; j < nq[k]; ++j) {
            double q = q2_knots[tot + j];
            if (!finite_pos(q)) return -1;
            if (j && !(q > q2_knots[tot + j - 1])) return -1;
        }
        /* L1714: sub-grids meet at the threshold knot, stored in both */
        if (k && q2_knots[tot] != q2_knots[tot - 1]) return -1;
        tot += nq[k];
    }
    oracle_grid *g = (oracle_grid *)calloc(1, sizeof *g);
    if (!g) return -2;
    g->nx = nx; g->nsub = nsub; g->nflav = nflav; g->nmem = nmem; g->nqtot = tot;
    g->x = (double *)malloc(sizeof(double) * nx);
    g->u = (double *)malloc(sizeof(double) * nx);
    g->nq = (int *)malloc(sizeof(int) * nsub);
    g->qoff = (int *)malloc(sizeof(int) * nsub);
    g->q2 = (double *)malloc(sizeof(double) * tot);
    g->s = (double *)malloc(sizeof(double) * tot);
    g->suboff = (size_t *)malloc(sizeof(size_t) * nsub);
    g->pids = (int *)malloc(sizeof(int) * nflav);
    for (int i = 0; i < nx; ++i) { g->x[i] = x_knots[i]; g->u[i] = log(x_knots[i]); }
    size_t off = 0; int qo = 0;
    for (int k = 0; k < nsub; ++k) {
        g->nq[k] = nq[k]; g->qoff[k] = qo; g->suboff[k] = off;
        off += (size_t)nx * nq[k] * nflav; qo += nq[k];
    }
    g->memstride = off;
    for (int j = 0; j < tot; ++j) { g->q2[j] = q2_knots[j]; g->s[j] = log(q2_knots[j]); }
    for (int f = 0; f < nflav; ++f) g->pids[f] = flavour_pids[f];
    size_t nval = off * (size_t)nmem;
    for (size_t e = 0; e < nval; ++e)
        if (!isfinite(values[e])) { oracle_grid_destroy(g); return -1; }
    g->values = (double *)malloc(sizeof(double) * nval);
    if (!g->values) { oracle_grid_destroy(g); return -2; }
    memcpy(g->values, values, sizeof(double) * nval);
    *out = g;
    return 0;
}

int oracle_grid_destroy(oracle_grid *g)
{
    if (!g) return 0;
    free(g->x); free(g->u); free(g->nq); free(g->qoff); free(g->q2); free(g->s);
    free(g->suboff); free(g->values); free(g->pids);
    free(g->aq2); free(g->as); free(g->aval); free(g->C);
    free(g);
    return 0;
}

int oracle_grid_set_alphas(oracle_grid *g, int n, const double *q2_knots,
                           const double *values)
{
    if (!g || n < 2 || !q2_knots || !values) return -1;
    /* knots increase; a knot may appear twice (a flavour threshold: the end of one sub-line and the start of the
     * next, L1835 "the sub-grids mechanism ... flavor thresholds"), every sub-line has at least 2 knots */
    for (int j = 0; j < n; ++j) {
        if (!finite_pos(q2_knots[j]) || !isfinite(values[j])) return -1;
        if (j && !(q2_knots[j] >= q2_knots[j - 1])) return -1;
        if (j && q2_knots[j] == q2_knots[j - 1] && (j == 1 || j == n - 1 || q2_knots[j - 1] == q2_knots[j - 2] ||
                                                      q2_knots[j + 1] == q2_knots[j])) return -1;
    }
    free(g->aq2); free(g->as); free(g->aval);
    g->na = n;
    g->aq2 = (double *)malloc(sizeof(double) * n);
    g->as = (double *)malloc(sizeof(double) * n);
    g->aval = (double *)malloc(sizeof(double) * n);
    for (int j = 0; j < n; ++j) {
        g->aq2[j] = q2_knots[j]; g->as[j] = log(q2_knots[j]); g->aval[j] = values[j];
    }
    return 0;
}

int oracle_grid_set_extrapolation(oracle_grid *g, int mode)
{
    if (!g || mode < ORACLE_EXTRAP_CONTINUATION || mode > ORACLE_EXTRAP_ERROR) return -1;
    g->extrap = mode;
    return 0;
}

int oracle_grid_set_alphas_mode(oracle_grid *g, int mode)
{
    if (!g || (mode != ORACLE_ALPHAS_FREEZE && mode != ORACLE_ALPHAS_LOGGRAD)) return -1;
    g->alphas_mode = mode;
    return 0;
}

int oracle_grid_set_coupling(oracle_grid *g, const double *C)
{
    if (!g || !C) return -1;
    size_t n = (size_t)g->nflav * g->nflav;
    for (size_t e = 0; e < n; ++e) if (!isfinite(C[e])) return -1;
    free(g->C);
    g->C = (double *)malloc(sizeof(double) * n);
    memcpy(g->C, C, sizeof(double) * n);
    return 0;
}

int oracle_grid_limits(const oracle_grid *g, double *xmin, double *xmax,
                       double *q2min, double *q2max)
{
    if (!g) return -1;
    if (xmin) *xmin = g->x[0];
    if (xmax) *xmax = g->x[g->nx - 1];
    if (q2min) *q2min = g->q2[0];
    if (q2max) *q2max = g->q2[g->nqtot - 1];
    return 0;
}

/* ------------------------------------------------------------------ */
/* C-5: 1-D cubic Hermite operator with finite-difference knot slopes   */
/* ------------------------------------------------------------------ */

/* slope m_c at knot c of the line (w_0..w_{m-1}; v at stride).  Interior knot:
 * plain average of the two secant slopes; end knots: the one secant. */
static double knot_slope(int m, const double *w, const double *v, long stride, int c)
{
    if (c == 0)
        return (v[stride] - v[0]) / (w[1] - w[0]);
    if (c == m - 1)
        return (v[(long)(m - 1) * stride] - v[(long)(m - 2) * stride]) / (w[m - 1] - w[m - 2]);
    double right = (v[(long)(c + 1) * stride] - v[(long)c * stride]) / (w[c + 1] - w[c]);
    double left = (v[(long)c * stride] - v[(long)(c - 1) * stride]) / (w[c] - w[c - 1]);
    return 0.5 * (right + left);
}

/* p(t) on cell c (knots c, c+1) at abscissa wpt */
static double hermite_cell(int m, const double *w, const double *v, long stride,
                           int c, double wpt)
{
    double delta = w[c + 1] - w[c];
    double t = (wpt - w[c]) / delta;
#ifdef ORACLE_S3_BILINEAR
    /* S-3 reading B, the literal one ("near grid edges ... automatically switches to
     * bilinear interpolation, which requires 2 neighbor knots only"): plain linear in an end cell of
     * the knot line.  Documentation switch only: the default build (reading A, S-3) keeps the
     * cubic with a one-sided end slope; tests/test_oracle_pins.py builds this variant to show what
     * distinguishes the two (C1 at the first interior knot). */
    if (c == 0 || c + 1 == m - 1)
        return v[(long)c * stride] + t * (v[(long)(c + 1) * stride] - v[(long)c * stride]);
#endif
    /* the four Hermite basis cubics 2t^3-3t^2+1, t^3-2t^2+t, -2t^3+3t^2, t^3-t^2, written in
     * factored form so that each keeps its relative accuracy where it vanishes (t -> 0, 1) */
    double omt = 1.0 - t;
    double h00 = (1.0 + 2.0 * t) * (omt * omt);
    double h10 = t * (omt * omt);
    double h01 = (t * t) * (3.0 - 2.0 * t);
    double h11 = -((t * t) * omt);
    double mc = knot_slope(m, w, v, stride, c);
    double mc1 = knot_slope(m, w, v, stride, c + 1);
    return h00 * v[(long)c * stride] + h10 * (delta * mc)
         + h01 * v[(long)(c + 1) * stride] + h11 * (delta * mc1);
}

/* dp/dt of the same cubic (used only for the condition scale of the parity metric) */
static double hermite_cell_dt(int m, const double *w, const double *v, long stride,
                              int c, double wpt)
{
    double delta = w[c + 1] - w[c];
    double t = (wpt - w[c]) / delta;
    double omt = 1.0 - t;
    double d00 = -6.0 * t * omt, d10 = omt * (1.0 - 3.0 * t), d01 = 6.0 * t * omt, d11 = t * (3.0 * t - 2.0);
    double mc = knot_slope(m, w, v, stride, c);
    double mc1 = knot_slope(m, w, v, stride, c + 1);
    return d00 * v[(long)c * stride] + d10 * (delta * mc)
         + d01 * v[(long)(c + 1) * stride] + d11 * (delta * mc1);
}

/* Condition numbers returned for the parity metric (C-12) come in two parts, kept apart so
 * that each has its own, physically meaningful floor:
 *   S[0] = sum |Wx_a Wq_b V_ab|: what the rounding of the 16-term sum acts on;
 *   S[1] = |df/dt_x| (1 + |ln x|/du) + |df/dt_q| (1 + |ln Q2|/ds): t = (ln v - ln knot)/delta is only
 *          known to a few 2^-52 (1 + |ln v|/delta) (one ulp each of ln v and ln knot, divided by delta),
 *          which moves the value by |df/dt| times that.
 * Both are propagated to first order (same coefficients) through the extrapolation formulas. */
static double t_cond(const double *w, int c, double wpt)
{
    return 1.0 + fabs(wpt) / (w[c + 1] - w[c]);
}

/* The knots a cell's cubic depends on are c-1..c+2 where they exist.  This
 * returns that window [lo,hi]; evaluating hermite_cell on the sub-line
 * (w+lo, hi-lo+1 knots, cell c-lo) is identical to evaluating it on the full
 * line, because a window end coincides with a line end whenever it is used as
 * an "end knot". */
static void cell_window(int m, int c, int *lo, int *hi)
{
    *lo = c > 0 ? c - 1 : 0;
    *hi = c + 2 < m ? c + 2 : m - 1;
}

int oracle_weights_1d(int m, const double *knots_log, double wlog, int cell, double w4[4])
{
    if (m < 2 || !knots_log || !w4 || cell < 0 || cell > m - 2) return -1;
    int lo, hi;
    cell_window(m, cell, &lo, &hi);
    for (int a = 0; a < 4; ++a) w4[a] = 0.0;
    for (int kn = lo; kn <= hi; ++kn) {
        double e[4] = {0.0, 0.0, 0.0, 0.0};
        e[kn - lo] = 1.0;
        w4[kn - (cell - 1)] = hermite_cell(hi - lo + 1, knots_log + lo, e, 1, cell - lo, wlog);
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* C-2, C-3, C-4: region, sub-grid, cell                                */
/* ------------------------------------------------------------------ */
static int find_subgrid(const oracle_grid *g, double q2)
{
    int k = g->nsub - 1;
    while (k > 0 && g->q2[g->qoff[k]] > q2) --k;   /* largest k with Q_{k,0} <= q2 */
    return k;
}

static int find_cell(int m, const double *knots, double v)
{
    int c = m - 2;
    while (c > 0 && knots[c] > v) --c;             /* largest c <= m-2 with knot_c <= v */
    return c;
}

static int classify(const oracle_grid *g, double x, double q2)
{
    if (!(isfinite(x) && isfinite(q2))) return ORACLE_REGION_INVALID;
    if (!(x > 0.0) || !(q2 > 0.0) || x > g->x[g->nx - 1]) return ORACLE_REGION_INVALID;
    int lowx = x < g->x[0];
    int lowq = q2 < g->q2[0];
    int highq = q2 > g->q2[g->nqtot - 1];
    if (lowx) return lowq ? ORACLE_REGION_LOWX_LOWQ : highq ? ORACLE_REGION_LOWX_HIGHQ : ORACLE_REGION_LOWX;
    return lowq ? ORACLE_REGION_LOWQ : highq ? ORACLE_REGION_HIGHQ : ORACLE_REGION_INTERIOR;
}

/* L1720 (reading R-7): the point a valid query is evaluated at under the grid's extrapolation option */
static void apply_extrapolation(const oracle_grid *g, double *x, double *q2)
{
    if (g->extrap == ORACLE_EXTRAP_CONTINUATION) return;
    int r = classify(g, *x, *q2);
    if (r == ORACLE_REGION_INVALID || r == ORACLE_REGION_INTERIOR) return;
    if (g->extrap == ORACLE_EXTRAP_ERROR) { *x = NAN; return; }           /* an error: the query is invalid */
    double q2min = g->q2[0], q2max = g->q2[g->nqtot - 1];                 /* freeze */
    if (*x < g->x[0]) *x = g->x[0];
    if (*q2 < q2min) *q2 = q2min;
    if (*q2 > q2max) *q2 = q2max;
}

int oracle_locate(const oracle_grid *g, long long n, const double *x,
                  const double *q2, int *ix, int *iq, int *isub, int *region)
{
    if (!g || n < 0 || !x || !q2) return -1;
#pragma omp parallel for schedule(static)
    for (long long e = 0; e < n; ++e) {
        double xe = x[e], qe = q2[e];
        apply_extrapolation(g, &xe, &qe);
        int r = classify(g, xe, qe);
        int i = -1, j = -1, k = -1;
        if (r != ORACLE_REGION_INVALID) {
            /* low-x is anchored on knots X_0, X_1 */
            i = (r == ORACLE_REGION_LOWX || r == ORACLE_REGION_LOWX_LOWQ ||
                 r == ORACLE_REGION_LOWX_HIGHQ) ? 0 : find_cell(g->nx, g->x, xe);
            if (r == ORACLE_REGION_LOWQ || r == ORACLE_REGION_LOWX_LOWQ) {
                k = 0; j = 0;                       /* anchored on Q2_min */
            } else if (r == ORACLE_REGION_HIGHQ || r == ORACLE_REGION_LOWX_HIGHQ) {
                k = g->nsub - 1; j = g->nq[k] - 2; /* two highest knots  */
            } else {
                k = find_subgrid(g, qe);
                j = find_cell(g->nq[k], g->q2 + g->qoff[k], qe);
            }
        }
        if (ix) ix[e] = i;
        if (iq) iq[e] = j;
        if (isub) isub[e] = k;
        if (region) region[e] = r;
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* C-6: interior value, x first then Q2                                 */
/* ------------------------------------------------------------------ */
static const double *block_ptr(const oracle_grid *g, int mem, int k)
{
    return g->values + (size_t)mem * g->memstride + g->suboff[k];
}

/* value and, if S != NULL, the two condition numbers S[0], S[1] (see t_cond) at an in-range point */
static void interior_value(const oracle_grid *g, int mem, int fcol, double x,
                           double q2, double *val, double *S)
{
    int k = find_subgrid(g, q2);
    int nqk = g->nq[k];
    const double *sk = g->s + g->qoff[k];
    int i = find_cell(g->nx, g->x, x);
    int j = find_cell(nqk, g->q2 + g->qoff[k], q2);
    double lx = log(x), lq = log(q2);
    const double *B = block_ptr(g, mem, k);
    long xstride = (long)nqk * g->nflav;
    int jlo, jhi;
    cell_window(nqk, j, &jlo, &jhi);
    double r[4];
    for (int b = jlo; b <= jhi; ++b)               /* C-5 along x on each Q2 row */
        r[b - jlo] = hermite_cell(g->nx, g->u, B + (long)b * g->nflav + fcol, xstride, i, lx);
    *val = hermite_cell(jhi - jlo + 1, sk + jlo, r, 1, j - jlo, lq); /* C-5 along ln Q2 */
    if (S) {
        double wx[4], wq[4];
        oracle_weights_1d(g->nx, g->u, lx, i, wx);
        oracle_weights_1d(nqk, sk, lq, j, wq);
        double acc = 0.0;
        for (int a = 0; a < 4; ++a) {
            int ia = i - 1 + a;
            if (ia < 0 || ia >= g->nx) continue;
            for (int b = 0; b < 4; ++b) {
                int jb = j - 1 + b;
                if (jb < 0 || jb >= nqk) continue;
                acc += fabs(wx[a] * wq[b] * B[((long)ia * nqk + jb) * g->nflav + fcol]);
            }
        }
        /* first-order sensitivity to the rounding of t_x and t_q */
        double rd[4];
        for (int b = jlo; b <= jhi; ++b)
            rd[b - jlo] = hermite_cell_dt(g->nx, g->u, B + (long)b * g->nflav + fcol, xstride, i, lx);
        double dfx = hermite_cell(jhi - jlo + 1, sk + jlo, rd, 1, j - jlo, lq);
        double dfq = hermite_cell_dt(jhi - jlo + 1, sk + jlo, r, 1, j - jlo, lq);
        S[0] = acc;
        S[1] = fabs(dfx) * t_cond(g->u, i, lx) + fabs(dfq) * t_cond(sk, j, lq);
    }
}

/* C-7 / C-8 switch: continuation from two anchor values at abscissa theta
 * (theta = 0 at anchor 0, 1 at anchor 1).  Log form iff both > 1e-3 (L1722). */
static void continue_two(double f0, const double *S0, double f1, const double *S1, double theta,
                         double theta_cond, double *val, double *S)
{
    if (f0 > 1e-3 && f1 > 1e-3) {
        double l0 = log(f0), l1 = log(f1);
        double v = exp(l0 + theta * (l1 - l0));
        *val = v;
        if (S) {
            for (int c = 0; c < 2; ++c)
                S[c] = fabs(v) * (fabs(1.0 - theta) * S0[c] / f0 + fabs(theta) * S1[c] / f1);
            S[1] += fabs(v) * theta_cond * fabs(l1 - l0);       /* rounding of theta itself */
        }
    } else {
        *val = f0 + theta * (f1 - f0);
        if (S) {
            for (int c = 0; c < 2; ++c) S[c] = fabs(1.0 - theta) * S0[c] + fabs(theta) * S1[c];
            S[1] += theta_cond * fabs(f1 - f0);
        }
    }
}

/* value at Q2_min <= q2 <= Q2_max for any valid x: C-6, or C-7 when x < X_0 */
static void value_inq(const oracle_grid *g, int mem, int fcol, double x, double q2,
                      double *val, double *S)
{
    if (x >= g->x[0]) { interior_value(g, mem, fcol, x, q2, val, S); return; }
    double f0, f1, S0[2], S1[2];
    interior_value(g, mem, fcol, g->x[0], q2, &f0, S ? S0 : NULL);
    interior_value(g, mem, fcol, g->x[1], q2, &f1, S ? S1 : NULL);
    double theta = (log(x) - g->u[0]) / (g->u[1] - g->u[0]);
    continue_two(f0, S0, f1, S1, theta, t_cond(g->u, 0, log(x)), val, S);
}

/* value for q2 >= Q2_min: in range, or C-8 (two highest knots, in ln Q2) */
static void value_geqmin(const oracle_grid *g, int mem, int fcol, double x, double q2,
                         double *val, double *S)
{
    int last = g->nqtot - 1;
    if (q2 <= g->q2[last]) { value_inq(g, mem, fcol, x, q2, val, S); return; }
    double g0, g1, S0[2], S1[2];
    value_inq(g, mem, fcol, x, g->q2[last - 1], &g0, S ? S0 : NULL);
    value_inq(g, mem, fcol, x, g->q2[last], &g1, S ? S1 : NULL);
    double theta = (log(q2) - g->s[last - 1]) / (g->s[last] - g->s[last - 1]);
    continue_two(g0, S0, g1, S1, theta, t_cond(g->s, last - 1, log(q2)), val, S);
}

/* full value for a valid query: adds C-9 (eq. 3.4, limits eq. 3.5) */
static void value_any(const oracle_grid *g, int mem, int fcol, double x, double q2,
                      double *val, double *S)
{
    double q2min = g->q2[0];
    if (q2 >= q2min) { value_geqmin(g, mem, fcol, x, q2, val, S); return; }
    double fmin, fplus, Smin[2], Splus[2];
    value_geqmin(g, mem, fcol, x, q2min, &fmin, S ? Smin : NULL);
    value_geqmin(g, mem, fcol, x, 1.01 * q2min, &fplus, S ? Splus : NULL);
    double r = q2 / q2min;
    double gamma = 1.0;
    int free_gamma = 0;
    if (fmin > 1e-5) {
        double gfd = (fplus - fmin) / (0.01 * fmin);
        if (gfd > -2.5) { gamma = gfd; free_gamma = 1; } else gamma = -2.5;
    }
    double v = fmin * pow(r, (gamma - 1.0) * r + 1.0);
    *val = v;
    if (S) {
        /* d v = (v/fmin) d fmin + v ln(r) r d gamma,  d gamma = d fplus/(0.01 fmin) - fplus d fmin/(0.01 fmin^2) */
        for (int c = 0; c < 2; ++c) {
            double sc = (fmin != 0.0) ? fabs(v / fmin) * Smin[c] : pow(r, (gamma - 1.0) * r + 1.0) * Smin[c];
            if (free_gamma)
                sc += fabs(v * log(r) * r) * (Splus[c] / (0.01 * fmin) + fabs(fplus) * Smin[c] / (0.01 * fmin * fmin));
            S[c] = sc;
        }
    }
}

static int pid_column(const oracle_grid *g, int pid)
{
    if (pid == 0) pid = 21;                         /* C-11: 0 is an alias of the gluon */
    for (int f = 0; f < g->nflav; ++f) if (g->pids[f] == pid) return f;
    return -1;
}

int oracle_xfxq2(const oracle_grid *g, const int *pids, int npid, long long n,
                 const double *x, const double *q2, const int *member,
                 double *out, double *scale)
{
    if (!g || !pids || npid < 1 || n < 0 || !x || !q2 || !out) return -1;
    int *col = (int *)malloc(sizeof(int) * npid);
    for (int p = 0; p < npid; ++p) col[p] = pid_column(g, pids[p]);
    int bad_member = 0;
#pragma omp parallel for schedule(static)
    for (long long e = 0; e < n; ++e) {
        int mem = member ? member[e] : 0;
        double xe = x[e], qe = q2[e];
        apply_extrapolation(g, &xe, &qe);
        int r = classify(g, xe, qe);
        if (mem < 0 || mem >= g->nmem) { r = ORACLE_REGION_INVALID; bad_member = 1; }
        for (int p = 0; p < npid; ++p) {
            double v, S[2] = {0.0, 0.0};
            if (r == ORACLE_REGION_INVALID) { v = NAN; S[0] = S[1] = NAN; }   /* C-10 */
            else if (col[p] < 0) { v = 0.0; }                                 /* C-11 */
            else value_any(g, mem, col[p], xe, qe, &v, scale ? S : NULL);
            out[e * npid + p] = v;
            if (scale) { scale[(e * npid + p) * 2] = S[0]; scale[(e * npid + p) * 2 + 1] = S[1]; }
        }
    }
    free(col);
    (void)bad_member;
    return 0;
}

/* ------------------------------------------------------------------ */
/* C-alpha                                                              */
/* ------------------------------------------------------------------ */
int oracle_alphas_q2(const oracle_grid *g, long long n, const double *q2, double *out)
{
    if (!g || g->na < 2 || n < 0 || !q2 || !out) return -1;
    int m = g->na;
#pragma omp parallel for schedule(static)
    for (long long e = 0; e < n; ++e) {
        double q = q2[e];
        double v;
        if (!(isfinite(q) && q > 0.0)) v = NAN;
        else if (q > g->aq2[m - 1]) v = g->aval[m - 1];                 /* L1746: constant */
        else if (q < g->aq2[0]) {
            if (g->alphas_mode == ORACLE_ALPHAS_LOGGRAD)                /* L1746, LHAPDF   */
                v = g->aval[0] * pow(q / g->aq2[0],
                                     log(g->aval[1] / g->aval[0]) / log(g->aq2[1] / g->aq2[0]));
            else v = g->aval[0];                                        /* L1835, PDFFlow  */
        } else {
            /* the sub-line of q: it starts at the last repeated knot <= q (a query on a threshold belongs to the
             * upper sub-line, as C-3) and ends at the next repeated knot; C-5 inside it, one-sided slopes at its ends */
            int lo = 0, hi = m - 1;
            for (int j = 1; j < m; ++j)
                if (g->aq2[j] == g->aq2[j - 1]) { if (g->aq2[j] <= q) lo = j; else { hi = j - 1; break; } }
            int c = find_cell(hi - lo + 1, g->aq2 + lo, q);
            v = hermite_cell(hi - lo + 1, g->as + lo, g->aval + lo, 1, c, log(q));
        }
        out[e] = v;
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* C-L: luminosity, eq. 3.3 / eq. 4.1                                   */
/* ------------------------------------------------------------------ */
int oracle_lumi(const oracle_grid *g, long long n, const double *x1,
                const double *x2, const double *q2, const double *weights,
                double *out, double *scale)
{
    if (!g || !g->C || n < 0 || !x1 || !x2 || !q2 || !weights || !out) return -1;
    int nf = g->nflav;
#pragma omp parallel for schedule(static)
    for (long long e = 0; e < n; ++e) {
        double xa = x1[e], qa = q2[e], xb = x2[e], qb = q2[e];       /* the points the two partons are evaluated at (L1720) */
        apply_extrapolation(g, &xa, &qa);
        apply_extrapolation(g, &xb, &qb);
        int r1 = classify(g, xa, qa), r2 = classify(g, xb, qb);
        if (r1 == ORACLE_REGION_INVALID || r2 == ORACLE_REGION_INVALID) {
            out[e] = NAN; if (scale) scale[2 * e] = scale[2 * e + 1] = NAN; continue;
        }
        double f1[64], f2[64], s1[64][2], s2[64][2];
        for (int f = 0; f < nf; ++f) {
            double v, S[2] = {0.0, 0.0};
            value_any(g, 0, f, xa, qa, &v, scale ? S : NULL);
            f1[f] = v / x1[e]; s1[f][0] = S[0] / x1[e]; s1[f][1] = S[1] / x1[e];
            value_any(g, 0, f, xb, qb, &v, scale ? S : NULL);
            f2[f] = v / x2[e]; s2[f][0] = S[0] / x2[e]; s2[f][1] = S[1] / x2[e];
        }
        double acc = 0.0, sacc[2] = {0.0, 0.0};
        for (int i = 0; i < nf; ++i)
            for (int j = 0; j < nf; ++j) {
                acc += g->C[i * nf + j] * f1[i] * f2[j];
                /* first-order propagation of the per-flavour condition numbers through the product */
                for (int c = 0; c < 2; ++c)
                    sacc[c] += fabs(g->C[i * nf + j]) * (s1[i][c] * fabs(f2[j]) + fabs(f1[i]) * s2[j][c]);
            }
        out[e] = weights[e] * acc;
        if (scale) { scale[2 * e] = fabs(weights[e]) * sacc[0]; scale[2 * e + 1] = fabs(weights[e]) * sacc[1]; }
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* P-10 self-check: three evaluation orders of the interior value       */
/* ------------------------------------------------------------------ */
int oracle_interior_order(const oracle_grid *g, int order, int fcol, int member,
                          long long n, const double *x, const double *q2, double *out)
{
    if (!g || fcol < 0 || fcol >= g->nflav || member < 0 || member >= g->nmem) return -1;
    for (long long e = 0; e < n; ++e) {
        if (classify(g, x[e], q2[e]) != ORACLE_REGION_INTERIOR) { out[e] = NAN; continue; }
        if (order == 0) { interior_value(g, member, fcol, x[e], q2[e], &out[e], NULL); continue; }
        int k = find_subgrid(g, q2[e]);
        int nqk = g->nq[k];
        const double *sk = g->s + g->qoff[k];
        int i = find_cell(g->nx, g->x, x[e]);
        int j = find_cell(nqk, g->q2 + g->qoff[k], q2[e]);
        double lx = log(x[e]), lq = log(q2[e]);
        const double *B = block_ptr(g, member, k);
        if (order == 1) {                           /* Q2 first on each x column, then x */
            int ilo, ihi;
            cell_window(g->nx, i, &ilo, &ihi);
            double c[4];
            for (int a = ilo; a <= ihi; ++a)
                c[a - ilo] = hermite_cell(nqk, sk, B + (long)a * nqk * g->nflav + fcol,
                                          g->nflav, j, lq);
            out[e] = hermite_cell(ihi - ilo + 1, g->u + ilo, c, 1, i - ilo, lx);
        } else {                                    /* 16-term tensor sum               */
            double wx[4], wq[4], acc = 0.0;
            oracle_weights_1d(g->nx, g->u, lx, i, wx);
            oracle_weights_1d(nqk, sk, lq, j, wq);
            for (int a = 0; a < 4; ++a) {
                int ia = i - 1 + a;
                if (ia < 0 || ia >= g->nx) continue;
                for (int b = 0; b < 4; ++b) {
                    int jb = j - 1 + b;
                    if (jb < 0 || jb >= nqk) continue;
                    acc += wx[a] * wq[b] * B[((long)ia * nqk + jb) * g->nflav + fcol];
                }
            }
            out[e] = acc;
        }
    }
    return 0;
}
