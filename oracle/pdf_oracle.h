/*
 * pdf_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, CPU fp64 statement of what the hot path computes, written from
 * /root/reference/PAPER.md (M. Rossi, arXiv:2302.03343, section 3.2, lines
 * L1712-L1746 and section 3.3.2) in the reading fixed by
 * DESIGN.md ("Readings of the paper", items C-1 ... C-L, S-1 ... S-22).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  It shares no code, header,
 * table or helper with the CUDA path in paper_2302_03343_b200/csrc/.
 *
 * Parity status: every function below is pinned by tests/test_oracle_pins.py
 * against closed forms / invariants / a literal brute-force restatement,
 * EXCEPT the constants of the low-Q continuation (1 % step, floor -2.5,
 * guard 1e-5; C-9) and the fidelity of the knot-slope rule to LHAPDF 6
 * itself, which are "parity unpinned" (no LHAPDF and no PDF set exist in
 * this environment; PAPER.md prints no worked numeric example).
 *
 * All pointers are HOST pointers.  All functions return 0 on success and a
 * negative code on argument errors.
 */
#ifndef PDF_ORACLE_H
#define PDF_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle_grid oracle_grid;

/* region codes shared by oracle_locate and the product's pdf_locate (values
 * are part of both interfaces' documentation, not shared code) */
enum {
    ORACLE_REGION_INTERIOR = 0,
    ORACLE_REGION_LOWX = 1,
    ORACLE_REGION_LOWQ = 2,
    ORACLE_REGION_HIGHQ = 3,
    ORACLE_REGION_LOWX_LOWQ = 4,
    ORACLE_REGION_LOWX_HIGHQ = 5,
    ORACLE_REGION_INVALID = 6
};

/* alpha_s behaviour below the first knot (PAPER.md L1746 vs L1835, S-16) */
enum { ORACLE_ALPHAS_FREEZE = 0, ORACLE_ALPHAS_LOGGRAD = 1 };
/* the extrapolation choices of LHAPDF 6.  CONTINUATION is the default (C-7 ... C-9); FREEZE returns
 * "the PDF value at the closest grid knot", read (R-7) as the interpolant at the coordinates moved to the closest
 * point of the grid's range (a coordinate inside its range is not touched); ERROR "raises an error if a point outside
 * the grid range is queried": such a query is an invalid query (C-10: NaN, counted by the CUDA path). */
enum { ORACLE_EXTRAP_CONTINUATION = 0, ORACLE_EXTRAP_FREEZE = 1, ORACLE_EXTRAP_ERROR = 2 };

/* Grid format of PAPER.md L1714: knots in (x,Q2), Q2 split in sub-grids whose
 * last knot equals the first knot of the next one.  values is
 * [nmem][ sub-grid 0 block | sub-grid 1 block | ... ], block k being
 * [nx][nq[k]][nflav] row-major.  Arrays are copied. */
int oracle_grid_create(oracle_grid **g, int nx, const double *x_knots, int nsub,
                       const int *nq, const double *q2_knots,
                       const double *values, int nflav,
                       const int *flavour_pids, int nmem);
int oracle_grid_set_alphas(oracle_grid *g, int n, const double *q2_knots,
                           const double *values);
int oracle_grid_set_alphas_mode(oracle_grid *g, int mode);
int oracle_grid_set_coupling(oracle_grid *g, const double *C /*[nflav][nflav]*/);
int oracle_grid_limits(const oracle_grid *g, double *xmin, double *xmax,
                       double *q2min, double *q2max);
int oracle_grid_destroy(oracle_grid *g);
/* L1720; applies to oracle_locate, oracle_xfxq2 and oracle_lumi (whose 1/x1, 1/x2 keep the query's own x) */
int oracle_grid_set_extrapolation(oracle_grid *g, int mode);

/* C-2, C-3, C-4: region class, sub-grid, lower-left knot (ix, iq local to the
 * sub-grid).  For out-of-range queries the indices are those of the cell the
 * extrapolation is anchored on ("pdf_locate conventions"). */
int oracle_locate(const oracle_grid *g, long long n, const double *x,
                  const double *q2, int *ix, int *iq, int *isub, int *region);

/* C-5 ... C-11.  out is [n][npid] row-major; member may be NULL (member 0);
 * scale, if not NULL, receives [n][npid][2] condition numbers for the parity
 * metric C-12, tol = REL |ref| + FLOOR_S scale[0] + FLOOR_T scale[1]:
 *   scale[0] = sum |Wx_a Wq_b V_ab|  (what the rounding of the 16-term sum acts on),
 *   scale[1] = |df/dt_x| (1 + |ln x|/du) + |df/dt_q| (1 + |ln Q2|/ds)  (what the rounding of
 *              t = (ln v - ln knot)/delta acts on, in units of the relative rounding of a logarithm),
 * both propagated to first order through the extrapolation formulas.  Pinned by
 * tests/test_oracle_pins.py::test_scale_* against an independent restatement. */
int oracle_xfxq2(const oracle_grid *g, const int *pids, int npid, long long n,
                 const double *x, const double *q2, const int *member,
                 double *out, double *scale);

/* C-alpha */
int oracle_alphas_q2(const oracle_grid *g, long long n, const double *q2,
                     double *out);

/* C-L.  scale, if not NULL, receives [n][2]: for c = 0, 1
 *   scale[c] = |w| sum_ij |C_ij| (S1_i[c] |f2_j| + |f1_i| S2_j[c]),   S1 = scale of xf(x1)/x1, S2 of xf(x2)/x2:
 * the per-flavour condition numbers propagated to first order through the product. */
int oracle_lumi(const oracle_grid *g, long long n, const double *x1,
                const double *x2, const double *q2, const double *weights,
                double *out, double *scale);

/* Self-check helpers for the pins (P-10): the same interior value in three
 * evaluation orders.  order 0: x then Q (the oracle's own), 1: Q then x,
 * 2: 16-term tensor sum of node weights.  Interior queries only. */
int oracle_interior_order(const oracle_grid *g, int order, int flavour_col,
                          int member, long long n, const double *x,
                          const double *q2, double *out);

/* 1-D node weights (C-5) of a query on one knot line; exposes the 4-weight
 * form for the Catmull-Rom pin P-4.  w4 receives the weights of knots
 * c-1, c, c+1, c+2 (0 where the knot does not exist); *cell receives c. */
int oracle_weights_1d(int m, const double *knots_log, double wlog, int cell,
                      double w4[4]);

/* number of OpenMP threads the evaluation loops will use (1 if built without) */
int oracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
