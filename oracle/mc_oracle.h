/*
 * mc_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain CPU fp64 statements of the Monte Carlo steps around the PDF hot path (SURVEY.md 8(f) NEXT-1, NEXT-2,
 * NEXT-4), written from /root/reference/PAPER.md: RAMBO (eq. 1.103-1.110; p_T cut L2070), the VEGAS
 * importance-sampling step (eq. 1.74-1.75, 1.80-1.83, L866-935) and the unweighting rule (L2028-2030).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may load this library; it shares no
 * code with paper_2302_03343_b200/csrc/.  All pointers are HOST pointers; 0 on success, negative on bad arguments.
 *
 * Parity status: pinned by tests/test_mc_pins.py (momentum conservation, mass shells, the closed two- and
 * three-body volumes, the closed two-body massive weight, jacobian = bin volume, equal-share refinement on
 * closed histograms, eq. 1.82-1.83 on hand-worked numbers).  Readings (R-1 ... R-5): the
 * xi^2 inside the root of eq. 1.109; Newton's iteration for xi; |f|/p as the refinement histogram; the
 * variance of E_N as eq. 1.75 over N - 1; the damping exponent alpha (not in the paper; 1 = none).
 */
#ifndef MC_ORACLE_H
#define MC_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

#define ORACLE_RAMBO_MAXN 16

/* eq. 1.108 */
double oracle_rambo_w0(int n, double s);

/* n final-state momenta p[e][i][0..3] = (E, px, py, pz) in the frame P = (sqrt_s[e], 0, 0, 0) from the uniforms
 * u[e][i][0..3] (eq. 1.107, 1.103-1.104) and the weight w[e] (eq. 1.108; with masses != NULL and any m_i > 0 the
 * massive momenta of eq. 1.109 and w0 w_m of eq. 1.110); ptmin > 0: w[e] = 0 if any p_T < ptmin (L2070) */
int oracle_rambo(long long nev, int n, const double *sqrt_s, const double *masses, const double *u, double ptmin,
                 double *p, double *w);

/* eq. 1.81: uniforms u[n][ndim] through the bin edges edges[ndim][nb+1] -> x[n][ndim], jac[n] = 1/p(x), bin[n][ndim] */
int oracle_vegas_map(int ndim, int nb, const double *edges, long long n, const double *u, double *x, double *jac, int *bin);
/* sums[0] = sum f jac, sums[1] = sum (f jac)^2 (eq. 1.74-1.75); hist[ndim][nb] = per-bin sums of |f jac| (L913) */
int oracle_vegas_accumulate(int ndim, int nb, long long n, const double *f, const double *jac, const int *bin,
                            double *sums, double *hist);
/* E_N (eq. 1.74) and the variance of E_N (eq. 1.75 over N - 1) */
int oracle_vegas_estimate(long long n, const double *sums, double *E, double *var);
/* new edges: nb equal shares of the histogram (piecewise constant in the old bins), contents damped by alpha */
int oracle_vegas_refine(int ndim, int nb, const double *hist, double alpha, double *edges);
/* eq. 1.82-1.83 */
int oracle_vegas_combine(int M, const double *E, const double *S2, double *Ebar, double *S2bar, double *chi2dof);

/* L2028-2030: accept[e] = w[e] > u[e] * max w */
int oracle_unweight(long long n, const double *w, const double *u, double *wmax, unsigned char *accept, long long *n_accept);

#ifdef __cplusplus
}
#endif
#endif
