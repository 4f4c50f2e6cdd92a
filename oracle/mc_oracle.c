/*
 * mc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see mc_oracle.h).
 *
 * Plain CPU fp64 statements of the Monte Carlo steps that surround the PDF hot path in the thesis
 * (SURVEY.md section 8(f), rows NEXT-1, NEXT-2, NEXT-4), written from /root/reference/PAPER.md:
 *   RAMBO phase space          section 1.3.5, eq. 1.103-1.104, 1.107-1.110 (L1101-1180), p_T cut L2070
 *   VEGAS importance sampling  section 1.3.3, eq. 1.74-1.75, 1.80-1.83 (L866-876, L909-935)
 *   unweighting                section 4.1.3 (L2028-2030)
 * Every function follows the paper's steps in its order and notation; no blocking, no tables.
 * It shares no code with paper_2302_03343_b200/csrc/.
 */
#define _GNU_SOURCE
#include "mc_oracle.h"

#include <math.h>
#include <stdlib.h>

/* ------------------------------------------------------------------ */
/* RAMBO                                                                */
/* ------------------------------------------------------------------ */

/* eq. 1.108: w0 = (2 pi)^(4-3n) (pi/2)^(n-1) (P^2)^(n-2) / (Gamma(n) Gamma(n-1)) */
double oracle_rambo_w0(int n, double s)
{
    return pow(2.0 * M_PI, 4.0 - 3.0 * n) * pow(M_PI / 2.0, n - 1.0) * pow(s, n - 2.0) / (tgamma((double)n) * tgamma(n - 1.0));
}

/* xi of eq. 1.109: sqrt(P^2) = sum_i sqrt(m_i^2 + (xi p_i^0)^2), "usually solved numerically": Newton's
 * iteration from xi_0 = sqrt(1 - (sum m / sqrt s)^2), until the step is below 1e-15 xi (reading: the paper
 * names no solver; the root is unique since the sum is increasing in xi) */
static double solve_xi(int n, const double *E, const double *m, double rs)
{
    double sm = 0.0;
    for (int i = 0; i < n; ++i) sm += m[i];
    double xi = sqrt(1.0 - (sm / rs) * (sm / rs));
    for (int it = 0; it < 100; ++it) {
        double g = -rs, dg = 0.0;
        for (int i = 0; i < n; ++i) {
            double k0 = sqrt(m[i] * m[i] + xi * xi * E[i] * E[i]);
            g += k0;
            dg += xi * E[i] * E[i] / k0;
        }
        double step = g / dg;
        xi -= step;
        if (fabs(step) <= 1e-15 * xi) break;
    }
    return xi;
}

int oracle_rambo(long long nev, int n, const double *sqrt_s, const double *masses, const double *u, double ptmin,
                 double *p, double *w)
{
    if (nev < 0 || n < 2 || n > ORACLE_RAMBO_MAXN || !sqrt_s || !u || !p || !w) return -1;
    int massive = 0;
    if (masses) for (int i = 0; i < n; ++i) { if (masses[i] < 0.0) return -1; if (masses[i] > 0.0) massive = 1; }
#pragma omp parallel for schedule(static)
    for (long long e = 0; e < nev; ++e) {
        const double *ue = u + (size_t)e * n * 4;
        double *pe = p + (size_t)e * n * 4;
        double q[ORACLE_RAMBO_MAXN][4], Q[4] = {0, 0, 0, 0};
        /* step 1, eq. 1.107 */
        for (int i = 0; i < n; ++i) {
            double c = 2.0 * ue[4 * i] - 1.0, phi = 2.0 * M_PI * ue[4 * i + 1];
            double q0 = -log(ue[4 * i + 2] * ue[4 * i + 3]);
            double st = sqrt(1.0 - c * c);
            q[i][0] = q0; q[i][1] = q0 * st * cos(phi); q[i][2] = q0 * st * sin(phi); q[i][3] = q0 * c;
            for (int k = 0; k < 4; ++k) Q[k] += q[i][k];
        }
        /* step 2, eq. 1.103-1.104 with P = (sqrt s, 0, 0, 0) */
        double rs = sqrt_s[e], s = rs * rs;
        if (massive) {
            /* reading R-6: below the threshold sqrt s <= sum m_i the delta function of eq. 1.102 has no support:
             * Phi_n = 0, so the event carries weight 0 and zero momenta (the paper gives no case for it) */
            double sm = 0.0;
            for (int i = 0; i < n; ++i) sm += masses[i];
            if (!(rs > sm)) { for (int k = 0; k < 4 * n; ++k) pe[k] = 0.0; w[e] = 0.0; continue; }
        }
        double M = sqrt(Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3]);
        double b[3] = {-Q[1] / M, -Q[2] / M, -Q[3] / M};
        double gamma = Q[0] / M, a = 1.0 / (1.0 + gamma), x = rs / M;
        double E[ORACLE_RAMBO_MAXN];
        for (int i = 0; i < n; ++i) {
            double bq = b[0] * q[i][1] + b[1] * q[i][2] + b[2] * q[i][3];
            pe[4 * i] = x * (gamma * q[i][0] + bq);
            for (int k = 0; k < 3; ++k) pe[4 * i + 1 + k] = x * (q[i][1 + k] + b[k] * q[i][0] + a * bq * b[k]);
            E[i] = pe[4 * i];
        }
        /* step 3, eq. 1.108 */
        double wt = oracle_rambo_w0(n, s);
        if (massive) {
            /* eq. 1.109-1.110 (k_i^0 with xi^2 inside the root, as the constraint below eq. 1.109 has it) */
            double xi = solve_xi(n, E, masses, rs);
            double sk = 0.0, prod = 1.0, sk2 = 0.0;
            for (int i = 0; i < n; ++i) {
                double kabs = xi * E[i];                 /* |k_i| = xi |p_i| = xi p_i^0 (massless p_i) */
                double k0 = sqrt(masses[i] * masses[i] + kabs * kabs);
                pe[4 * i] = k0;
                for (int k = 1; k < 4; ++k) pe[4 * i + k] *= xi;
                sk += kabs; prod *= kabs / k0; sk2 += kabs * kabs / k0;
            }
            wt *= pow(s, 2.0 - n) * pow(sk, 2.0 * n - 3.0) * prod / sk2;
        }
        /* L2070: cut on the transverse momentum of the final-state particles */
        if (ptmin > 0.0)
            for (int i = 0; i < n; ++i)
                if (sqrt(pe[4 * i + 1] * pe[4 * i + 1] + pe[4 * i + 2] * pe[4 * i + 2]) < ptmin) wt = 0.0;
        w[e] = wt;
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* VEGAS                                                                */
/* ------------------------------------------------------------------ */

/* separable piecewise-constant p(x) = prod_d p_d(x_d) (eq. 1.81) on nb bins per dimension with edges
 * e[d][0..nb], every bin equally probable: u_d in [0,1) picks bin k = floor(u_d nb) and the point
 * x_d = e[d][k] + (u_d nb - k) (e[d][k+1] - e[d][k]); 1/p(x) = prod_d nb (e[d][k+1] - e[d][k]) */
int oracle_vegas_map(int ndim, int nb, const double *edges, long long n, const double *u, double *x, double *jac, int *bin)
{
    if (ndim < 1 || nb < 1 || n < 0 || !edges || !u || !x || !jac) return -1;
#pragma omp parallel for schedule(static)
    for (long long e = 0; e < n; ++e) {
        double j = 1.0;
        for (int d = 0; d < ndim; ++d) {
            double y = u[e * ndim + d] * nb;
            int k = (int)y;
            if (k > nb - 1) k = nb - 1;
            if (k < 0) k = 0;
            const double *ed = edges + (size_t)d * (nb + 1);
            double width = ed[k + 1] - ed[k];
            x[e * ndim + d] = ed[k] + (y - k) * width;
            j *= nb * width;
            if (bin) bin[e * ndim + d] = k;
        }
        jac[e] = j;
    }
    return 0;
}

/* eq. 1.74-1.75 sums: sums[0] = sum f/p, sums[1] = sum (f/p)^2; hist[d][k] = sum over the points of bin k
 * of dimension d of |f/p| (L913: "histogram of the absolute value of the integrand") */
int oracle_vegas_accumulate(int ndim, int nb, long long n, const double *f, const double *jac, const int *bin,
                            double *sums, double *hist)
{
    if (ndim < 1 || nb < 1 || n < 0 || !f || !jac || !sums) return -1;
    sums[0] = sums[1] = 0.0;
    if (hist) for (int k = 0; k < ndim * nb; ++k) hist[k] = 0.0;
    for (long long e = 0; e < n; ++e) {
        double fw = f[e] * jac[e];
        sums[0] += fw; sums[1] += fw * fw;
        if (hist && bin) for (int d = 0; d < ndim; ++d) hist[d * nb + bin[e * ndim + d]] += fabs(fw);
    }
    return 0;
}

/* E_N and the variance of E_N from the sums: eq. 1.74, and eq. 1.75 over N - 1 (eq. 1.65 / 1.66 reading: the
 * error of the estimate is S_N / sqrt(N), the unbiased sample variance over N) */
int oracle_vegas_estimate(long long n, const double *sums, double *E, double *var)
{
    if (n < 2 || !sums || !E || !var) return -1;
    double mean = sums[0] / n;
    *E = mean;
    *var = (sums[1] / n - mean * mean) / (n - 1);
    return 0;
}

/* grid refinement (L913: "the number of bins ... kept constant ..., gradually adjusting their width ... a finer
 * grid in regions providing large contributions"): the new edges cut the accumulated histogram, taken as
 * piecewise constant inside the old bins, in nb equal shares.  alpha damps the adaptation by raising the
 * normalised bin contents to the power alpha before cutting (alpha = 1: none) [alpha is not in the paper]. */
int oracle_vegas_refine(int ndim, int nb, const double *hist, double alpha, double *edges)
{
    if (ndim < 1 || nb < 1 || !hist || !edges) return -1;
    double *h = (double *)malloc(sizeof(double) * nb), *ne = (double *)malloc(sizeof(double) * (nb + 1));
    for (int d = 0; d < ndim; ++d) {
        double *ed = edges + (size_t)d * (nb + 1);
        double tot = 0.0;
        for (int k = 0; k < nb; ++k) tot += hist[d * nb + k];
        if (!(tot > 0.0)) continue;
        double tot2 = 0.0;
        for (int k = 0; k < nb; ++k) { h[k] = pow(hist[d * nb + k] / tot, alpha); tot2 += h[k]; }
        double share = tot2 / nb, acc = 0.0;
        int k = 0;
        ne[0] = ed[0]; ne[nb] = ed[nb];
        for (int j = 1; j < nb; ++j) {
            double target = share * j;
            while (k < nb - 1 && acc + h[k] < target) { acc += h[k]; ++k; }
            double frac = h[k] > 0.0 ? (target - acc) / h[k] : 0.0;
            if (frac > 1.0) frac = 1.0;
            ne[j] = ed[k] + frac * (ed[k + 1] - ed[k]);
        }
        for (int j = 0; j <= nb; ++j) ed[j] = ne[j];
    }
    free(h); free(ne);
    return 0;
}

/* eq. 1.82-1.83 */
int oracle_vegas_combine(int M, const double *E, const double *S2, double *Ebar, double *S2bar, double *chi2dof)
{
    if (M < 1 || !E || !S2 || !Ebar || !S2bar) return -1;
    double sw = 0.0, swe = 0.0;
    for (int i = 0; i < M; ++i) { sw += 1.0 / S2[i]; swe += E[i] / S2[i]; }
    *S2bar = 1.0 / sw;
    *Ebar = *S2bar * swe;
    if (chi2dof) {
        double c = 0.0;
        for (int i = 0; i < M; ++i) c += (E[i] - *Ebar) * (E[i] - *Ebar) / S2[i];
        *chi2dof = M > 1 ? c / (M - 1) : 0.0;
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* unweighting, L2028-2030                                              */
/* ------------------------------------------------------------------ */
int oracle_unweight(long long n, const double *w, const double *u, double *wmax_out, unsigned char *accept, long long *n_accept)
{
    if (n < 0 || !w || !u || !accept) return -1;
    double wmax = 0.0;
    for (long long e = 0; e < n; ++e) if (w[e] > wmax) wmax = w[e];      /* "the highest weight in the list" */
    long long cnt = 0;
    for (long long e = 0; e < n; ++e) { accept[e] = w[e] > u[e] * wmax ? 1 : 0; cnt += accept[e]; }
    if (wmax_out) *wmax_out = wmax;
    if (n_accept) *n_accept = cnt;
    return 0;
}
