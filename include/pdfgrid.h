/*
 * pdfgrid.h -- C ABI of the B200-native (sm_100a) batched PDF interpolation library.
 *
 * What it computes (citations: /root/reference/PAPER.md = M. Rossi, arXiv:2302.03343):
 *   - xf_i(x,Q2) by LHAPDF-style log-bicubic interpolation: cubic Hermite splines in
 *     (log x, log Q2) on the 4 neighbour knots per axis (section 3.2, Fig. 3.1(a)),
 *     on knot grids split in Q2 sub-grids at quark-mass thresholds (L1714, L1833);
 *   - the default (MSTW / LHAPDF5) extrapolation outside the grid: low-x and high-Q linear
 *     continuation from the two outermost knots, of log(xf) when both values exceed 1e-3
 *     (L1720-1722); low-Q anomalous-dimension continuation eq. 3.4 with the limits of eq. 3.5
 *     (L1724-1742); corners: x rule first, then Q rule (L1744);
 *   - alpha_s(Q2): cubic Hermite spline on the log Q2 line, constant beyond the knots
 *     (L1746, L1835);
 *   - the two-parton luminosity  w * sum_ij C_ij f_i(x1,Q2) f_j(x2,Q2),  f = xf/x
 *     (eq. 3.3, eq. 4.1).
 * Readings of every point the paper leaves open are listed in DESIGN.md (C-1..C-L, S-1..S-22).
 *
 * Conventions
 *   - Every function returns an int status: PDF_OK (0) or a negative code; nothing throws.
 *   - HOST / DEVICE says where a pointer must live.  `stream` is a cudaStream_t passed as void*
 *     (NULL = the legacy default stream).  Evaluation calls only ENQUEUE work on `stream` and
 *     return; they never synchronise.  HOST arrays (pids, knots, values) are consumed before the
 *     call returns.
 *   - Ownership: pdf_grid_create copies its host arrays into device tables owned by the handle;
 *     query / output / workspace buffers are caller-owned (e.g. torch tensors, data_ptr()).
 *     The library allocates device memory only in pdf_grid_create / set_* and, for the *_host
 *     convenience calls, a staging area kept in the handle.
 *   - q2 is Q^2 in GeV^2; outputs are x*f (L1712 "always in the xf(x,Q2) format").
 *   - Per-query domain errors (x <= 0, x > xmax, Q2 <= 0, non-finite, member out of range) write
 *     quiet NaN to every requested column of that row and increment a device counter that
 *     pdf_error_count reads.
 *   - A requested pid that is not in the grid's flavour list yields a column of 0.0; pid 0 is
 *     an alias of 21 (gluon).
 */
#ifndef PDFGRID_H
#define PDFGRID_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    PDF_OK = 0,
    PDF_EINVAL = -1,     /* bad argument (NULL, size, non-monotonic knots, non-finite value ...) */
    PDF_ENOMEM = -2,     /* host or device allocation failed                                     */
    PDF_ECUDA = -3,      /* a CUDA runtime call failed (see pdf_last_cuda_error)                 */
    PDF_EWORKSPACE = -4, /* the binned path needs a workspace and none / too small was supplied  */
    PDF_ESTATE = -5,     /* call needs data that was not set (alpha_s knots, coupling matrix)    */
    PDF_ELIMIT = -6      /* pdf_xfxq2_noalloc: n (or the grid) beyond what its static scratch holds */
};

/* region codes written by pdf_locate (Fig. 3.1(b)) */
enum {
    PDF_REGION_INTERIOR = 0,
    PDF_REGION_LOWX = 1,
    PDF_REGION_LOWQ = 2,
    PDF_REGION_HIGHQ = 3,
    PDF_REGION_LOWX_LOWQ = 4,
    PDF_REGION_LOWX_HIGHQ = 5,
    PDF_REGION_INVALID = 6
};

/* alpha_s below its first knot: PDFFlow's constant (L1835, default) or LHAPDF's logarithmic
 * gradient continuation (L1746) */
enum { PDF_ALPHAS_FREEZE = 0, PDF_ALPHAS_LOGGRAD = 1 };

/* evaluation strategy of pdf_xfxq2 / pdf_lumi (pdf_grid_set_option(PDF_OPT_PATH, ...)) */
enum {
    PDF_PATH_AUTO = 0,    /* binned when a workspace is attached and the call qualifies, else direct */
    PDF_PATH_DIRECT = 1,  /* one thread per query, stencil gathered through L1/L2; pdf_lumi: one fused
                             kernel, the per-flavour values never leave the registers               */
    PDF_PATH_BINNED = 2   /* queries binned by cell so that warps share one stencil (needs workspace;
                             11-flavour grids); with a member array the queries are first partitioned
                             by member (<= 4096 members, npid <= nflav); pdf_lumi: sliced binned
                             evaluation of both partons into workspace scratch + a combine kernel     */
};
enum { PDF_OPT_PATH = 1, PDF_OPT_ALPHAS_MODE = 2, PDF_OPT_CHUNK = 3, PDF_OPT_EXTRAPOLATION = 4 };

/* extrapolation outside the grid's range (pdf_grid_set_option(PDF_OPT_EXTRAPOLATION, ...)):
 * CONTINUATION is LHAPDF's default (low-x / high-Q continuation L1722, low-Q rule eq. 3.4-3.5); FREEZE "freezes the
 * grid edges, returning the PDF value at the closest grid knot": the interpolant at the query moved to the closest
 * point of the range (a coordinate inside its range is not touched); ERROR "raises an error if a point outside the
 * grid range is queried": such a query gives a NaN row and counts in pdf_error_count, like any invalid query.
 * The option acts on pdf_xfxq2 / _ex / _xgrid / _noalloc, pdf_xfxq, pdf_lumi (whose factors 1/x1, 1/x2 keep the
 * query's own x) and pdf_locate (which reports the cell of the point that is evaluated). */
enum { PDF_EXTRAP_CONTINUATION = 0, PDF_EXTRAP_FREEZE = 1, PDF_EXTRAP_ERROR = 2 };

typedef struct pdf_grid pdf_grid; /* opaque; owns its device tables */

/* ---- grid handle (a-1: grid layout; L1714, L1833) -------------------------------------------
 * x_knots   HOST [nx], strictly increasing, > 0, nx >= 2.
 * nq        HOST [nsub], every nq[k] >= 2.
 * q2_knots  HOST, the sub-grids' knots concatenated ([sum nq]); strictly increasing inside a
 *           sub-grid; last knot of sub-grid k == first knot of sub-grid k+1 (bitwise).
 * values    HOST [nmem][ block 0 | block 1 | ... ], block k = [nx][nq[k]][nflav] row-major,
 *           all finite.  values are x*f at the knots.
 * flavour_pids HOST [nflav] PDG ids of the value columns.
 * The device currently selected (cudaGetDevice) becomes the grid's device.
 * Errors: PDF_EINVAL on any violated condition, PDF_ENOMEM / PDF_ECUDA on allocation failure. */
int pdf_grid_create(pdf_grid **g, int nx, const double *x_knots, int nsub, const int *nq,
                    const double *q2_knots, const double *values, int nflav,
                    const int *flavour_pids, int nmem);
int pdf_grid_destroy(pdf_grid *g);

/* alpha_s knots (HOST [n], Q2 > 0 increasing, n >= 2) and values (HOST [n]); L1746.  A knot may appear twice (not at
 * the ends, not three times): a flavour threshold, the end of one sub-line and the start of the next with its own value
 * on either side (L1835 "the sub-grids mechanism ... flavor thresholds"); the Hermite cubic then uses one-sided slopes
 * at the ends of every sub-line and a query on a threshold belongs to the upper sub-line. */
int pdf_grid_set_alphas(pdf_grid *g, int n, const double *q2_knots, const double *values);
/* flavour-pair coupling C, HOST [nflav][nflav] row-major, in the grid's column order; eq. 4.1 */
int pdf_grid_set_coupling(pdf_grid *g, const double *C);
/* caller-owned DEVICE scratch for the binned path; must stay valid until replaced or the grid is
 * destroyed; bytes >= pdf_workspace_bytes(g, n) for the largest n it will be used with (the
 * figure grows by the luminosity scratch (176 bytes per event, up to 2^24 events) once a coupling
 * has been set, so query it after pdf_grid_set_coupling; for a grid with nmem > 1 it includes the member-partition scratch,
 * 108 bytes per query up to 2^25 queries).  The contents are scratch: one evaluation call at a time may use it.
 * dev_ptr == NULL detaches. */
int pdf_grid_set_workspace(pdf_grid *g, void *dev_ptr, size_t bytes);
size_t pdf_workspace_bytes(const pdf_grid *g, long long n);
int pdf_grid_set_option(pdf_grid *g, int option, long long value);
/* xMin/xMax/Q2Min/Q2Max of L1714; any output pointer may be NULL */
int pdf_grid_limits(const pdf_grid *g, double *xmin, double *xmax, double *q2min, double *q2max);

/* ---- evaluation (a-2 ... a-5, a-8) ----------------------------------------------------------
 * pids HOST [npid]; x, q2 DEVICE [n]; out DEVICE [n][npid] row-major (leading dimension npid).
 * n == 0 is a no-op.  Enqueues on `stream`. */
int pdf_xfxq2(const pdf_grid *g, const int *pids, int npid, long long n, const double *x,
              const double *q2, double *out, void *stream);
/* as above with a per-query member index (DEVICE int32 [n] or NULL = member 0) and an explicit
 * leading dimension ld_out >= npid (in doubles). */
int pdf_xfxq2_ex(const pdf_grid *g, const int *pids, int npid, long long n, const double *x,
                 const double *q2, const int *member, double *out, long long ld_out, void *stream);

/* NEXT-3, multi-member evaluation on one shared list of points ("load multiple members of
 * a PDF set at once ... PDFs evaluated in a grid of x points"; the workload of Table 3.3):
 *   out[(r * npts + p) * ld_out + k] = xf_{pids[k]}(member members[r]; x[p], q2[p]),  r < nrep, p < npts.
 * pids HOST [npid]; x, q2 DEVICE [npts]; members DEVICE int32 [nrep] or NULL (= 0 .. nrep-1); out DEVICE
 * [nrep][npts][ld_out], ld_out >= npid; caller-owned, nothing is allocated.  Same values as pdf_xfxq2_ex
 * on the member-major expansion of the points (bit-identical to its direct path); validity, cell search
 * and node weights are computed once per point.  A point outside the domain, or a member id outside
 * [0, nmem), gives a quiet-NaN row and one error count per (point, member).  npts == 0 or nrep == 0 is a
 * no-op.  Enqueues one kernel on `stream`; PDF_EINVAL on bad arguments. */
/* xfxQ ("PDF::xfxQ(...) and PDF::xfxQ2(...)"): pdf_xfxq2 at Q2 = Q * Q; q DEVICE [n] holds Q in GeV.
 * Q <= 0 or non-finite is an invalid query (NaN row, counted) although its square is not. */
int pdf_xfxq(const pdf_grid *g, const int *pids, int npid, long long n, const double *x,
             const double *q, double *out, void *stream);

int pdf_xfxq2_xgrid(const pdf_grid *g, const int *pids, int npid, long long npts, const double *x,
                    const double *q2, int nrep, const int *members, double *out, long long ld_out,
                    void *stream);

/* a-6: alpha_s(Q2); q2, out DEVICE [n].  PDF_ESTATE if no alpha_s knots were set. */
int pdf_alphas_q2(const pdf_grid *g, long long n, const double *q2, double *out, void *stream);

/* a-7: out[e] = weights[e] * sum_ij C_ij [xf_i(x1,q2)/x1] [xf_j(x2,q2)/x2] over the grid's own
 * flavour columns (member 0); all arrays DEVICE [n].  PDF_ESTATE if no coupling was set. */
int pdf_lumi(const pdf_grid *g, long long n, const double *x1, const double *x2, const double *q2,
             const double *weights, double *out, void *stream);

/* a-2 exposed for validation (L1714-1720, L1735): region class, sub-grid, lower-left knot of the cell (ix,
 * and iq local to the sub-grid); DEVICE int32 [n] each, any may be NULL.  For extrapolated queries the
 * indices are those of the knots the continuation is anchored on (low-x: ix = 0; low-Q:
 * isub = 0, iq = 0; high-Q: last sub-grid, iq = nq-2); invalid queries get -1.
 * The call runs the search of the evaluation path that is selected: under PDF_PATH_AUTO / PDF_PATH_BINNED
 * (and a grid the binned path supports) the table-driven search of the binned kernel's A tiles
 * (s3_locate, the function k_pdf_stream calls), under PDF_PATH_DIRECT the binary search of the direct
 * kernels.  Both compare raw values only, so both must equal the oracle bit for bit. */
int pdf_locate(const pdf_grid *g, long long n, const double *x, const double *q2, int *ix,
               int *iq, int *isub, int *region, void *stream);

/* which path the last evaluation call (pdf_xfxq2 / _ex / pdf_lumi / pdf_locate) on this handle ran:
 * PDF_PATH_DIRECT or PDF_PATH_BINNED (0 before the first call).  PDF_PATH_AUTO falls back to the direct
 * kernels for grids the binned path does not support (flavour count other than 11, > 1024 cells per axis),
 * small calls and calls without a sufficient workspace; this call makes that visible. */
int pdf_last_path(const pdf_grid *g);

/* ---- the no-allocation entry point ------------------------------------------------------------
 * pdf_xfxq2 (same operation, same results: PAPER.md L1712-1746) for callers that may not
 * allocate device memory -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
 * It runs the binned path's kernel with its scratch in a static device array of PDF_NOALLOC_SCRATCH_BYTES that every
 * GPU which loads the library holds until the process exits; no workspace is attached or used, and the call makes no
 * cudaMalloc / cudaFree and calls no allocating routine (one memset and one launch on `stream`).
 *   pids HOST [npid]; x, q2 DEVICE [n]; out DEVICE [n][npid] row-major (ld = npid).
 *   max_n: HOST, optional; receives the largest n this grid's geometry allows (also when the call is rejected):
 *          the whole call is one chunk in one ring slot, ~290 B of scratch per query plus 32 B x 32 per grid cell
 *          (about 1.8e5 queries for a 196 x 54-knot grid).
 * Errors: PDF_ELIMIT when n > *max_n, or when the grid does not fit the binned path (flavour count other than 11,
 * > 1024 cells per axis) or the array at all; PDF_EINVAL on bad arguments; PDF_ECUDA if the array's address could
 * not be resolved when the grid was created.  Invalid queries give NaN rows and count in pdf_error_count as usual.
 * The array is shared by every call on a device and keeps the last call's contents (the call clears the counters it
 * needs at zero, on `stream`): calls that overlap on the GPU -- different streams, or two grids on one device --
 * race on it, so order them on one stream or with events. */
#define PDF_NOALLOC_SCRATCH_BYTES (64u * 1024u * 1024u)
int pdf_xfxq2_noalloc(const pdf_grid *g, const int *pids, int npid, long long n, const double *x, const double *q2,
                      double *out, long long *max_n, void *stream);

/* number of invalid queries seen by this grid since creation / the last call of this function
 * (reads and resets the device counter; synchronises `stream`). */
int pdf_error_count(const pdf_grid *g, long long *n_invalid, void *stream);

/* ---- host-buffer convenience calls (the e2e path) -------------------------------------------
 * Same results as the calls above, but x, q2, out (x1, x2, weights) are HOST pointers, pinned
 * memory recommended.  The call copies inputs to the device in chunks, evaluates, copies the
 * results back, overlapping the three on internal streams, and returns when `out` is complete. */
int pdf_xfxq2_host(pdf_grid *g, const int *pids, int npid, long long n, const double *x,
                   const double *q2, double *out);
int pdf_alphas_q2_host(pdf_grid *g, long long n, const double *q2, double *out);
int pdf_lumi_host(pdf_grid *g, long long n, const double *x1, const double *x2, const double *q2,
                  const double *weights, double *out);

/* ---- diagnostics ---------------------------------------------------------------------------- */
const char *pdf_status_string(int status);
const char *pdf_last_cuda_error(void);
/* kernels launched by this library in this process since load (the bench's gpu_launches) */
long long pdf_launch_count(void);
/* name and launch time (ms, CUDA events on `stream`) of the kernels of the last evaluation call
 * when profiling was switched on with pdf_profile_enable(1); returns the number of entries. */
int pdf_profile_enable(int on);
int pdf_profile_read(int max_entries, const char **names, float *ms);
/* sustained fp64 FMA throughput of the device (an independent-DFMA-chain kernel), in TFLOP/s;
 * the measured denominator of the "alu" roofline of pdf_lumi. */
int pdf_measure_fp64_tflops(double *tflops, void *stream);

/* diagnostic: out[i] = the logarithm the path computes its abscissae with (t = (ln v - ln knot)/delta, L1716), for
 * finite x[i] > 0; DEVICE [n] each.  Tested against the host's log (<= 1 ulp). */
int pdf_log_f64(long long n, const double *x, double *out, void *stream);

/* ---- Monte Carlo steps around the hot path -----------------------------
 * All array arguments are DEVICE pointers unless marked HOST; calls enqueue on `stream`.  Random numbers are
 * inputs (uniforms in [0, 1)): the library draws none. */

/* RAMBO (section 1.3.5, eq. 1.103-1.104, 1.107-1.110, L1101-1180): npart (2..16) final-state momenta
 * p[nev][npart][4] = (E, px, py, pz) in the frame P = (sqrt_s[e], 0, 0, 0) from the uniforms u[nev][npart][4], and the
 * weight w[nev]: eq. 1.108 for massless particles (masses == NULL or all 0; HOST [npart]), w0 w_m of eq. 1.110 with
 * the momenta of eq. 1.109 (xi by Newton's iteration on its energy constraint) otherwise.  ptmin > 0 sets w = 0
 * for events with a final-state p_T below it (L2070); the momenta are written either way. */
int pdf_rambo(long long nev, int npart, const double *sqrt_s, const double *masses, const double *u, double ptmin,
              double *p, double *w, void *stream);

/* VEGAS importance sampling (section 1.3.3): a separable density p(x) = prod_d p_d(x_d) (eq. 1.81), piecewise
 * constant on nbins equally probable bins per dimension with edges[ndim][nbins + 1].
 * pdf_vegas_map: u[n][ndim] -> x[n][ndim], jac[n] = 1/p(x) = prod_d nbins * width, bin[n][ndim] (may be NULL).
 * pdf_vegas_accumulate: sums[0] = sum f jac, sums[1] = sum (f jac)^2 (eq. 1.74-1.75), hist[ndim][nbins] = per-bin sums
 *   of |f jac| (L913; may be NULL); both are zeroed first.  Across GPUs these are the only numbers to all-reduce.
 * pdf_vegas_estimate: res[0] = E_N (eq. 1.74), res[1] = variance of E_N (eq. 1.75 over N - 1).
 * pdf_vegas_refine: new edges = nbins equal shares of the histogram, taken piecewise constant in the old bins and
 *   damped by the exponent alpha (1 = none; not in the paper); scratch is DEVICE [ndim][2 nbins + 1] doubles.
 * pdf_vegas_combine: res = {Ebar, S2bar, chi2/dof} of M iterations (eq. 1.82-1.83); E, S2 DEVICE [M]. */
int pdf_vegas_map(int ndim, int nbins, const double *edges, long long n, const double *u, double *x, double *jac,
                  int *bin, void *stream);
int pdf_vegas_accumulate(int ndim, int nbins, long long n, const double *f, const double *jac, const int *bin,
                         double *sums, double *hist, void *stream);
int pdf_vegas_estimate(long long n, const double *sums, double *res, void *stream);
int pdf_vegas_refine(int ndim, int nbins, const double *hist, double alpha, double *edges, double *scratch, void *stream);
int pdf_vegas_combine(int M, const double *E, const double *S2, double *res, void *stream);

/* unweighting (section 4.1.3): accept[e] = w[e] > u[e] * max_e w[e] (uint8).  scratch16 is 16 DEVICE
 * bytes; wmax and n_accept (HOST, may be NULL) are read back after a stream synchronise when given. */
int pdf_unweight(long long n, const double *w, const double *u, unsigned char *accept, void *scratch16,
                 double *wmax, long long *n_accept, void *stream);

#ifdef __cplusplus
}
#endif
#endif
