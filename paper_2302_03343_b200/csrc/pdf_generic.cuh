// pdf_generic.cuh -- layout kernels (a-1) and the DIRECT evaluation kernels: one thread per
// query, any nflav / pid list / member axis, stencil gathered through L1/L2.  These are the
// general-purpose path (PDF_PATH_DIRECT); the binned, warp-coherent path lives in pdf_binned.cuh.
#pragma once
#include "pdf_common.cuh"

namespace pdfg {

// ---- a-1: grid layout ------------------------------------------------------------------------
// ln of the knots with the path's own logarithm (so that t == 0 exactly on a knot), one thread per knot
__global__ void k_log_knots(const double *__restrict__ k, double *__restrict__ lk, int n)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) lk[i] = pdf_log(k[i]);
}

// per-cell Hermite constants of one knot line [first, first+m) (a sub-grid, the x line, alpha_s)
__global__ void k_cell_tables(const double *__restrict__ lk, CellTab *__restrict__ tab, int first, int m)
{
    int c = blockIdx.x * blockDim.x + threadIdx.x;      // local cell
    if (c >= m - 1) return;
    const double *w = lk + first;
    double d = w[c + 1] - w[c];
    CellTab t;
    t.lo_log = w[c];
    t.inv_d = 1.0 / d;
    bool left = c > 0, right = c + 2 < m;
    t.aL = left ? 0.5 : 1.0;
    t.bL = left ? 0.5 * (d / (w[c] - w[c - 1])) : 0.0;
    t.aR = right ? 0.5 : 1.0;
    t.bR = right ? 0.5 * (d / (w[c + 2] - w[c + 1])) : 0.0;
    tab[first + c] = t;
}

// values [mem][block k: [ix][iq][f]]  ->  V[mem][jg][ix][nfp] (pad columns = 0)
__global__ void k_relayout(const double *__restrict__ src, double *__restrict__ dst, int nx, int nqk,
                           int nflav, int nfp, int nqtot, int qoff_k, size_t src_memstride,
                           size_t src_suboff, int nmem)
{
    size_t per_mem = (size_t)nx * nqk * nfp;
    size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= per_mem * nmem) return;
    int mem = (int)(e / per_mem);
    size_t r = e % per_mem;
    int f = (int)(r % nfp);
    size_t node = r / nfp;
    int ix = (int)(node % nx);
    int iq = (int)(node / nx);
    double v = 0.0;
    if (f < nflav) v = src[(size_t)mem * src_memstride + src_suboff + ((size_t)ix * nqk + iq) * nflav + f];
    dst[(size_t)mem * ((size_t)nqtot * nx * nfp) + ((size_t)(qoff_k + iq) * nx + ix) * nfp + f] = v;
}

// ---- a-2: locate -----------------------------------------------------------------------------
__global__ void k_locate(GridDev G, long long n, const double *__restrict__ x, const double *__restrict__ q2,
                         int *ix, int *iq, int *isub, int *region)
{
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    double xv = x[e], qv = q2[e];
    apply_extrapolation(G, xv, qv);
    int r = classify(G, xv, qv);
    int i = -1, j = -1, k = -1;
    if (r != kRegionInvalid) {
        bool lowx = (r == kRegionLowX || r == kRegionLowXLowQ || r == kRegionLowXHighQ);
        i = lowx ? 0 : find_cell(G.xk, G.nx, xv);
        if (r == kRegionLowQ || r == kRegionLowXLowQ) { k = 0; j = 0; }
        else if (r == kRegionHighQ || r == kRegionLowXHighQ) { k = G.nsub - 1; j = G.qoff[k + 1] - G.qoff[k] - 2; }
        else { int jg; k = q_locate(G, qv, j, jg); }
    }
    if (ix) ix[e] = i;
    if (iq) iq[e] = j;
    if (isub) isub[e] = k;
    if (region) region[e] = r;
}

// ---- a-3 ... a-5, a-8: direct evaluation -----------------------------------------------------
// cols[p] = value column of requested pid p, or -1 (unknown pid -> 0.0)
struct ColMap { int n; int col[64]; };

__global__ void __launch_bounds__(128)
k_xfxq2_direct(GridDev G, ColMap cm, long long n, const double *__restrict__ x,
               const double *__restrict__ q2, const int *__restrict__ member,
               double *__restrict__ out, long long ld, int q_is_q)
{
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    double xv = x[e], qv = q2[e];
    if (q_is_q) qv = q_to_q2(qv);
    apply_extrapolation(G, xv, qv);
    int mem = member ? member[e] : 0;
    int r = classify(G, xv, qv);
    double *o = out + e * ld;
    if (r == kRegionInvalid || mem < 0 || mem >= G.nmem) {
        for (int p = 0; p < cm.n; ++p) o[p] = qnan();
        atomicAdd(G.err_count, 1ULL);
        return;
    }
    const double *Vm = G.V + (size_t)mem * G.memstride;
    QueryPlan P;
    make_plan(G, xv, qv, P);
    for (int p = 0; p < cm.n; ++p) {
        int c = cm.col[p];
        o[p] = c < 0 ? 0.0 : plan_value(G, Vm, P, c);
    }
}

// ---- NEXT-3: multi-member evaluation on one shared list of points (Table 3.3) ----
// out[(r * npts + p) * ld + k] = xf_{pids[k]}(member members[r]; x[p], q2[p]).  A thread owns one point:
// validity, search and the 2 x 4 node weights are done ONCE and reused for every member of its slice
// (blockIdx.y strides over the member list); the direct kernel repeats them per (point, member).
// For the 11-flavour layout (rows of 12 doubles) the stencil is read row-wise, 6 x LDG.128 per node, in
// the summation order of stencil_col (x-sum, then Q2-sum), so the rows are bit-identical to
// k_xfxq2_direct's.  Points are in increasing x in the paper's workload, so the lanes of a warp share
// cells and the loads coalesce to a few L1 wavefronts.  With contiguous rows (ld == npid == 11) a warp's
// 32 rows (requested columns = the 11 value columns in order) are transposed through shared memory and
// leave as 11 coalesced 256-byte stores (a lane writing its own row would touch 32 sectors per
// instruction).  Extrapolated points and other layouts take plan_value column by column.
// Measured (Table 3.3 shape, N_rep = 400): 0.092 ms against 0.169 ms for the direct kernel; what bounds it is
// the L1 request path (96 LDG.128 per (point, member), 4-5 distinct rows per warp instruction): large member
// lists go to k_xfxq2_xgrid_cell below, which reads a (member, cell) stencil once.
constexpr int kXgridThreads = 128;

// an extrapolated point of the 11-flavour layout: full plan, column by column (rare; kept out of line so
// that its registers do not weigh on the interior path)
__device__ __noinline__ void xgrid_slow_row(const GridDev &G, const double *Vm, double xv, double qv, double *dst)
{
    QueryPlan P;
    make_plan(G, xv, qv, P);
    for (int f = 0; f < 11; ++f) dst[f] = plan_value(G, Vm, P, f);
}

__global__ void __launch_bounds__(kXgridThreads, 4)
k_xfxq2_xgrid(const __grid_constant__ GridDev G, const __grid_constant__ ColMap cm, long long npts, const double *__restrict__ x, const double *__restrict__ q2,
              int nrep, const int *__restrict__ members, double *__restrict__ out, long long ld, int fast11, int coalesce)
{
    __shared__ double stage[kXgridThreads / 32][32 * 11];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long p = (long long)blockIdx.x * kXgridThreads + threadIdx.x;
    const long long p0 = p - lane;                             // first point of the warp
    const bool live = p < npts;
    double xv = 1.0, qv = 1.0;
    if (live) { xv = x[p]; qv = q2[p]; apply_extrapolation(G, xv, qv); }
    const bool valid = live && classify(G, xv, qv) != kRegionInvalid;
    // only the interior plan (2 x 4 node indices and weights) stays in registers across the member loop;
    // the rare extrapolated point rebuilds its full plan per member
    Point1D X0, Q0;
    bool interior = false;
    if (valid) {
        QueryPlan P;
        make_plan(G, xv, qv, P);
        interior = !P.X.low && !P.lowq && !P.Q.high;
        X0 = P.X.p0; Q0 = P.Q.p0;
    }
    const int rows_w = (int)((npts - p0) < 32 ? (npts - p0) : 32);   // rows of this warp (warp-uniform; <= 0: none)
    unsigned long long errs = 0;
    for (int r = blockIdx.y; r < nrep; r += gridDim.y) {
        const int mem = members ? __ldg(members + r) : r;
        const bool ok = valid && mem >= 0 && mem < G.nmem;
        if (fast11) {
            double *srow = &stage[warp][lane * 11];               // every row goes through shared memory
            // A member's rows are touched by this CTA only, once, so every stencil load would start a DRAM
            // round trip in the thread's critical path: the NEXT member's 16 rows are requested now (both ends
            // of a 96-byte row, which may straddle two lines), under this member's arithmetic.
            if (interior && r + (int)gridDim.y < nrep) {
                const int mn = members ? __ldg(members + r + gridDim.y) : r + (int)gridDim.y;
                if (mn >= 0 && mn < G.nmem) {
                    const double *Vn = G.V + (size_t)mn * G.memstride;
#pragma unroll
                    for (int b = 0; b < 4; ++b)
#pragma unroll
                        for (int a = 0; a < 4; ++a) {
                            const double *row = Vn + ((size_t)Q0.idx[b] * G.nx + X0.idx[a]) * 12;
                            asm volatile("prefetch.global.L1 [%0];" ::"l"(row));
                            asm volatile("prefetch.global.L1 [%0];" ::"l"(row + 11));
                        }
                }
            }
            __syncwarp();
            if (ok && interior) {
                const double *Vm = G.V + (size_t)mem * G.memstride;
                double acc[11];
#pragma unroll
                for (int f = 0; f < 11; ++f) acc[f] = 0.0;
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    double rb[11];
#pragma unroll
                    for (int f = 0; f < 11; ++f) rb[f] = 0.0;
                    const double *qrow = Vm + (size_t)Q0.idx[b] * G.nx * 12;
#pragma unroll
                    for (int a = 0; a < 4; ++a) {
                        const double2 *row = reinterpret_cast<const double2 *>(qrow + (size_t)X0.idx[a] * 12);
                        const double w = X0.w[a];
                        const double2 v0 = __ldg(row), v1 = __ldg(row + 1), v2 = __ldg(row + 2), v3 = __ldg(row + 3),
                                      v4 = __ldg(row + 4), v5 = __ldg(row + 5);
                        rb[0] = fma(w, v0.x, rb[0]); rb[1] = fma(w, v0.y, rb[1]);
                        rb[2] = fma(w, v1.x, rb[2]); rb[3] = fma(w, v1.y, rb[3]);
                        rb[4] = fma(w, v2.x, rb[4]); rb[5] = fma(w, v2.y, rb[5]);
                        rb[6] = fma(w, v3.x, rb[6]); rb[7] = fma(w, v3.y, rb[7]);
                        rb[8] = fma(w, v4.x, rb[8]); rb[9] = fma(w, v4.y, rb[9]);
                        rb[10] = fma(w, v5.x, rb[10]);
                    }
                    const double wq = Q0.w[b];
#pragma unroll
                    for (int f = 0; f < 11; ++f) acc[f] = fma(wq, rb[f], acc[f]);
                }
#pragma unroll
                for (int f = 0; f < 11; ++f) srow[f] = acc[f];
            } else if (ok) {
                xgrid_slow_row(G, G.V + (size_t)mem * G.memstride, xv, qv, srow);
            } else {
#pragma unroll
                for (int f = 0; f < 11; ++f) srow[f] = qnan();
                if (live) ++errs;
            }
            __syncwarp();
            double *o = out + ((long long)r * npts + p0) * ld;     // the warp's first row for this member
            if (coalesce) {
                const int tot = rows_w * 11;
#pragma unroll
                for (int k = 0; k < 11; ++k) {
                    const int e = k * 32 + lane;
                    if (e < tot) o[e] = stage[warp][e];
                }
            } else if (live) {
                double *orow = o + (long long)lane * ld;
                for (int k = 0; k < cm.n; ++k) {
                    const int c = cm.col[k];
                    orow[k] = !ok ? qnan() : (c < 0 ? 0.0 : srow[c]);      // an invalid row is NaN in every requested column
                }
            }
        } else if (live) {                                         // any other layout: column by column
            double *orow = out + ((long long)r * npts + p) * ld;
            if (ok) {
                const double *Vm = G.V + (size_t)mem * G.memstride;
                QueryPlan P;
                make_plan(G, xv, qv, P);
                for (int k = 0; k < cm.n; ++k) { const int c = cm.col[k]; orow[k] = c < 0 ? 0.0 : plan_value(G, Vm, P, c); }
            } else {
                for (int k = 0; k < cm.n; ++k) orow[k] = qnan();
                ++errs;
            }
        }
    }
    if (errs) atomicAdd(G.err_count, errs);
}

// The same call with the stencil of a (member, cell) read ONCE for all points of the cell.  A CTA takes a
// tile of kXcT consecutive points: their plans (2 x 4 node indices and weights, 96 B) go to shared memory and
// consecutive interior points with the same 16 nodes form a run (any order of points is correct; sorted x at
// one Q2, the paper's workload, gives runs of ~9-60 points).  Thread (g, j) serves member g of the CTA's
// current group of kXcMem members and flavour pair j (6 pairs = one 96-byte row per 6 threads): it holds
// V[16 nodes][2 flavours] of its member for the run in registers and walks the run's points with their
// weights broadcast from shared memory, in stencil_col's summation order (bit-identical rows).  The six
// threads of a member write one contiguous 88-byte row per point; consecutive points fill the sectors
// while the lines are still in L2.
constexpr int kXcT = 64, kXcThreads = 128, kXcMem = kXcThreads / 6;     // 21 members x 6 pairs = 126 threads
struct XcPoint { double wx[4], wq[4]; int xi[4], qi[4]; };

__global__ void __launch_bounds__(kXcThreads, 4)
k_xfxq2_xgrid_cell(const __grid_constant__ GridDev G, long long npts, const double *__restrict__ x,
                   const double *__restrict__ q2, int nrep, const int *__restrict__ members, double *__restrict__ out)
{
    __shared__ __align__(16) XcPoint sp[kXcT];
    __shared__ int s_kind[kXcT];               // 0 invalid, 1 interior, 2 extrapolated
    __shared__ int s_run[kXcT + 1];
    __shared__ int s_nrun;
    const long long p0 = (long long)blockIdx.x * kXcT;
    const int np = (int)((npts - p0) < kXcT ? (npts - p0) : kXcT);
    if ((int)threadIdx.x < np) {
        double xv = x[p0 + threadIdx.x], qv = q2[p0 + threadIdx.x];
        apply_extrapolation(G, xv, qv);
        int kind = 0;
        if (classify(G, xv, qv) != kRegionInvalid) {
            QueryPlan P;
            make_plan(G, xv, qv, P);
            kind = (!P.X.low && !P.lowq && !P.Q.high) ? 1 : 2;
            XcPoint &d = sp[threadIdx.x];
#pragma unroll
            for (int k = 0; k < 4; ++k) { d.wx[k] = P.X.p0.w[k]; d.wq[k] = P.Q.p0.w[k]; d.xi[k] = P.X.p0.idx[k]; d.qi[k] = P.Q.p0.idx[k]; }
        }
        s_kind[threadIdx.x] = kind;
    }
    __syncthreads();
    // runs: maximal stretches of interior points on the same 16 nodes.  Thread p flags whether point p opens a
    // run; the two warps that hold the tile's points ballot, and a flagged thread's rank among the flags is
    // its run number.
    {
        __shared__ unsigned s_ballot[2];
        bool fresh = false;
        const int p = threadIdx.x;
        if (p < np) {
            fresh = p == 0 || s_kind[p] != 1 || s_kind[p - 1] != 1;
            if (!fresh)
#pragma unroll
                for (int k = 0; k < 4; ++k) fresh |= sp[p].xi[k] != sp[p - 1].xi[k] || sp[p].qi[k] != sp[p - 1].qi[k];
        }
        if (p < kXcT) {
            const unsigned bal = __ballot_sync(0xffffffffu, fresh);
            if ((p & 31) == 0) s_ballot[p >> 5] = bal;
        }
        __syncthreads();
        const unsigned b0 = s_ballot[0], b1 = s_ballot[1];
        if (fresh) {
            const int idx = p < 32 ? __popc(b0 & ((1u << p) - 1u)) : __popc(b0) + __popc(b1 & ((1u << (p - 32)) - 1u));
            s_run[idx] = p;
        }
        if (p == 0) { const int n = __popc(b0) + __popc(b1); s_run[n] = np; s_nrun = n; }
    }
    __syncthreads();
    const int nrun = s_nrun;
    const int g = threadIdx.x / 6, j = threadIdx.x - 6 * g;
    unsigned long long errs = 0;
    if (g < kXcMem)
    for (int r = blockIdx.y * kXcMem + g; r < nrep; r += gridDim.y * kXcMem) {
        const int mem = members ? __ldg(members + r) : r;
        const bool okm = mem >= 0 && mem < G.nmem;
        const double *Vm = G.V + (size_t)(okm ? mem : 0) * G.memstride;
        double *orow0 = out + ((long long)r * npts + p0) * 11;
        for (int run = 0; run < nrun; ++run) {
            const int a0 = s_run[run], a1 = s_run[run + 1];
            const int kind = s_kind[a0];
            if (kind == 1 && okm) {
                double2 v[4][4];
#pragma unroll
                for (int b = 0; b < 4; ++b)
#pragma unroll
                    for (int a = 0; a < 4; ++a)
                        v[b][a] = __ldg(reinterpret_cast<const double2 *>(Vm + ((size_t)sp[a0].qi[b] * G.nx + sp[a0].xi[a]) * 12) + j);
                if (run + 1 < nrun && s_kind[s_run[run + 1]] == 1) {          // the next run's rows, under this run's arithmetic
                    const XcPoint &nx = sp[s_run[run + 1]];
#pragma unroll
                    for (int b = 0; b < 4; ++b)
#pragma unroll
                        for (int a = 0; a < 4; ++a) {
                            const double *row = Vm + ((size_t)nx.qi[b] * G.nx + nx.xi[a]) * 12 + 2 * j;
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(row));
                        }
                }
                // two points per step: their 2 x 10 dependent-FMA chains interleave (with one point per step the
                // loop waited on its own chains: profile r1k, 27 % "wait" at 3 warps per scheduler)
                auto point = [&](int p, double &acc0, double &acc1) {
                    const double2 wx01 = *reinterpret_cast<const double2 *>(&sp[p].wx[0]), wx23 = *reinterpret_cast<const double2 *>(&sp[p].wx[2]);
                    const double2 wq01 = *reinterpret_cast<const double2 *>(&sp[p].wq[0]), wq23 = *reinterpret_cast<const double2 *>(&sp[p].wq[2]);
                    const double wx[4] = {wx01.x, wx01.y, wx23.x, wx23.y}, wq[4] = {wq01.x, wq01.y, wq23.x, wq23.y};
                    acc0 = 0.0; acc1 = 0.0;
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        double rb0 = 0.0, rb1 = 0.0;
#pragma unroll
                        for (int a = 0; a < 4; ++a) { rb0 = fma(wx[a], v[b][a].x, rb0); rb1 = fma(wx[a], v[b][a].y, rb1); }
                        acc0 = fma(wq[b], rb0, acc0); acc1 = fma(wq[b], rb1, acc1);
                    }
                };
                double *o = orow0 + (long long)a0 * 11 + 2 * j;
                int p = a0;
#pragma unroll 1
                for (; p + 1 < a1; p += 2, o += 22) {
                    double c0, c1, d0, d1;
                    point(p, c0, c1);
                    point(p + 1, d0, d1);
                    o[0] = c0; o[11] = d0;
                    if (j < 5) { o[1] = c1; o[12] = d1; }
                }
                if (p < a1) {
                    double c0, c1;
                    point(p, c0, c1);
                    o[0] = c0;
                    if (j < 5) o[1] = c1;
                }
            } else if (kind == 1) {                                           // member id out of range: NaN rows
                for (int p = a0; p < a1; ++p) {
                    double *o = orow0 + (long long)p * 11 + 2 * j;
                    o[0] = qnan();
                    if (j < 5) o[1] = qnan();
                    if (j == 0) ++errs;
                }
            } else if (j == 0) {                                              // a single invalid or extrapolated point
                double *o = orow0 + (long long)a0 * 11;
                if (kind == 2 && okm) xgrid_slow_row(G, Vm, x[p0 + a0], q2[p0 + a0], o);
                else {
                    for (int f = 0; f < 11; ++f) o[f] = qnan();
                    ++errs;
                }
            }
        }
    }
    if (errs) atomicAdd(G.err_count, errs);
}

// ---- a-6: alpha_s ----------------------------------------------------------------------------
// Per cell the Hermite cubic of C-5 is kept in monomial form in t (built once by k_alphas_cells from
// the same cell constants the PDF path uses):  with H00 = A_c, H01 = A_{c+1},
//   H10 = -bL A_{c-1} + (bL - aL) A_c + aL A_{c+1},   H11 = -aR A_c + (aR - bR) A_{c+1} + bR A_{c+2},
//   alpha_s(t) = H00 h00 + H10 h10 + H01 h01 + H11 h11 = c0 + t (c1 + t (c2 + t c3)).
// alpha_s values are positive and smooth, so the monomial form loses nothing (1e-15 relative).
__global__ void k_alphas_cells(const CellTab *__restrict__ ca, const double *__restrict__ av, double *__restrict__ cell, int m)
{
    int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= m - 1) return;
    CellTab t = ca[c];
    double am = av[c > 0 ? c - 1 : c], a0 = av[c], a1 = av[c + 1], a2 = av[c + 2 < m ? c + 2 : c + 1];
    double H00 = a0, H01 = a1;
    double H10 = -t.bL * am + (t.bL - t.aL) * a0 + t.aL * a1;
    double H11 = -t.aR * a0 + (t.aR - t.bR) * a1 + t.bR * a2;
    double *o = cell + 6 * c;
    o[0] = t.lo_log; o[1] = t.inv_d;
    o[2] = H00; o[3] = H10;
    o[4] = -3.0 * H00 - 2.0 * H10 + 3.0 * H01 - H11;
    o[5] = 2.0 * H00 + H10 - 2.0 * H01 + H11;
}

constexpr int kAlphasIlp = 4;

// The cell comes from a table on the bit pattern of Q2 (exponent and top mantissa bits) and a walk on the raw
// knots (C-4, exact), so the search does not wait for the logarithm; ln Q2 is pdf_log (38 instructions).
__global__ void __launch_bounds__(256)
k_alphas(GridDev G, long long n, const double *__restrict__ q2, double *__restrict__ out)
{
    extern __shared__ __align__(16) double sm[];
    const int m = G.na;
    double *ak = sm;                               // [na] raw knots
    double *av = sm + m;                           // [na] values
    double *cell = sm + 2 * m;                     // [na-1][6]
    unsigned short *lut = reinterpret_cast<unsigned short *>(cell + 6 * (m - 1));
    for (int i = threadIdx.x; i < m; i += blockDim.x) { ak[i] = G.ak[i]; av[i] = G.av[i]; }
    for (int i = threadIdx.x; i < 6 * (m - 1); i += blockDim.x) cell[i] = G.acell[i];
    for (int i = threadIdx.x; i < G.nalut; i += blockDim.x) lut[i] = G.alut[i];
    __syncthreads();
    const double kmin = ak[0], kmax = ak[m - 1];
    const int shift = G.ashift, base = G.abase, nb = G.nalut;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long e0 = (long long)blockIdx.x * blockDim.x + threadIdx.x; e0 < n; e0 += stride * kAlphasIlp) {
        double q[kAlphasIlp], v[kAlphasIlp];
#pragma unroll
        for (int k = 0; k < kAlphasIlp; ++k) { long long e = e0 + k * stride; q[k] = e < n ? __ldcs(q2 + e) : 1.0; }
#pragma unroll
        for (int k = 0; k < kAlphasIlp; ++k) {
            const double qq = q[k];
            if (!finite_pos(qq)) { v[k] = qnan(); continue; }
            if (qq > kmax) { v[k] = av[m - 1]; continue; }                 // L1746: constant above the last knot
            if (qq < kmin) {      // L1835 constant (default) or L1746 logarithmic-gradient continuation
                v[k] = G.alphas_mode ? av[0] * pow(qq / kmin, log(av[1] / av[0]) / log(ak[1] / kmin)) : av[0];
                continue;
            }
            int b = (__double2hiint(qq) >> shift) - base;
            b = b < 0 ? 0 : (b >= nb ? nb - 1 : b);
            int c = lut[b];                                                // at the bucket's lower edge: never above the cell
            while (c < m - 2 && ak[c + 1] <= qq) ++c;                      // C-4 on the raw knots
            const double2 *cc = reinterpret_cast<const double2 *>(cell + 6 * c);
            const double2 c01 = cc[0], c23 = cc[1], c45 = cc[2];
            const double t = (pdf_log(qq) - c01.x) * c01.y;
            const double poly = fma(fma(fma(c45.y, t, c45.x), t, c23.y), t, c23.x);
            v[k] = (qq == ak[c + 1]) ? av[c + 1] : poly;                   // a knot returns its stored value
        }
#pragma unroll
        for (int k = 0; k < kAlphasIlp; ++k) { long long e = e0 + k * stride; if (e < n) __stcs(out + e, v[k]); }
    }
}

// the path's logarithm on an array (diagnostic: pdf_log_f64 of the C ABI, tested against the host's)
__global__ void k_log_f64(long long n, const double *__restrict__ x, double *__restrict__ out)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < n) out[e] = pdf_log(x[e]);
}

// ---- a-7: direct luminosity ------------------------------------------------------------------
__global__ void __launch_bounds__(128)
k_lumi_direct(GridDev G, long long n, const double *__restrict__ x1, const double *__restrict__ x2,
              const double *__restrict__ q2, const double *__restrict__ w, double *__restrict__ out)
{
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    const double a0 = x1[e], b0 = x2[e];
    double a = a0, b = b0, qa = q2[e], qb = qa;            // the points the partons are evaluated at (L1720); 1/x keeps the query's x
    apply_extrapolation(G, a, qa);
    apply_extrapolation(G, b, qb);
    if (classify(G, a, qa) == kRegionInvalid || classify(G, b, qb) == kRegionInvalid) {
        out[e] = qnan();
        atomicAdd(G.err_count, 1ULL);
        return;
    }
    double f2[kMaxLumiFlav];
    QueryPlan P;
    make_plan(G, b, qb, P);
    double inv_b = 1.0 / b0;
    for (int j = 0; j < G.nflav; ++j) f2[j] = plan_value(G, G.V, P, j) * inv_b;
    make_plan(G, a, qa, P);
    double inv_a = 1.0 / a0;
    double acc = 0.0;
    for (int i = 0; i < G.nflav; ++i) {
        double f1 = plan_value(G, G.V, P, i) * inv_a;
        double row = 0.0;
        for (int j = 0; j < G.nflav; ++j) row = fma(__ldg(G.C + i * G.nflav + j), f2[j], row);
        acc = fma(f1, row, acc);
    }
    out[e] = w[e] * acc;
}

// ---- fp64 peak micro-benchmark (denominator of the "alu" roofline) ----------------------------
__global__ void __launch_bounds__(256)
k_dfma_chain(double *sink, int iters, double a, double b)
{
    double r0 = threadIdx.x, r1 = r0 + 1, r2 = r0 + 2, r3 = r0 + 3, r4 = r0 + 4, r5 = r0 + 5, r6 = r0 + 6, r7 = r0 + 7;
    for (int i = 0; i < iters; ++i) {
        r0 = fma(r0, a, b); r1 = fma(r1, a, b); r2 = fma(r2, a, b); r3 = fma(r3, a, b);
        r4 = fma(r4, a, b); r5 = fma(r5, a, b); r6 = fma(r6, a, b); r7 = fma(r7, a, b);
    }
    double s = r0 + r1 + r2 + r3 + r4 + r5 + r6 + r7;
    if (s == 12345.678) sink[0] = s;
}

}  // namespace pdfg
