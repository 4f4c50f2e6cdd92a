// pdf_stream.cuh -- the binned, cell-coherent evaluation path (PDF_PATH_BINNED), version 3:
// one persistent kernel of independent WARPS, bins per CELL, no CTA barrier on the path.
//
// Why binning at all: a query needs a 4 x 4 stencil x 11 flavours = 1408 B of grid
// data; gathered per lane that is >= 12 clk/query/SM of L1 / shared-memory bandwidth against a
// budget of 7.9 clk/query/SM at 60 % of the HBM roofline.  Queries that share a cell take the
// cell's 16 x 11 values ONCE, as operand fragments of FP64 mma.sync tiles.  With ~10^4 cells that
// needs a sort domain of ~3 x 10^5 queries: they are binned through L2 in chunks.
//
// What changed against version 2 (one coarse bin per x cell, tile-local counting sorts in shared
// memory in A, payload staging + counting sort by Q2 cell in B, 46 warp instructions per query, 16
// warps/SM, profiles/r1i, r1j): the bin IS the cell.
//   A tile (one warp, 256 queries): coalesced loads of x, Q2; validity / region class on the bit
//     patterns; cell search from a table indexed by the exponent and top mantissa bits (integer
//     compares on the raw knots: C-3 / C-4 bit-exact, FP64 pipe untouched); t_x, t_q (two logs);
//     ONE global atomic per query reserves a slot in the cell's bin, the 32-byte payload
//     {a, b, idx} is stored as one whole sector.  The tile's output rows are zero-filled with
//     coalesced 32-byte stores first, so that the scattered 88-byte rows of B merge into valid
//     L2-resident sectors (scattered partial-sector stores into untouched
//     memory run at 0.9 TB/s).  No shared-memory sort, no barrier.
//   B unit (one warp, 8 consecutive Q2 cells of one x cell): reads the 8 counts, then per cell the
//     16 x 11 values as 8 fragment registers per lane (L1/L2), its payloads in batches of 32
//     through a double-buffered cp.async stage, and runs DMMA m8n8k4 tiles of 8 queries x 8
//     flavours; rows leave from the accumulator fragments.  No staging of grid columns, no
//     counting sort, no batch descriptors.
//   Extrapolation classes (a-5) are bins of their own ((x cell, low-Q), (x cell, high-Q), (low-x,
//   Q2 cell), two corners) and run the same DMMA contraction with class-specific node sets and
//   weights, followed by the per-flavour continuation formulas (C-7 ... C-9) on the fragments.
// Work is handed out per warp by a global ticket counter in the order
//      round r = [ A(r) tiles | B(r - kLag) units ],
// B(c) waits until every A tile of chunk c has been released, A(c) until B(c - kRing) has drained
// the ring slot; a ticket only ever waits on lower tickets and every CTA is resident, so the
// scheme cannot deadlock.  Queries beyond a bin's capacity go to an overflow list evaluated by the
// generic per-thread code: correctness never depends on the distribution of the queries.
#pragma once
#include "pdf_common.cuh"
#include "pdf_generic.cuh"

namespace pdfg {

#ifndef PDF_S3_THREADS
#define PDF_S3_THREADS 256
#endif
#ifndef PDF_S3_MINB
#define PDF_S3_MINB 3
#endif
#ifndef PDF_S3_LAG
#define PDF_S3_LAG 1
#endif
#ifndef PDF_S3_RING
#define PDF_S3_RING 3
#endif
#ifndef PDF_S3_GRP
#define PDF_S3_GRP 4
#endif
constexpr int kS3Threads = PDF_S3_THREADS;          // CTA size of the persistent kernel; every warp works alone
constexpr int kS3Warps = kS3Threads / 32;
constexpr int kS3TileQ = 8;                          // queries per lane in an A tile
constexpr int kS3TileA = 32 * kS3TileQ;              // 256 queries per A tile (one warp)
constexpr int kS3Grp = PDF_S3_GRP;                   // queries of a lane that go through the A steps together
static_assert(kS3TileQ % kS3Grp == 0, "kS3TileQ must be a multiple of kS3Grp");
constexpr int kS3Batch = 32;                         // payloads per cp.async stage
constexpr int kS3FkPerUnit = 8;                      // fine keys (Q2 cells) per B unit
constexpr int kS3ClassParts = 2;                     // B units per x key that share its two extrapolation-class bins (low-Q, high-Q)
constexpr int kS3Ovf = 8;                            // B units per chunk that drain the overflow list
constexpr int kS3Lag = PDF_S3_LAG;                   // B(c) tickets follow A(c) tickets by this many rounds
constexpr int kS3Ring = PDF_S3_RING;                 // chunk slots in flight
static_assert(kS3Ring >= kS3Lag + 2, "A(c) must find the slot of B(c - kRing) drained");
constexpr int kS3LutMax = 2048;                      // search-table buckets per axis
constexpr int kNF = 11, kNFP = 12;                   // the path is specialised for 11 flavours (rows padded to 12)
constexpr int kS3MaxCells = 1024;                    // x cells / Q2 knots the path supports (u16 tables, 32-bit payload offsets)

struct __align__(32) Payload {                       // one sector
    double a, b;                                     // class-dependent abscissae (t_x, t_q / theta / r)
    unsigned idx, pad0;                              // query index inside its chunk
    double pad1;
};

// geometry of the key space and the search tables; host copy in StreamPlan, passed by value
struct StreamDev {
    int ncx, nqt, nfk, nbins;                        // x cells, Q2 knots, fine keys per x key (nqt + 2), bins ((ncx + 1) * nfk)
    int jgplus;                                      // cell (global lower-knot index) of 1.01*Q2min
    double tqplus;                                   // and its t_q  (C-9)
    int cap_int, cap_cls, cap_lx, cap_lxc;           // bin capacities: interior cell, (x cell, class), (low-x, Q2 cell), corner
    int rowcap, lxbase, slab;                        // payloads per x key, offset of the low-x key, payloads per ring slot
    int ng, tb;                                      // fine-key groups per x key, B units per chunk
    int xshift, xbase, nbx, qshift, qbase, nbq;      // bucket = (high word >> shift) - base
    const unsigned short *lutx, *lutq;               // [nbx], [nbq] cell at the lower edge of the bucket
    const double2 *cxs, *cqs;                        // [ncx], [nqt] {ln lower knot, 1/dln} per cell
};

struct StreamWorkspace {                             // carved out of the caller's workspace
    unsigned long long *ctrl;                        // [0] ticket; then per ring slot a_done, b_fin, b_done, each on a 128-byte line of its own
    unsigned *counts;                                // [kS3Ring][nbins]
    unsigned *ovf_count;                             // [kS3Ring]
    Payload *bins;                                   // [kS3Ring][slab]
    Payload *ovf;                                    // [kS3Ring][chunk]  (raw x, q2)
};

struct StreamArgs {
    GridDev G;
    StreamDev B;
    ColMap cm;
    StreamWorkspace W;
    const double *x, *q2;
    double *out;
    long long n, ld;
    long long chunk;           // queries per chunk (multiple of kS3TileA)
    int nchunks, ta;           // chunks, A tiles per chunk
    int identity;              // 1: requested columns == the grid's 11 columns in order
    int zfill;                 // 1: rows are contiguous (ld == npid): A tiles zero-fill their rows of `out`
    int count_err;             // 1: invalid queries bump the grid's error counter
    // member axis (a-8, pdf_members.cuh): the queries arrive sorted by member and every chunk lies
    // inside one member's run; ctab[c] = {first query, queries, member, 0}, *nchunks_dev chunks.
    const int *ctab;
    const int *nchunks_dev;
};

// ---- small device helpers ----------------------------------------------------------------------
// explicit shared-window accessors (32-bit addresses)
__device__ __forceinline__ double lds_f64(unsigned a) { double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a)); return v; }
__device__ __forceinline__ long long lds_s64(unsigned a) { long long v; asm volatile("ld.shared.s64 %0, [%1];" : "=l"(v) : "r"(a)); return v; }
__device__ __forceinline__ unsigned lds_u32(unsigned a) { unsigned v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ unsigned lds_u16(unsigned a) { unsigned short v; asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a)); return (unsigned)v; }
__device__ __forceinline__ double2 lds_v2f64(unsigned a)
{
    double2 v; asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a)); return v;
}
// loads of data written by other SMs during this launch (counters, payloads): through L2, never L1
__device__ __forceinline__ unsigned ldcg_u32(const unsigned *p) { unsigned v; asm volatile("ld.global.cg.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v; }
// The counters of the pipeline are polled with RELAXED gpu-scope loads and bumped with RELEASE atomics: neither
// invalidates L1 (an acquire load or __threadfence emits CCTL.IVALL, which with 24 independent warps per SM
// signalling every few microseconds left no L1 at all for the grid values, and ~3000 warps spinning with
// acquire loads on one line starved the ticket and release atomics behind them: profile r2b, 90 % of the
// samples in the wait loops).  That is sound here because everything another SM wrote during this launch
// (counters, payloads, overflow entries) is read through L2 (.cg / cp.async.cg), never through L1, and is
// only read after the poll that observed the release has returned (the loop exit depends on its value).
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
// called by all 32 lanes of a converged warp: lane 0 polls (one request per iteration), the warp leaves together
__device__ __forceinline__ void warp_wait(const unsigned long long *p, unsigned long long target)
{
    unsigned ns = 64;
    for (;;) {
        unsigned long long v = 0;
        if ((threadIdx.x & 31) == 0) v = ld_relaxed_u64(p);
        v = __shfl_sync(0xffffffffu, v, 0);
        if (v >= target) break;
        __nanosleep(ns);
        if (ns < 2048) ns <<= 1;
    }
}
// release by one warp: every lane's stores are ordered before lane 0's release by the warp barrier, and the
// release is cumulative (the pattern of a grid barrier: sync; one thread releases)
__device__ __forceinline__ unsigned long long warp_release_add(unsigned long long *p, unsigned long long v)
{
    unsigned long long old = 0;
    __syncwarp();
    if ((threadIdx.x & 31) == 0)
        asm volatile("atom.add.release.gpu.global.u64 %0, [%1], %2;" : "=l"(old) : "l"(p), "l"(v) : "memory");
    return __shfl_sync(0xffffffffu, old, 0);
}
// one payload = one 32-byte sector, stored whole (STG.256): never a partial-sector write
__device__ __forceinline__ void store_payload(Payload *dst, double a, double b, unsigned idx)
{
    const double w2 = __hiloint2double(0, (int)idx);
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(dst), "d"(a), "d"(b), "d"(w2), "d"(0.0) : "memory");
}
__device__ __forceinline__ void cp_async16(unsigned saddr, const void *g)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(saddr), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- key space ---------------------------------------------------------------------------------
// x key X in [0, ncx]: the x cell, or ncx for x < X_0.  Fine key fk: the Q2 cell (global lower-knot
// index), nqt for Q2 < Q2min, nqt + 1 for Q2 > Q2max.  A (X, fk) pair is one cell or one
// extrapolation class (a-5): every batch is class-uniform and every branch warp-uniform.
__device__ __forceinline__ int bin_off(const StreamDev &B, int X, int fk)
{
    if (X < B.ncx) return X * B.rowcap + (fk < B.nqt ? fk * B.cap_int : B.nqt * B.cap_int + (fk - B.nqt) * B.cap_cls);
    return B.lxbase + (fk < B.nqt ? fk * B.cap_lx : B.nqt * B.cap_lx + (fk - B.nqt) * B.cap_lxc);
}
__device__ __forceinline__ int bin_cap(const StreamDev &B, int X, int fk)
{
    if (X < B.ncx) return fk < B.nqt ? B.cap_int : B.cap_cls;
    return fk < B.nqt ? B.cap_lx : B.cap_lxc;
}

// ---- a-2 on this path: region class and cell from the raw bit patterns ---------------------------
struct StreamTab {        // shared-window addresses of the tables staged once per CTA
    unsigned xk, qk, cxs, cqs, lutx, lutq;
};
constexpr long long kInfBits = 0x7ff0000000000000LL;

// largest c <= lim with k[c] <= v, for v >= k[0]: the table gives the cell at the lower edge of v's
// bucket (never above the answer), the walk up runs on integer compares of the bit patterns
// (positive doubles order like their bits), so the result is exact for any knots (C-3 / C-4).
__device__ __forceinline__ int s3_search(unsigned s_k, unsigned s_lut, int shift, int base, int nb, int lim, int m, double v)
{
    int b = (__double2hiint(v) >> shift) - base;
    b = b < 0 ? 0 : (b >= nb ? nb - 1 : b);
    int c = (int)lds_u16(s_lut + 2u * b);
    const long long vb = __double_as_longlong(v);
    const long long k1 = lds_s64(s_k + 8u * min(c + 1, m - 1)), k2 = lds_s64(s_k + 8u * min(c + 2, m - 1));
    if (c < lim && k1 <= vb) {
        ++c;
        if (c < lim && k2 <= vb) {
            ++c;
            while (c < lim && lds_s64(s_k + 8u * (c + 1)) <= vb) ++c;
        }
    }
    return c;
}

struct Located { int region, i, g; };     // i: x cell (0 when x < X_0); g: last Q2 knot <= q2 (in-range Q2 only)
__device__ __forceinline__ Located s3_locate(const GridDev &G, const StreamDev &B, const StreamTab &T, double x, double q2,
                                             long long xminb, long long xmaxb, long long qminb, long long qmaxb)
{
    Located L;
    const long long xb = __double_as_longlong(x), qb = __double_as_longlong(q2);
    // C-2 / C-10: 0 < x <= X_last, Q2 > 0, both finite  (NaN, negative and zero patterns fail the unsigned range test)
    const bool valid = (unsigned long long)(xb - 1) < (unsigned long long)xmaxb &&
                       (unsigned long long)(qb - 1) < (unsigned long long)(kInfBits - 1);
    const bool lowx = xb < xminb, lowq = qb < qminb, highq = qb > qmaxb;
    L.region = !valid ? kRegionInvalid
             : lowx ? (lowq ? kRegionLowXLowQ : highq ? kRegionLowXHighQ : kRegionLowX)
                    : (lowq ? kRegionLowQ : highq ? kRegionHighQ : kRegionInterior);
    L.i = 0; L.g = 0;
    if (valid && !lowx) L.i = s3_search(T.xk, T.lutx, B.xshift, B.xbase, B.nbx, G.nx - 2, G.nx, x);
    if (valid && !lowq && !highq) L.g = s3_search(T.qk, T.lutq, B.qshift, B.qbase, B.nbq, G.nqtot - 1, G.nqtot, q2);
    return L;
}

// pdf_locate on this path: the search the evaluation kernel runs, exported (ix, iq local to the sub-grid)
__global__ void __launch_bounds__(256)
k_locate_stream(const __grid_constant__ GridDev G, const __grid_constant__ StreamDev B, long long n,
                const double *__restrict__ x, const double *__restrict__ q2, int *ix, int *iq, int *isub, int *region);

// ---- A tile: classify, locate, t_x / t_q, one slot per query in its cell's bin -----------------
// zero-fill rows [r0, r1) of `out` (contiguous rows of ld doubles) with coalesced 32-byte stores of one warp
__device__ __forceinline__ void zero_fill_warp(double *out, long long ld, long long r0, long long r1, int lane)
{
    double *p = out + r0 * ld, *e = out + r1 * ld;
    if (p >= e) return;
    // head: up to 3 doubles to the next 32-byte boundary
    const int head = (int)(((32u - (unsigned)(reinterpret_cast<size_t>(p) & 31u)) & 31u) >> 3);
    const long long tot = e - p;
    const int h = (long long)head < tot ? head : (int)tot;
    if (lane < h) p[lane] = 0.0;
    p += h;
    const long long n4 = (e - p) >> 2;
    for (long long k = lane; k < n4; k += 32)
        asm volatile("st.global.v4.f64 [%0], {%1,%1,%1,%1};" ::"l"(p + 4 * k), "d"(0.0) : "memory");
    p += 4 * n4;
    if (lane < (int)(e - p)) p[lane] = 0.0;
}

__device__ __forceinline__ void a_tile(const StreamArgs &A, const StreamTab &T, int slot, long long chunk_base, long long chunk_end,
                                       int tile, unsigned long long &err_local)
{
    const GridDev &G = A.G;
    const StreamDev &B = A.B;
    const int lane = threadIdx.x & 31;
    const long long t0 = chunk_base + (long long)tile * kS3TileA;
    long long t1 = t0 + kS3TileA;
    if (t1 > chunk_end) t1 = chunk_end;
    if (t0 >= t1) return;
    unsigned *counts = A.W.counts + (size_t)slot * B.nbins;
    Payload *bins = A.W.bins + (size_t)slot * B.slab;
    if (A.zfill) zero_fill_warp(A.out, A.ld, t0, t1, lane);
    __syncwarp();                                      // the NaN rows below are written by other lanes than the zeros
    const int nx = G.nx, nqt = G.nqtot;
    const long long xminb = lds_s64(T.xk), xmaxb = lds_s64(T.xk + 8u * (nx - 1));
    const long long qminb = lds_s64(T.qk), qmaxb = lds_s64(T.qk + 8u * (nqt - 1));
    const double u0 = __ldg(G.uk);
    // the extrapolation abscissae through reciprocals (one division each per tile instead of per query)
    const double inv_du0 = 1.0 / (__ldg(G.uk + 1) - u0);
    const double sA = __ldg(G.sk + nqt - 2), inv_ds = 1.0 / (__ldg(G.sk + nqt - 1) - sA);
    const double inv_qmin = 1.0 / __longlong_as_double(qminb);
#pragma unroll 1
    for (int g0 = 0; g0 < kS3TileQ; g0 += kS3Grp) {
        double xv[kS3Grp], qv[kS3Grp];
#pragma unroll
        for (int q = 0; q < kS3Grp; ++q) {
            const long long e = t0 + (g0 + q) * 32 + lane;
            xv[q] = 1.0; qv[q] = 1.0;
            if (e < t1) { xv[q] = __ldcs(A.x + e); qv[q] = __ldcs(A.q2 + e); }
        }
        Located L[kS3Grp];
#pragma unroll
        for (int q = 0; q < kS3Grp; ++q) L[q] = s3_locate(G, B, T, xv[q], qv[q], xminb, xmaxb, qminb, qmaxb);
        double pa[kS3Grp], pb[kS3Grp];
        int bin[kS3Grp];
#pragma unroll
        for (int q = 0; q < kS3Grp; ++q) {
            const int r = L[q].region;
            const bool lowx = r == kRegionLowX || r == kRegionLowXLowQ || r == kRegionLowXHighQ;
            const bool lowq = r == kRegionLowQ || r == kRegionLowXLowQ, highq = r == kRegionHighQ || r == kRegionLowXHighQ;
            const int i = L[q].i;
            const int jg = L[q].g < nqt - 1 ? L[q].g : nqt - 2;       // only Q2 == Q2max lands on the last knot: it belongs to the last cell
            const double2 ci = lds_v2f64(T.cxs + 16u * i), cj = lds_v2f64(T.cqs + 16u * jg);
            double lx = 0.0, lq = 0.0;
            if (r != kRegionInvalid) { lx = log(xv[q]); lq = log(qv[q]); }
            // t = 1 exactly on the last knot (the only knot that belongs to the cell on its left, C-4)
            pa[q] = lowx ? (lx - u0) * inv_du0                                    // theta_x (C-7)
                         : (__double_as_longlong(xv[q]) == xmaxb) ? 1.0 : (lx - ci.x) * ci.y;
            pb[q] = lowq ? qv[q] * inv_qmin                                       // r (C-9)
                  : highq ? (lq - sA) * inv_ds                                    // theta_q (C-8)
                          : (__double_as_longlong(qv[q]) == qmaxb) ? 1.0 : (lq - cj.x) * cj.y;
            const int X = lowx ? B.ncx : i;
            const int fk = lowq ? nqt : highq ? nqt + 1 : jg;
            bin[q] = r == kRegionInvalid ? -1 : X * B.nfk + fk;
        }
        unsigned pos[kS3Grp];
#pragma unroll
        for (int q = 0; q < kS3Grp; ++q) {
            const long long e = t0 + (g0 + q) * 32 + lane;
            pos[q] = 0u;
            if (e < t1 && bin[q] >= 0) pos[q] = atomicAdd(counts + bin[q], 1u);
        }
#pragma unroll
        for (int q = 0; q < kS3Grp; ++q) {
            const long long e = t0 + (g0 + q) * 32 + lane;
            if (e >= t1) continue;
            if (bin[q] < 0) {                                                     // C-10: NaN row, counted
                double *o = A.out + e * A.ld;
                for (int p = 0; p < A.cm.n; ++p) o[p] = qnan();
                if (A.count_err) ++err_local;
                continue;
            }
            const int X = bin[q] / B.nfk, fk = bin[q] - X * B.nfk;
            if (pos[q] < (unsigned)bin_cap(B, X, fk))
                store_payload(bins + bin_off(B, X, fk) + pos[q], pa[q], pb[q], (unsigned)(e - chunk_base));
            else {                                                                // bin full: raw query to the overflow list
                const unsigned o = atomicAdd(A.W.ovf_count + slot, 1u);
                store_payload(A.W.ovf + (size_t)slot * A.chunk + o, xv[q], qv[q], (unsigned)(e - chunk_base));
            }
        }
    }
}

// ---- B units: DMMA contractions on the cell's values ---------------------------------------------
// out[q][f] = sum_n W[q][n] V[n][f] is a (queries x 16 nodes) x (16 nodes x 11 flavours) contraction.  As
// mma.sync.m8n8k4 tiles (8 queries x 8 flavours, k = 4 nodes) the cell's values are read ONCE per cell, 8
// doubles per lane.  DMMA runs on the same FP64 pipe as DFMA: this buys operand
// traffic and instruction count, not flops.  Lane (g = lane/4, t = lane%4) serves query g of the 8-query
// tile and holds flavours 2t, 2t+1, 8+2t, 9+2t of it in the accumulator fragments.
// Step r of 4 uses Q2-row (t ^ r) and x-node t:  A[g][t] = wq_g[t^r] wx_g[t],  B[t][n] = V[row t^r][node t][n].
__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
struct Acc { double d00, d01, d10, d11; };              // flavours 2t, 2t+1, 8+2t, 9+2t (the last two exist for t < 2, t == 0)
__device__ __forceinline__ void kstep(Acc &d, double a, double2 f) { dmma884(d.d00, d.d01, a, f.x); dmma884(d.d10, d.d11, a, f.y); }
// fragment of node (row, col): flavour g in .x, flavour 8 + g in .y (the 12th column of a row is a zero pad)
__device__ __forceinline__ double2 fragld(const double *__restrict__ Vm, int nx, int row, int col, int g)
{
    const double *p = Vm + ((size_t)row * nx + col) * kNFP;
    return make_double2(__ldg(p + g), g < 4 ? __ldg(p + 8 + g) : 0.0);
}

// node weight number t of the 1-D Hermite operator in the factored form
//   w_t = (1-s)^2 (c0 + c1 s) + s^2 (c2 + c3 (1-s))        (same weights as hermite_weights)
struct WCoef { double c0, c1, c2, c3; };
__device__ __forceinline__ WCoef weight_coef(const CellTab &c, int t)
{
    WCoef w;
    w.c0 = t == 1 ? 1.0 : 0.0;
    w.c1 = t == 0 ? -c.bL : t == 1 ? 2.0 + c.bL - c.aL : t == 2 ? c.aL : 0.0;
    w.c2 = t == 2 ? 1.0 : 0.0;
    w.c3 = t == 1 ? c.aR : t == 2 ? 2.0 - c.aR + c.bR : t == 3 ? -c.bR : 0.0;
    return w;
}
__device__ __forceinline__ double weight_eval(const WCoef &w, double s)
{
    double om = 1.0 - s, om2 = om * om, s2 = s * s;
    return fma(om2, fma(w.c1, s, w.c0), s2 * fma(w.c3, om, w.c2));
}
// Q2 row number tr (0..3) of cell jg: jg-1 .. jg+2, clamped at the ends of the sub-grid (q_point_cell)
__device__ __forceinline__ int qrow(const CellTab &cq, int jg, int tr)
{
    return jg - 1 + tr + ((tr == 0 && cq.aL == 1.0) ? 1 : 0) - ((tr == 3 && cq.aR == 1.0) ? 1 : 0);
}
// x node number t (0..3) of cell i: i-1 .. i+2, clamped at the ends of the knot line (x_point_cell)
__device__ __forceinline__ int xnode(int i, int t, int nx)
{
    const int c = i - 1 + t;
    return c < 0 ? 0 : (c >= nx ? nx - 1 : c);
}

// the per-flavour continuation formulas on accumulator fragments (kept out of line: ~12 inlined
// transcendental calls each)
__device__ __noinline__ void acc_two(Acc &o, const Acc &a, const Acc &b, double theta, int t)
{
    o.d00 = continue_two(a.d00, b.d00, theta);
    o.d01 = continue_two(a.d01, b.d01, theta);
    o.d10 = t < 2 ? continue_two(a.d10, b.d10, theta) : 0.0;
    o.d11 = t == 0 ? continue_two(a.d11, b.d11, theta) : 0.0;
}
__device__ __noinline__ void acc_lowq(Acc &o, const Acc &fmin, const Acc &fplus, double r, int t)
{
    const double lnr = log(r);
    o.d00 = lowq_continue_ln(fmin.d00, fplus.d00, r, lnr);
    o.d01 = lowq_continue_ln(fmin.d01, fplus.d01, r, lnr);
    o.d10 = t < 2 ? lowq_continue_ln(fmin.d10, fplus.d10, r, lnr) : 0.0;
    o.d11 = t == 0 ? lowq_continue_ln(fmin.d11, fplus.d11, r, lnr) : 0.0;
}

// one row from the accumulator fragments: 4 lanes write one row
__device__ __forceinline__ void store_row(const StreamArgs &A, double *rp, int t, const Acc &d)
{
    if (A.identity) {
        rp[2 * t] = d.d00; rp[2 * t + 1] = d.d01;
        if (t < 2) rp[8 + 2 * t] = d.d10;
        if (t == 0) rp[9] = d.d11;
    } else {
        for (int p = 0; p < A.cm.n; ++p) {
            const int c = A.cm.col[p];
            if (c < 0) { if (t == 0) rp[p] = 0.0; continue; }
            if (((c & 7) >> 1) == t) rp[p] = (c & 8) ? ((c & 1) ? d.d11 : d.d10) : ((c & 1) ? d.d01 : d.d00);
        }
    }
}

// payload batches of one bin through a double-buffered cp.async stage (one warp): the caller's
// body(n, sbuf) sees n <= 32 payloads at shared-window address sbuf
template <typename Body>
__device__ __forceinline__ void for_batches(const Payload *bin, int first, int count, unsigned sbuf, int lane, Body body)
{
    if (count <= 0) return;
    auto issue = [&](int o, unsigned dst) {
        const int n = min(kS3Batch, count - o);
        if (lane < n) {
            const char *src = reinterpret_cast<const char *>(bin + first + o + lane);
            cp_async16(dst + 32u * lane, src);
            cp_async16(dst + 32u * lane + 16u, src + 16);
        }
        cp_async_commit();
    };
    issue(0, sbuf);
    int p = 0;
    for (int o = 0; o < count; o += kS3Batch) {
        if (o + kS3Batch < count) { issue(o + kS3Batch, sbuf + (unsigned)((p ^ 1) * kS3Batch * 32)); cp_async_wait<1>(); }
        else cp_async_wait<0>();
        __syncwarp();
        body(min(kS3Batch, count - o), sbuf + (unsigned)(p * kS3Batch * 32));
        __syncwarp();
        p ^= 1;
    }
}

// interior cells (X = i < ncx, fine keys [fk0, fk1) are Q2 cells)
__device__ __forceinline__ void b_unit_interior(const StreamArgs &A, const double *__restrict__ Vm, int slot, long long chunk_base,
                                                int i, int fk0, int fk1, unsigned sbuf)
{
    const GridDev &G = A.G;
    const StreamDev &B = A.B;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const unsigned *counts = A.W.counts + (size_t)slot * B.nbins + (size_t)i * B.nfk;
    const Payload *bins = A.W.bins + (size_t)slot * B.slab;
    int mycnt = 0;
    if (fk0 + lane < fk1) mycnt = min((int)ldcg_u32(counts + fk0 + lane), B.cap_int);
    if (__ballot_sync(0xffffffffu, mycnt > 0) == 0u) return;
    const WCoef kx = weight_coef(G.cx[i], t);          // x-axis weight of this lane's node, fixed for the unit
    const int xc = xnode(i, t, G.nx);
    for (int fk = fk0; fk < fk1; ++fk) {
        const int cnt = __shfl_sync(0xffffffffu, mycnt, fk - fk0);
        if (cnt == 0) continue;
        const CellTab cq = G.cq[fk];
        const WCoef kq = weight_coef(cq, t);
        double2 f[4];
#pragma unroll
        for (int r = 0; r < 4; ++r) f[r] = fragld(Vm, G.nx, qrow(cq, fk, t ^ r), xc, g);
        for_batches(bins + bin_off(B, i, fk), 0, cnt, sbuf, lane, [&](int nact, unsigned sb) {
            // the next tile's abscissae are fetched under this tile's arithmetic
            bool vn = g < nact;
            double2 abn = make_double2(0.0, 0.0);
            unsigned idxn = 0;
            if (vn) { abn = lds_v2f64(sb + 32u * g); idxn = lds_u32(sb + 32u * g + 16u); }
            for (int m0 = 0; m0 < nact; m0 += 8) {
                const bool valid = vn;
                const double tx = abn.x, tq = abn.y;
                const unsigned idx = idxn;
                const int qn = m0 + 8 + g;
                vn = qn < nact;
                if (vn) { abn = lds_v2f64(sb + 32u * qn); idxn = lds_u32(sb + 32u * qn + 16u); }
                const double wx = valid ? weight_eval(kx, tx) : 0.0;
                const double wq0 = weight_eval(kq, tq);
                const double wq1 = __shfl_xor_sync(0xffffffffu, wq0, 1);
                const double wq2 = __shfl_xor_sync(0xffffffffu, wq0, 2);
                const double wq3 = __shfl_xor_sync(0xffffffffu, wq0, 3);
                Acc d = {0.0, 0.0, 0.0, 0.0};
                kstep(d, wq0 * wx, f[0]);
                kstep(d, wq1 * wx, f[1]);
                kstep(d, wq2 * wx, f[2]);
                kstep(d, wq3 * wx, f[3]);
                if (valid) store_row(A, A.out + (chunk_base + idx) * A.ld, t, d);
            }
        });
    }
}

// extrapolation classes (a-5): bin (X, fk) with X == ncx (x < X_0) or fk >= nqt (Q2 outside); slots
// [first, first + count) of the bin.  Same 4-lanes-per-query layout: the linear parts are k-steps on node
// sets fixed by the class, the continuation formulas run on the fragments.
//   X < ncx, fk == nqt   (low-Q, C-9):   a = t_x, b = r        e0 = row Q2min,       e1 = cell of 1.01 Q2min at tqplus
//   X < ncx, fk == nqt+1 (high-Q, C-8):  a = t_x, b = theta_q  e0 = row last-1,      e1 = row last
//   X == ncx, fk < nqt   (low-x, C-7):   a = theta_x, b = t_q  e0 = column X_0,      e1 = column X_1 (4 rows of cell fk)
//   X == ncx, fk == nqt  (corner):       a = theta_x, b = r    x rule on (Q2min) and on (1.01 Q2min), then C-9  (L1744)
//   X == ncx, fk == nqt+1 (corner):      a = theta_x, b = theta_q   x rule on rows last-1 and last, then C-8
__device__ __noinline__ void b_unit_class(const StreamArgs &A, const double *__restrict__ Vm, long long chunk_base,
                                          const Payload *bin, int first, int count, int X, int fk, unsigned sbuf)
{
    const GridDev &G = A.G;
    const StreamDev &B = A.B;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const int nx = G.nx, last = G.nqtot - 1;
    const bool lowx = X == B.ncx;
    const int i = lowx ? 0 : X;
    const WCoef kx = weight_coef(G.cx[i], t);
    const int xc = xnode(i, t, nx);
    const CellTab cqp = G.cq[B.jgplus];
    const double unit0 = t == 0 ? 1.0 : 0.0;           // k-step weight that picks node slot 0 alone
    // weights of the cell of 1.01*Q2min at tqplus (C-9), by row
    double wqp[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) wqp[r] = weight_eval(weight_coef(cqp, r), B.tqplus);
    const CellTab cqf = G.cq[fk < B.nqt ? fk : 0];
    const WCoef kq = weight_coef(cqf, t);
    for_batches(bin, first, count, sbuf, lane, [&](int nact, unsigned sb) {
        for (int m0 = 0; m0 < nact; m0 += 8) {
            const int q = m0 + g;
            const bool valid = q < nact;
            double pa = 0.0, pb = 1.0;
            unsigned idx = 0;
            if (valid) { const double2 ab = lds_v2f64(sb + 32u * q); pa = ab.x; pb = ab.y; idx = lds_u32(sb + 32u * q + 16u); }
            Acc o;
            if (!lowx) {
                const double wx = weight_eval(kx, pa);
                Acc e0 = {0.0, 0.0, 0.0, 0.0}, e1 = {0.0, 0.0, 0.0, 0.0};
                if (fk == B.nqt) {
                    kstep(e0, wx, fragld(Vm, nx, 0, xc, g));
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        // step r pairs row (t ^ r) with x-node t: the row weight is a select among the 4 constants
                        const int tr = t ^ r;
                        const double w = tr == 0 ? wqp[0] : tr == 1 ? wqp[1] : tr == 2 ? wqp[2] : wqp[3];
                        kstep(e1, w * wx, fragld(Vm, nx, qrow(cqp, B.jgplus, tr), xc, g));
                    }
                    acc_lowq(o, e0, e1, pb, t);
                } else {
                    kstep(e0, wx, fragld(Vm, nx, last - 1, xc, g));
                    kstep(e1, wx, fragld(Vm, nx, last, xc, g));
                    acc_two(o, e0, e1, pb, t);
                }
            } else if (fk < B.nqt) {
                const double wq = weight_eval(kq, pb);
                const int row = qrow(cqf, fk, t);
                Acc e0 = {0.0, 0.0, 0.0, 0.0}, e1 = {0.0, 0.0, 0.0, 0.0};
                kstep(e0, wq, fragld(Vm, nx, row, 0, g));
                kstep(e1, wq, fragld(Vm, nx, row, 1, g));
                acc_two(o, e0, e1, pa, t);
            } else {
                Acc e0 = {0.0, 0.0, 0.0, 0.0}, e1 = {0.0, 0.0, 0.0, 0.0}, e2 = {0.0, 0.0, 0.0, 0.0}, e3 = {0.0, 0.0, 0.0, 0.0};
                if (fk == B.nqt) {
                    const double w = t == 0 ? wqp[0] : t == 1 ? wqp[1] : t == 2 ? wqp[2] : wqp[3];
                    const int row = qrow(cqp, B.jgplus, t);
                    kstep(e0, unit0, fragld(Vm, nx, 0, 0, g));
                    kstep(e1, unit0, fragld(Vm, nx, 0, 1, g));
                    kstep(e2, w, fragld(Vm, nx, row, 0, g));
                    kstep(e3, w, fragld(Vm, nx, row, 1, g));
                } else {
                    kstep(e0, unit0, fragld(Vm, nx, last - 1, 0, g));
                    kstep(e1, unit0, fragld(Vm, nx, last - 1, 1, g));
                    kstep(e2, unit0, fragld(Vm, nx, last, 0, g));
                    kstep(e3, unit0, fragld(Vm, nx, last, 1, g));
                }
                Acc lo, hi;
                acc_two(lo, e0, e1, pa, t);
                acc_two(hi, e2, e3, pa, t);
                if (fk == B.nqt) acc_lowq(o, lo, hi, pb, t); else acc_two(o, lo, hi, pb, t);
            }
            if (valid) store_row(A, A.out + (chunk_base + idx) * A.ld, t, o);
        }
    });
}

// low-x key, fine keys [fk0, fk1) are Q2 cells: one class bin per cell
__device__ __forceinline__ void b_unit_lowx(const StreamArgs &A, const double *__restrict__ Vm, int slot, long long chunk_base,
                                            int fk0, int fk1, unsigned sbuf)
{
    const StreamDev &B = A.B;
    const int lane = threadIdx.x & 31;
    const unsigned *counts = A.W.counts + (size_t)slot * B.nbins + (size_t)B.ncx * B.nfk;
    const Payload *bins = A.W.bins + (size_t)slot * B.slab;
    int mycnt = 0;
    if (fk0 + lane < fk1) mycnt = min((int)ldcg_u32(counts + fk0 + lane), B.cap_lx);
    for (int fk = fk0; fk < fk1; ++fk) {
        const int cnt = __shfl_sync(0xffffffffu, mycnt, fk - fk0);
        if (cnt) b_unit_class(A, Vm, chunk_base, bins + bin_off(B, B.ncx, fk), 0, cnt, B.ncx, fk, sbuf);
    }
}

// overflow list: raw queries evaluated by the generic per-thread code (rare)
__device__ __noinline__ void ovf_unit(const StreamArgs &A, const double *V, int slot, long long chunk_base, int part)
{
    const unsigned cnt = ldcg_u32(A.W.ovf_count + slot);
    const Payload *ovf = A.W.ovf + (size_t)slot * A.chunk;
    for (unsigned e = part * 32 + (threadIdx.x & 31); e < cnt; e += kS3Ovf * 32) {
        const double2 ab = __ldcg(reinterpret_cast<const double2 *>(ovf + e));
        const unsigned idx = __ldcg(reinterpret_cast<const unsigned *>(ovf + e) + 4);
        QueryPlan P;
        make_plan(A.G, ab.x, ab.y, P);
        double *o = A.out + (chunk_base + idx) * A.ld;
        for (int p = 0; p < A.cm.n; ++p) {
            const int c = A.cm.col[p];
            o[p] = c < 0 ? 0.0 : plan_value(A.G, V, P, c);
        }
    }
}

// ---- the persistent kernel -----------------------------------------------------------------------
// dynamic shared memory: [x knots | Q2 knots | x cell {ln lo, 1/d} | Q2 cell {ln lo, 1/d} | lutx | lutq | per-warp payload stage]
__host__ __device__ inline size_t s3_table_bytes(int nx, int nqt, int nbx, int nbq)
{
    size_t b = sizeof(double) * (size_t)(nx + nqt) + 16u * (size_t)(nx + nqt) + 2u * (size_t)(nbx + nbq);
    return (b + 31) / 32 * 32;
}
__device__ __forceinline__ StreamTab s3_stage_tables(const GridDev &G, const StreamDev &B, unsigned char *smem, int nthreads)
{
    double *s_xk = reinterpret_cast<double *>(smem);
    double *s_qk = s_xk + G.nx;
    double2 *s_cx = reinterpret_cast<double2 *>(s_qk + G.nqtot + ((G.nx + G.nqtot) & 1));
    double2 *s_cq = s_cx + G.nx;
    unsigned short *s_lx = reinterpret_cast<unsigned short *>(s_cq + G.nqtot);
    unsigned short *s_lq = s_lx + B.nbx;
    for (int k = threadIdx.x; k < G.nx; k += nthreads) s_xk[k] = G.xk[k];
    for (int k = threadIdx.x; k < G.nqtot; k += nthreads) s_qk[k] = G.qk[k];
    for (int k = threadIdx.x; k < B.ncx; k += nthreads) s_cx[k] = B.cxs[k];
    for (int k = threadIdx.x; k < G.nqtot; k += nthreads) s_cq[k] = B.cqs[k];
    for (int k = threadIdx.x; k < B.nbx; k += nthreads) s_lx[k] = B.lutx[k];
    for (int k = threadIdx.x; k < B.nbq; k += nthreads) s_lq[k] = B.lutq[k];
    StreamTab T;
    T.xk = (unsigned)__cvta_generic_to_shared(s_xk); T.qk = (unsigned)__cvta_generic_to_shared(s_qk);
    T.cxs = (unsigned)__cvta_generic_to_shared(s_cx); T.cqs = (unsigned)__cvta_generic_to_shared(s_cq);
    T.lutx = (unsigned)__cvta_generic_to_shared(s_lx); T.lutq = (unsigned)__cvta_generic_to_shared(s_lq);
    return T;
}
__host__ __device__ inline size_t s3_table_bytes_padded(int nx, int nqt, int nbx, int nbq)
{
    return s3_table_bytes(nx, nqt, nbx, nbq) + 64;       // alignment slack of the double2 tables
}

__global__ void __launch_bounds__(256)
k_locate_stream(const __grid_constant__ GridDev G, const __grid_constant__ StreamDev B, long long n,
                const double *__restrict__ x, const double *__restrict__ q2, int *ix, int *iq, int *isub, int *region)
{
    extern __shared__ __align__(32) unsigned char smem_raw[];
    const StreamTab T = s3_stage_tables(G, B, smem_raw, 256);
    __syncthreads();
    const long long xminb = lds_s64(T.xk), xmaxb = lds_s64(T.xk + 8u * (G.nx - 1));
    const long long qminb = lds_s64(T.qk), qmaxb = lds_s64(T.qk + 8u * (G.nqtot - 1));
    for (long long e = (long long)blockIdx.x * 256 + threadIdx.x; e < n; e += (long long)gridDim.x * 256) {
        const Located L = s3_locate(G, B, T, x[e], q2[e], xminb, xmaxb, qminb, qmaxb);
        const int r = L.region;
        int i = -1, j = -1, k = -1;
        if (r != kRegionInvalid) {
            i = L.i;                                                        // 0 for the low-x classes (anchored on X_0, X_1)
            if (r == kRegionLowQ || r == kRegionLowXLowQ) { k = 0; j = 0; }
            else if (r == kRegionHighQ || r == kRegionLowXHighQ) { k = G.nsub - 1; j = G.qoff[k + 1] - G.qoff[k] - 2; }
            else {
                const int jg = L.g < G.nqtot - 1 ? L.g : G.nqtot - 2;
                k = G.sub_of[jg];
                j = jg - G.qoff[k];
            }
        }
        if (ix) ix[e] = i;
        if (iq) iq[e] = j;
        if (isub) isub[e] = k;
        if (region) region[e] = r;
    }
}

__global__ void __launch_bounds__(kS3Threads, PDF_S3_MINB) k_pdf_stream(const __grid_constant__ StreamArgs A)
{
    extern __shared__ __align__(32) unsigned char smem_raw[];
    const StreamTab T = s3_stage_tables(A.G, A.B, smem_raw, kS3Threads);
    const unsigned stage0 = (unsigned)__cvta_generic_to_shared(smem_raw) +
                            (unsigned)s3_table_bytes_padded(A.G.nx, A.G.nqtot, A.B.nbx, A.B.nbq);
    __syncthreads();                                   // the only CTA barrier: every warp works alone from here on
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned sbuf = ((stage0 + 31u) & ~31u) + (unsigned)(warp * 2 * kS3Batch * 32);

    unsigned long long *ctrl = A.W.ctrl;
    const StreamDev &B = A.B;
    const unsigned long long TA = A.ta, TB = B.tb, per = TA + TB;
    const int nchunks = A.ctab ? __ldg(A.nchunks_dev) : A.nchunks;
    const unsigned long long total = (unsigned long long)nchunks * per;
    unsigned long long err_local = 0;
    // the last wait that was satisfied: consecutive units of one chunk need not poll again
    const unsigned long long *seen_p = nullptr;
    unsigned long long seen_v = 0;
    auto wait_for = [&](const unsigned long long *p, unsigned long long target) {
        if (p == seen_p && target <= seen_v) return;
        warp_wait(p, target);
        seen_p = p; seen_v = target;
    };

    // the next ticket is fetched while the current item runs (a global atomic is ~1 us)
    unsigned long long next_t = 0;
    if (lane == 0) next_t = atomicAdd(ctrl, 1ULL);
    for (;;) {
        const unsigned long long t = __shfl_sync(0xffffffffu, next_t, 0);
        if (t >= total) break;
        if (lane == 0) next_t = atomicAdd(ctrl, 1ULL);
        // ticket order, lag L = kS3Lag rounds:  round r = [A(r) tiles | B(r-L) units]
        bool isA; long long c; int sub;
        {
            const unsigned long long RA = (unsigned long long)(nchunks < kS3Lag ? nchunks : kS3Lag);   // A-only rounds
            const unsigned long long F = (unsigned long long)nchunks - RA;                               // full rounds
            if (t < RA * TA) { isA = true; c = (long long)(t / TA); sub = (int)(t % TA); }
            else {
                const unsigned long long tp = t - RA * TA;
                if (tp < F * per) {
                    const unsigned long long round = RA + tp / per, w = tp % per;
                    isA = w < TA;
                    c = isA ? (long long)round : (long long)(round - RA);
                    sub = (int)(isA ? w : w - TA);
                } else {
                    const unsigned long long tq = tp - F * per;
                    isA = false; c = (long long)(F + tq / TB); sub = (int)(tq % TB);
                }
            }
        }
        const int slot = (int)(c % kS3Ring);
        const unsigned long long gen = (unsigned long long)(c / kS3Ring);
        unsigned long long *a_done = ctrl + 32 + slot * 48, *b_fin = a_done + 16, *b_done = a_done + 32;
        long long chunk_base = c * A.chunk, chunk_end = chunk_base + A.chunk;
        if (chunk_end > A.n) chunk_end = A.n;
        const double *V = A.G.V;
        if (A.ctab) {                                              // a-8: the chunk is a piece of one member's run
            const int4 ce = __ldg(reinterpret_cast<const int4 *>(A.ctab) + c);
            chunk_base = ce.x; chunk_end = (long long)ce.x + ce.y;
            V += (size_t)ce.z * A.G.memstride;
        }
        if (isA) {
            // the ring slot must have been drained by B(c - kS3Ring) before this tile touches its bins
            if (gen) wait_for(b_done, gen * TB);
            a_tile(A, T, slot, chunk_base, chunk_end, sub, err_local);
            warp_release_add(a_done, 1ULL);
        } else {
            wait_for(a_done, (gen + 1) * TA);                      // every tile of A(c) has been released
            const int ncls = (B.ncx + 1) * kS3ClassParts;
            const int ncell = (B.ncx + 1) * B.ng;
            if (sub < ncls) {                                      // class bins first: the long units must not end the round
                const int X = B.ncx - sub / kS3ClassParts, part = sub % kS3ClassParts;
                unsigned c2 = 0;
                if (lane < 2) c2 = ldcg_u32(A.W.counts + (size_t)slot * B.nbins + (size_t)X * B.nfk + B.nqt + lane);
                for (int cls = 0; cls < 2; ++cls) {                // low-Q, then high-Q
                    const int fk = B.nqt + cls;
                    const int cap = bin_cap(B, X, fk), seg = (cap + kS3ClassParts - 1) / kS3ClassParts;
                    int cnt = (int)__shfl_sync(0xffffffffu, c2, cls);
                    cnt = cnt < cap ? cnt : cap;
                    const int first = part * seg, cntp = min(seg, cnt - first);
                    if (cntp > 0)
                        b_unit_class(A, V, chunk_base, A.W.bins + (size_t)slot * B.slab + bin_off(B, X, fk), first, cntp, X, fk, sbuf);
                }
            } else if (sub < ncls + ncell) {
                const int v = sub - ncls;
                const int X = B.ncx - v / B.ng, grp = v % B.ng;    // the low-x key first
                const int fk0 = grp * kS3FkPerUnit, fk1 = min(B.nqt, fk0 + kS3FkPerUnit);
                if (X == B.ncx) b_unit_lowx(A, V, slot, chunk_base, fk0, fk1, sbuf);
                else b_unit_interior(A, V, slot, chunk_base, X, fk0, fk1, sbuf);
            } else {
                ovf_unit(A, V, slot, chunk_base, sub - ncls - ncell);
            }
            const unsigned long long old = warp_release_add(b_fin, 1ULL);
            if (old + 1 == (gen + 1) * TB) {                       // last unit of the chunk: the slot's counters are reset for the ring
                unsigned *cz = A.W.counts + (size_t)slot * B.nbins;
                for (int k = lane; k < B.nbins; k += 32) cz[k] = 0u;
                if (lane == 0) A.W.ovf_count[slot] = 0u;
                warp_release_add(b_done, TB);
            }
        }
    }
    if (err_local) atomicAdd(A.G.err_count, err_local);
}

__host__ __device__ inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace pdfg

#include "pdf_members.cuh"
#include "pdf_stream_host.cuh"
