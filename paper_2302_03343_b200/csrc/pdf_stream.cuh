// pdf_stream.cuh -- the binned, cell-coherent evaluation path (PDF_PATH_BINNED), version 3:
// one persistent kernel of independent WARPS, one bin per CELL, no CTA barrier on the path.
//
// Why binning at all: a query needs a 4 x 4 stencil x 11 flavours = 1408 B of grid
// data; gathered per lane that is >= 12 clk/query/SM of L1 / shared-memory bandwidth against a
// budget of 7.9 clk/query/SM at 60 % of the HBM roofline.  Queries that share a cell take the
// cell's 16 x 11 values ONCE, as operand fragments of FP64 mma.sync tiles.  With ~10^4 cells that
// needs a sort domain of ~3 x 10^5 queries: they are binned through L2 in chunks.
//
// What changed against version 2 (one coarse bin per x cell, tile-local counting sorts in shared
// memory in A, payload staging + counting sort by Q2 cell in B, 46 warp instructions per query, 16
// warps/SM, profiles/r1i, r1j): the bin IS the cell, and every work item belongs to ONE warp.
//   A tile (one warp, 256 queries): coalesced loads of x, Q2; validity / region class on the bit
//     patterns; cell search from a table indexed by the exponent and top mantissa bits (integer
//     compares on the raw knots: C-3 / C-4 bit-exact, FP64 pipe untouched); t_x, t_q (two logs);
//     ONE global atomic per query reserves a slot in the cell's bin, the 32-byte payload
//     {a, b, idx, cell} is stored as one whole sector.  The tile's output rows are zero-filled with
//     coalesced 32-byte stores first, so that the scattered 88-byte rows of B merge into valid
//     L2-resident sectors (scattered partial-sector stores into untouched
//     memory run at 0.9 TB/s).  No shared-memory sort, no barrier.
//   B unit (one warp, 8 consecutive Q2 cells of one x cell): reads the 8 counts, then walks the
//     cells' payload batches (<= 32 queries) through a double-buffered cp.async stage that also
//     carries the cell's 16 node rows (the next batch and the next cell's values are in flight
//     under the current batch's arithmetic), and runs DMMA m8n8k4 tiles of 8 queries x 8 flavours;
//     rows leave from the accumulator fragments.  No counting sort, no batch descriptors.
//   E unit (one warp): the extrapolation classes (a-5) are 5 % of configs[2] but cost ~40 x an
//     interior query each (11 flavours x two logarithms and an exponential); as bins of the cell
//     pipeline their units ran 250 us and stalled the ring (first build of this version, profile
//     r2b).  They go to per-class lists of the chunk instead (one warp-aggregated atomic per warp
//     and class), and E units claim batches of 32 entries from the lists dynamically: one query per
//     lane, node rows gathered through L1 (8 rows per query; C-9's second anchor row, the values at
//     1.01 Q2min, is tabulated once per grid), class-uniform branches.  Queries beyond a cell bin's
//     capacity go to a sixth list that the same evaluator serves with the full 16-row stencil:
//     correctness never depends on the distribution of the queries.
// Work is handed out per warp by a global ticket counter in the order
//      round r = [ A(r) tiles | E(r - kLag), B(r - kLag) units ],
// B/E(c) wait until every A tile of chunk c has been released, A(c) until the units of chunk
// c - kRing have drained the ring slot; a ticket only ever waits on lower tickets and every CTA is
// resident, so the scheme cannot deadlock.
#pragma once
#include <climits>
#include "pdf_common.cuh"
#include "pdf_generic.cuh"

namespace pdfg {

#ifndef PDF_S3_GRP
#define PDF_S3_GRP 2
#endif
#ifndef PDF_S3_EDIV
#define PDF_S3_EDIV 1024                             // one E unit per this many queries of a chunk
#endif
#ifndef PDF_S3_LAG
#define PDF_S3_LAG 2
#endif
#ifndef PDF_S3_RING
#define PDF_S3_RING 8
#endif
#ifndef PDF_S3_MINB
#define PDF_S3_MINB 2                                // 2 CTAs of 256 threads per SM: 128 registers, no spills (80 registers
                                                     // and 3 CTAs spilled ~250 B per thread and ran 1.5x slower)
#endif
#ifndef PDF_S3_THREADS
#define PDF_S3_THREADS 256
#endif
constexpr int kS3Threads = PDF_S3_THREADS;                      // CTA size of the persistent kernel; every warp works alone
constexpr int kS3Warps = kS3Threads / 32;
#ifndef PDF_S3_TILEQ
#define PDF_S3_TILEQ 8
#endif
constexpr int kS3TileQ = PDF_S3_TILEQ;               // queries per lane in an A tile
constexpr int kS3TileA = 32 * kS3TileQ;              // 256 queries per A tile (one warp)
constexpr int kS3Grp = PDF_S3_GRP;                   // queries of a lane that go through the A steps together
static_assert(kS3TileQ % kS3Grp == 0, "kS3TileQ must be a multiple of kS3Grp");
constexpr int kS3Batch = 32;                         // list entries per E batch
#ifndef PDF_S3_FKU
#define PDF_S3_FKU 16
#endif
#ifndef PDF_S3_FKU_LUMI2
#define PDF_S3_FKU_LUMI2 8
#endif
// Q2 cells per B unit (at most 32: a lane per cell): 16 for rows (7.71 -> 7.55 ms per 1e8 C2 queries against 8); pass 2 of
// the luminosity, whose units also fetch the rows of pass 1, runs best with 8 (11.6 against 13.9 ms per 1e8 C4 events)
constexpr int kS3FkPerUnit = PDF_S3_FKU, kS3FkPerUnitLumi2 = PDF_S3_FKU_LUMI2;
static_assert(kS3FkPerUnit <= 32 && kS3FkPerUnitLumi2 <= 32, "a B unit keeps one cell count per lane");
constexpr int kS3Lag = PDF_S3_LAG;                   // B(c) tickets follow A(c) tickets by this many rounds
constexpr int kS3Ring = PDF_S3_RING;                 // chunk slots in flight
static_assert(kS3Ring >= kS3Lag + 2, "A(c) must find the slot of B(c - kRing) drained");
constexpr int kS3LutMax = 2048;                      // search-table buckets per axis
constexpr int kNF = 11, kNFP = 12;                   // the path is specialised for 11 flavours (rows padded to 12)
constexpr int kS3MaxCells = 1024;                    // x cells / Q2 knots the path supports (u16 tables)
// lists of the E units: entries that are not evaluated from a cell bin (1..5 = the region codes)
constexpr int kListOvf = 0, kListLowX = 1, kListLowQ = 2, kListHighQ = 3, kListLowXLowQ = 4, kListLowXHighQ = 5, kNumLists = 6;
static_assert(kListLowX == kRegionLowX && kListLowQ == kRegionLowQ && kListHighQ == kRegionHighQ &&
              kListLowXLowQ == kRegionLowXLowQ && kListLowXHighQ == kRegionLowXHighQ, "list numbers are the region codes");
#ifndef PDF_EV_BATCH
#define PDF_EV_BATCH 48
#endif
#ifndef PDF_EV_DEPTH
#define PDF_EV_DEPTH 2
#endif
constexpr int kEvBatch = PDF_EV_BATCH;               // payloads per stage of a B unit (whole 8-query tiles)
constexpr int kEvDepth = PDF_EV_DEPTH;               // stages per warp: kEvDepth - 1 batches are in flight under the arithmetic
constexpr int kEvHdr = 32;                           // stage header {payloads, Q2 cell}
constexpr int kStageV = 16 * kNFP * 8;               // bytes of a cell's 16 node rows
constexpr int kEvStage = kEvHdr + kEvBatch * 32 + kStageV;   // a self-contained stage: header | payloads | node rows
constexpr int kStageBytes = kEvDepth * kEvStage;     // per warp
static_assert(kEvBatch % 8 == 0 && kEvBatch <= 64, "a stage holds whole 8-query tiles; its payload pieces are copied by 32 lanes x 4");

struct __align__(32) Payload {                       // one sector
    double a, b;                                     // class-dependent abscissae (t_x, t_q / theta / r)
    unsigned idx;                                    // query index inside its chunk
    unsigned cell;                                   // lists: x cell (low-Q, high-Q), Q2 cell (low-x), i | jg << 16 (overflow)
    double pad;
};

// geometry of the key space and the search tables; host copy in StreamPlan, passed by value
struct StreamDev {
    int ncx, nqt, nbins;                             // x cells, Q2 knots, cell bins (ncx * nqt; a last knot of a sub-grid owns an unused bin)
    int jgplus;                                      // cell (global lower-knot index) of 1.01*Q2min
    double tqplus;                                   // and its t_q  (C-9)
    int cap;                                         // payloads per cell bin
    int fku, ng, ne, tb;                             // Q2 cells per B unit, Q2-cell groups per x cell, E units per chunk, B + E units per chunk
    int xshift, xbase, nbx, qshift, qbase, nbq;      // bucket = (high word >> shift) - base
    const unsigned short *lutx, *lutq;               // [nbx], [nbq] cell at the lower edge of the bucket
    const double *rowplus;                           // [nmem][nx][12]: the grid's values at Q2 = 1.01 Q2min (C-9's second anchor), per x knot
};

struct StreamWorkspace {                             // carved out of the caller's workspace
    unsigned long long *ctrl;                        // [0] ticket; then per ring slot a_done, b_fin, b_done, each on a 128-byte line of its own
    unsigned *counts;                                // [kS3Ring][nbins + 32]: cell bins, then list counts [kNumLists] and list cursors [kNumLists]
    Payload *bins;                                   // [kS3Ring][nbins * cap]
    Payload *lists;                                  // [kS3Ring][kNumLists][chunk]
};
constexpr int kCtrlWords = 1024;                     // 8 KB control block
constexpr int kCtrlSlot0 = 32, kCtrlSlotStride = 48; // u64 words: 3 counters x 128 B per slot

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
    int count_err;             // 1: invalid queries bump the grid's error counter
    int q_is_q;                // 1: the q2 array holds Q (pdf_xfxq): squared on load
    // member axis (a-8, pdf_members.cuh): the queries arrive sorted by member and every chunk lies
    // inside one member's run; ctab[c] = {first query, queries, member, 0}, *nchunks_dev chunks.
    const int *ctab;
    const int *nchunks_dev;
    const unsigned *orig;      // with ctab: the query (row of `out`) of every sorted slot; the payload carries it
    // fused luminosity (a-7): pass 1 (k_lumi_first) writes rows [xf_0..xf_10, w/(x1 x2)] of 12 doubles into `out` (the
    // scratch), pass 2 (k_lumi_second) reads them back as `f1` and reduces the coupling against its own row on the fly
    const double *x2, *w;      // pass 1: the other parton's x and the event weight (for the scale column)
    const double *f1;          // pass 2: the rows of pass 1
    const double *coup;        // pass 2: C[i][j] as [12][16] doubles, zero padded
};
constexpr int kModeRows = 0, kModeLumiFirst = 1, kModeLumiSecond = 2;
constexpr int kCoupBytes = kNFP * 16 * 8;

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
// invalidates L1 (an acquire load or __threadfence emits CCTL.IVALL; with independent warps signalling every few
// microseconds that left no L1 for the grid values, and ~3000 warps spinning with acquire loads on one line
// starved the ticket and release atomics behind them: profile r2b, 90 % of the samples in the wait loops).
// That is sound here because everything another SM wrote during this launch (counters, payloads, list
// entries) is read through L2 (.cg / cp.async.cg), never through L1, and is only read after the poll that
// observed the release has returned (the loop exit depends on its value).
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
// called by all 32 lanes of a converged warp: lane 0 polls (one request per iteration), the warp leaves together
__device__ __forceinline__ void warp_wait(const unsigned long long *p, unsigned long long target)
{
    unsigned ns = 256;
    for (;;) {
        unsigned long long v = 0;
        if ((threadIdx.x & 31) == 0) v = ld_relaxed_u64(p);
        v = __shfl_sync(0xffffffffu, v, 0);
        if (v >= target) break;
        __nanosleep(ns);
        if (ns < 4096) ns <<= 1;
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
// the count of a chunk's finished units needs no fence: a unit only READ the slot (its counts have been consumed, its
// copies waited for) and wrote rows of `out` that nothing in this launch reads.  The unit that sees the full count
// zeroes the slot's counters and publishes that with a release (b_done).
__device__ __forceinline__ unsigned long long warp_count_add(unsigned long long *p, unsigned long long v)
{
    unsigned long long old = 0;
    __syncwarp();
    if ((threadIdx.x & 31) == 0)
        asm volatile("atom.add.relaxed.gpu.global.u64 %0, [%1], %2;" : "=l"(old) : "l"(p), "l"(v) : "memory");
    return __shfl_sync(0xffffffffu, old, 0);
}
// release without a returned value (A tiles): nothing waits for the atomic's round trip
__device__ __forceinline__ void warp_release_red(unsigned long long *p, unsigned long long v)
{
    __syncwarp();
    if ((threadIdx.x & 31) == 0) asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// one payload = one 32-byte sector, stored whole (STG.256): never a partial-sector write
__device__ __forceinline__ void store_payload(Payload *dst, double a, double b, unsigned idx, unsigned cell, double pad = 0.0)
{
    const double w2 = __hiloint2double((int)cell, (int)idx);       // low word idx, high word cell
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(dst), "d"(a), "d"(b), "d"(w2), "d"(pad) : "memory");
}
__device__ __forceinline__ void cp_async16_cg(unsigned saddr, const void *g)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(saddr), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async16_ca(unsigned saddr, const void *g)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(saddr), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }


// ---- a-2 on this path: region class and cell from the raw bit patterns ---------------------------
struct StreamTab {        // shared-window addresses of the tables staged once per CTA
    unsigned xk, qk, cx, cq, lutx, lutq;       // knots, cell tables (CellTab, 48 B each), search tables
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

// Out-of-line copies of the transcendental pieces of the E units: inlined, the library logarithms and the
// continuation formulas made the kernel 22 700 instructions (364 KB), and warps of three different work kinds
// per SM evicted one another's code from the instruction caches (~20 clk per issued instruction).
__device__ __noinline__ double s3_log(double v) { return pdf_log(v); }
__device__ __noinline__ double s3_two(double f0, double f1, double theta) { return continue_two(f0, f1, theta); }
__device__ __noinline__ double s3_lowq(double fmin, double fplus, double r, double lnr) { return lowq_continue_ln(fmin, fplus, r, lnr); }

// ---- A tile: classify, locate, t_x / t_q, one slot per query in its cell's bin -----------------
template <int MODE, bool OPT>
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
    unsigned *counts = A.W.counts + (size_t)slot * (B.nbins + 32);
    unsigned *lcount = counts + B.nbins;
    Payload *bins = A.W.bins + (size_t)slot * B.nbins * B.cap;
    Payload *lists = A.W.lists + (size_t)slot * kNumLists * A.chunk;
    const int nx = G.nx, nqt = G.nqtot;
    const long long xminb = lds_s64(T.xk), xmaxb = lds_s64(T.xk + 8u * (nx - 1));
    const long long qminb = lds_s64(T.qk), qmaxb = lds_s64(T.qk + 8u * (nqt - 1));
    const double u0 = __ldg(G.uk);
    // the extrapolation abscissae through reciprocals (one division each per tile instead of per query)
    const double inv_du0 = 1.0 / (__ldg(G.uk + 1) - u0);
    const double sA = __ldg(G.sk + nqt - 2), inv_ds = 1.0 / (__ldg(G.sk + nqt - 1) - sA);
    const double inv_qmin = 1.0 / __longlong_as_double(qminb);
    // The groups of kS3Grp queries per lane go through a software pipeline: the loads of group g + 1 are issued before
    // group g is located and its logarithms taken, and the payloads of group g are stored after group g + 1 has been
    // computed, so that the ~1 us of the input loads and the ~1-2 us of the slot atomics travel under arithmetic
    // instead of adding up per group (phase clocks of profile note r2c: 19.9 us per 256-query tile, 40 % of every
    // warp's time, with the four groups strictly one after the other).
    struct Grp { double xv[kS3Grp], qv[kS3Grp], sc[kS3Grp]; };
    struct Out { double pa[kS3Grp], pb[kS3Grp], sc[kS3Grp]; int key[kS3Grp]; unsigned cell[kS3Grp], pos[kS3Grp]; bool any_list; };
    auto load = [&](int g0) {
        Grp r;
#pragma unroll
        for (int q = 0; q < kS3Grp; ++q) {
            const long long e = t0 + (g0 + q) * 32 + lane;
            r.xv[q] = 1.0; r.qv[q] = 1.0; r.sc[q] = 0.0;
            if (e < t1) {
                r.xv[q] = __ldcs(A.x + e); r.qv[q] = __ldcs(A.q2 + e);
                if (MODE == kModeLumiFirst) r.sc[q] = __ldcs(A.w + e) / (r.xv[q] * __ldcs(A.x2 + e));   // f = xf / x on both sides (eq. 3.3): the query's own x
                // pdf_xfxq and the extrapolation options of L1720 (kernels of their own: even as two warp-uniform
                // branches that are never taken they cost the default kernel 0.58 ms per 1e8 queries)
                if (OPT) { if (A.q_is_q) r.qv[q] = q_to_q2(r.qv[q]); apply_extrapolation(G, r.xv[q], r.qv[q]); }
            }
        }
        return r;
    };
    // classify, locate, abscissae, and the slot atomics of the cell bins (in flight when this returns)
    auto compute = [&](const Grp &in, int g0) {
        Out o;
        Located L[kS3Grp];
#pragma unroll
        for (int q = 0; q < kS3Grp; ++q) L[q] = s3_locate(G, B, T, in.xv[q], in.qv[q], xminb, xmaxb, qminb, qmaxb);
        o.any_list = false;
#pragma unroll
        for (int q = 0; q < kS3Grp; ++q) {
            const long long e = t0 + (g0 + q) * 32 + lane;
            const int r = L[q].region;
            const bool lowx = r == kRegionLowX || r == kRegionLowXLowQ || r == kRegionLowXHighQ;
            const bool lowq = r == kRegionLowQ || r == kRegionLowXLowQ, highq = r == kRegionHighQ || r == kRegionLowXHighQ;
            const int i = L[q].i;
            const int jg = L[q].g < nqt - 1 ? L[q].g : nqt - 2;       // only Q2 == Q2max lands on the last knot: it belongs to the last cell
            const double2 ci = lds_v2f64(T.cx + 48u * i), cj = lds_v2f64(T.cq + 48u * jg);   // {ln lower knot, 1/dln}
            double lx = 0.0, lq = 0.0;
            if (r != kRegionInvalid) { lx = pdf_log(in.xv[q]); lq = pdf_log(in.qv[q]); }
            // t = 1 exactly on the last knot (the only knot that belongs to the cell on its left, C-4)
            o.pa[q] = lowx ? (lx - u0) * inv_du0                                    // theta_x (C-7)
                           : (__double_as_longlong(in.xv[q]) == xmaxb) ? 1.0 : (lx - ci.x) * ci.y;
            o.pb[q] = lowq ? in.qv[q] * inv_qmin                                    // r (C-9)
                    : highq ? (lq - sA) * inv_ds                                    // theta_q (C-8)
                            : (__double_as_longlong(in.qv[q]) == qmaxb) ? 1.0 : (lq - cj.x) * cj.y;
            o.sc[q] = in.sc[q];
            o.key[q] = r == kRegionInterior ? i * nqt + jg : -1 - r;               // region codes 1..5 are the list numbers
            o.cell[q] = r == kRegionInterior ? ((unsigned)i | ((unsigned)jg << 16)) : lowx ? (unsigned)jg : (unsigned)i;
            if (e >= t1 || r == kRegionInvalid) o.key[q] = INT_MIN;
            o.any_list |= o.key[q] < 0 && o.key[q] != INT_MIN;
        }
#pragma unroll
        for (int q = 0; q < kS3Grp; ++q) {
            o.pos[q] = 0u;
            if (o.key[q] >= 0) o.pos[q] = atomicAdd(counts + o.key[q], 1u);
        }
        return o;
    };
    // bin overflow, list slots, payload stores (reads the atomics' results)
    auto finish = [&](Out &o, int g0) {
#pragma unroll
        for (int q = 0; q < kS3Grp; ++q)
            if (o.key[q] >= 0 && o.pos[q] >= (unsigned)B.cap) { o.key[q] = -1 - kListOvf; o.any_list = true; }   // bin full: to the overflow list
        // list entries (extrapolated queries, bin overflow).  With a few entries per warp (C2: 5 % of the queries) one
        // atomic per entry is cheapest (the match.any reservation below costs ~50 warp instructions per query slot and
        // nearly every group of 64 has an entry); with many (C4: 25 % of the events take the low-Q2 list) the entries of
        // a warp reserve their run with ONE atomic per list, or the list's counter serialises them.
        if (__any_sync(0xffffffffu, o.any_list)) {
#pragma unroll
            for (int q = 0; q < kS3Grp; ++q) {
                const bool mine = o.key[q] < 0 && o.key[q] != INT_MIN;
                const unsigned act = __ballot_sync(0xffffffffu, mine);
                if (act == 0u) continue;
                if (__popc(act) <= 3) {
                    if (mine) o.pos[q] = atomicAdd(lcount + (-1 - o.key[q]), 1u);
                } else if (mine) {
                    const int k = -1 - o.key[q];
                    const unsigned peers = __match_any_sync(act, k);
                    const int leader = __ffs(peers) - 1;
                    unsigned base = 0;
                    if (lane == leader) base = atomicAdd(lcount + k, (unsigned)__popc(peers));
                    base = __shfl_sync(peers, base, leader);
                    o.pos[q] = base + (unsigned)__popc(peers & ((1u << lane) - 1u));
                }
            }
        }
#pragma unroll
        for (int q = 0; q < kS3Grp; ++q) {
            const long long e = t0 + (g0 + q) * 32 + lane;
            if (e >= t1) continue;
            const unsigned idx = A.orig ? __ldcs(A.orig + e) : (unsigned)(e - chunk_base);
            if (o.key[q] == INT_MIN) {                                              // C-10: NaN row, counted
                double *op = A.out + (A.orig ? (long long)idx : e) * A.ld;
                const int ncol = MODE == kModeLumiFirst ? kNFP : A.cm.n;
                for (int p = 0; p < ncol; ++p) op[p] = qnan();
                if (A.count_err) ++err_local;
            } else if (o.key[q] < 0) store_payload(lists + (size_t)(-1 - o.key[q]) * A.chunk + o.pos[q], o.pa[q], o.pb[q], idx, o.cell[q], o.sc[q]);
            else store_payload(bins + (size_t)o.key[q] * B.cap + o.pos[q], o.pa[q], o.pb[q], idx, o.cell[q], o.sc[q]);
        }
    };
    Grp next = load(0);
    Out prev;
    prev.any_list = false;
#pragma unroll
    for (int q = 0; q < kS3Grp; ++q) { prev.key[q] = INT_MIN; prev.pos[q] = 0u; prev.cell[q] = 0u; prev.pa[q] = prev.pb[q] = prev.sc[q] = 0.0; }
#pragma unroll 1
    for (int g0 = 0; g0 < kS3TileQ; g0 += kS3Grp) {
        const Grp cur = next;
        if (g0 + kS3Grp < kS3TileQ) next = load(g0 + kS3Grp);
        Out o = compute(cur, g0);
        if (g0 > 0) finish(prev, g0 - kS3Grp);
        prev = o;
    }
    finish(prev, kS3TileQ - kS3Grp);
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

// node weight number t of the 1-D Hermite operator in the factored form
//   w_t = (1-s)^2 (c0 + c1 s) + s^2 (c2 + c3 (1-s))        (same weights as hermite_weights)
struct WCoef { double c0, c1, c2, c3; };
__device__ __forceinline__ WCoef weight_coef(double aL, double bL, double aR, double bR, int t)
{
    WCoef w;
    w.c0 = t == 1 ? 1.0 : 0.0;
    w.c1 = t == 0 ? -bL : t == 1 ? 2.0 + bL - aL : t == 2 ? aL : 0.0;
    w.c2 = t == 2 ? 1.0 : 0.0;
    w.c3 = t == 1 ? aR : t == 2 ? 2.0 - aR + bR : t == 3 ? -bR : 0.0;
    return w;
}
__device__ __forceinline__ double weight_eval(const WCoef &w, double s)
{
    double om = 1.0 - s, om2 = om * om, s2 = s * s;
    return fma(om2, fma(w.c1, s, w.c0), s2 * fma(w.c3, om, w.c2));
}
// x node number t (0..3) of cell i: i-1 .. i+2, clamped at the ends of the knot line (x_point_cell)
__device__ __forceinline__ int xnode(int i, int t, int nx)
{
    const int c = i - 1 + t;
    return c < 0 ? 0 : (c >= nx ? nx - 1 : c);
}

// one row from the accumulator fragments through a column map: 4 lanes write one row (the general form; calls with the
// grid's own 11 columns in order take the four fixed stores in b_unit)
__device__ __forceinline__ void store_row(const StreamArgs &A, double *rp, int t, const Acc &d)
{
    for (int p = 0; p < A.cm.n; ++p) {
        const int c = A.cm.col[p];
        if (c < 0) { if (t == 0) rp[p] = 0.0; continue; }
        if (((c & 7) >> 1) == t) rp[p] = (c & 8) ? ((c & 1) ? d.d11 : d.d10) : ((c & 1) ? d.d01 : d.d00);
    }
}

// interior cells of x cell i, Q2 cells [fk0, fk1).  The unit is a stream of batches: <= kEvBatch payloads of ONE cell
// together with that cell's 16 node rows (node n = 4 * (Q2 row) + (x node)), copied by cp.async into one of the warp's
// kEvDepth self-contained stages [header | payloads | node rows].  The issuing side of the loop runs kEvDepth - 1
// batches ahead of the arithmetic (one commit group per loop turn, empty ones once the unit's cells are exhausted), so
// the ~1.5 us L2 latency of a batch is paid once per unit, not once per batch: with one batch in flight (versions 3
// and 4) a warp computed ~0.4 us per batch and waited ~1 us for the next (profile note r2c).
// The arithmetic of a tile (version 4, profile r2a: version 3 spent 108 warp instructions per 8-query tile, 8 of them
// DMMAs): the cell's operand fragments and the coefficients of both node weights are read once per batch and stay in
// registers, rows with the grid's own 11 columns (FAST) leave by four fixed stores from one 64-bit multiply-add, lanes
// beyond the batch run on whatever the stage holds (a row of A only ever meets its own row of D) and only their
// stores are predicated.
template <int MODE, bool FAST>
__device__ __forceinline__ void b_unit(const StreamArgs &A, const StreamTab &T, const double *__restrict__ Vm, int slot,
                                       long long chunk_base, int i, int fk0, int fk1, unsigned sbuf, unsigned sC,
                                       unsigned long long &err_local)
{
    const GridDev &G = A.G;
    const StreamDev &B = A.B;
    const int lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const unsigned *counts = A.W.counts + (size_t)slot * (B.nbins + 32) + (size_t)i * B.nqt;
    int mycnt = 0;
    if (fk0 + lane < fk1) mycnt = min((int)ldcg_u32(counts + fk0 + lane), B.cap);
    unsigned live = __ballot_sync(0xffffffffu, mycnt > 0);      // cells of the unit that hold queries
    if (live == 0u) return;
    const int nx = G.nx;
    const char *bin0 = reinterpret_cast<const char *>(A.W.bins + ((size_t)slot * B.nbins + (size_t)i * B.nqt) * B.cap);
    const unsigned capb = 32u * (unsigned)B.cap;
    const char *Vb = reinterpret_cast<const char *>(Vm);
    const unsigned rowb = (unsigned)(nx * kNFP * 8);
    int o = 0;                                                  // payloads of the current cell already issued
    // the next batch into stage `st`; an empty commit group behind a zero header once the cells are exhausted
    auto produce = [&](unsigned st) {
        if (live == 0u) {
            if (lane == 0) asm volatile("st.shared.v2.u32 [%0], {%1,%1};" ::"r"(st), "r"(0) : "memory");
            cp_async_commit();
            return;
        }
        const int j = __ffs(live) - 1, fk = fk0 + j;
        const int cntj = __shfl_sync(0xffffffffu, mycnt, j);
        const int n = min(kEvBatch, cntj - o);
        {
            // payloads: 2 n pieces of 16 bytes, contiguous in the bin
            const char *src = bin0 + ((size_t)(unsigned)fk * capb + 32u * (unsigned)o);
#pragma unroll
            for (int k = 0; k < (2 * kEvBatch + 31) / 32; ++k) {
                const int e = lane + 32 * k;
                if (e < 2 * n) cp_async16_cg(st + kEvHdr + 16u * e, src + 16 * e);
            }
        }
        {
            // the cell's 16 node rows: 96 pieces, piece e = lane + 32 k, node = e / 6 = 4 b + a (Q2 row b, x node a)
            const double aL = lds_f64(T.cq + 48u * fk + 16u), aR = lds_f64(T.cq + 48u * fk + 32u);
            const int elo = aL == 1.0 ? 1 : 0, ehi = aR == 1.0 ? 1 : 0;       // one-sided ends of a sub-grid (q_point_cell)
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const int e = lane + 32 * k, node = e / 6, piece = e - node * 6, b = node >> 2;
                const int row = fk - 1 + b + (b == 0 ? elo : 0) - (b == 3 ? ehi : 0);
                cp_async16_ca(st + kEvHdr + kEvBatch * 32 + 16u * e,
                              Vb + ((size_t)((unsigned)row * rowb) + (unsigned)((xnode(i, node & 3, nx) * kNFP + 2 * piece) * 8)));
            }
        }
        if (lane == 0) asm volatile("st.shared.v2.u32 [%0], {%1,%2};" ::"r"(st), "r"(n), "r"(fk) : "memory");
        cp_async_commit();
        o += n;
        if (o >= cntj) { live &= live - 1; o = 0; }
    };
    WCoef kx;
    {
        const double2 ab = lds_v2f64(T.cx + 48u * i + 16u), cd = lds_v2f64(T.cx + 48u * i + 32u);
        kx = weight_coef(ab.x, ab.y, cd.x, cd.y, t);            // x-axis weight of this lane's node, fixed for the unit
    }
    // pass 2 of the luminosity: the coupling's fragments (flavour 4 s + t of parton 1 against flavours g, 8 + g of parton 2)
    double cf0x = 0.0, cf0y = 0.0, cf1x = 0.0, cf1y = 0.0, cf2x = 0.0, cf2y = 0.0;
    if (MODE == kModeLumiSecond) {
        const unsigned pc = sC + (unsigned)(t * 128 + 8 * g);
        cf0x = lds_f64(pc); cf1x = lds_f64(pc + 512u); cf2x = lds_f64(pc + 1024u);
        if (g < 4) { cf0y = lds_f64(pc + 64u); cf1y = lds_f64(pc + 512u + 64u); cf2y = lds_f64(pc + 1024u + 64u); }
    }
    // rows of A.ld doubles, this lane's columns 2t, 2t+1 (all t), 8 + 2t (t < 2), 9 (t == 0)
    const unsigned ldb = (unsigned)(A.ld * 8);
    char *outl = reinterpret_cast<char *>(A.out + chunk_base * (MODE == kModeLumiFirst ? (long long)kNFP : A.ld)) + 16 * t;
#pragma unroll 1
    for (int k = 0; k < kEvDepth - 1; ++k) produce(sbuf + (unsigned)(k * kEvStage));
#pragma unroll 1
    for (unsigned seq = 0;; ++seq) {
        produce(sbuf + (unsigned)(((seq + kEvDepth - 1) % kEvDepth) * kEvStage));
        cp_async_wait<kEvDepth - 1>();
        __syncwarp();
        const unsigned st = sbuf + (unsigned)((seq % kEvDepth) * kEvStage);
        int n, fk;
        asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(n), "=r"(fk) : "r"(st));
        if (n == 0) break;
        WCoef kq;
        {
            const double2 ab = lds_v2f64(T.cq + 48u * fk + 16u), cd = lds_v2f64(T.cq + 48u * fk + 32u);
            kq = weight_coef(ab.x, ab.y, cd.x, cd.y, t);
        }
        // the cell's operand fragments: step r pairs Q2 row (t ^ r) with x node t; flavours g and 8 + g
        const unsigned sv = st + kEvHdr + kEvBatch * 32 + (unsigned)(t * kNFP * 8 + 8 * g);
        const double fb0 = lds_f64(sv + (unsigned)(4 * (t ^ 0) * kNFP * 8)), fb1 = lds_f64(sv + (unsigned)(4 * (t ^ 1) * kNFP * 8));
        const double fb2 = lds_f64(sv + (unsigned)(4 * (t ^ 2) * kNFP * 8)), fb3 = lds_f64(sv + (unsigned)(4 * (t ^ 3) * kNFP * 8));
        double fc0 = 0.0, fc1 = 0.0, fc2 = 0.0, fc3 = 0.0;
        if (g < 4) {
            fc0 = lds_f64(sv + (unsigned)(4 * (t ^ 0) * kNFP * 8) + 64u); fc1 = lds_f64(sv + (unsigned)(4 * (t ^ 1) * kNFP * 8) + 64u);
            fc2 = lds_f64(sv + (unsigned)(4 * (t ^ 2) * kNFP * 8) + 64u); fc3 = lds_f64(sv + (unsigned)(4 * (t ^ 3) * kNFP * 8) + 64u);
        }
        const unsigned sb = st + kEvHdr + 32u * g;
        // the next tile's abscissae are fetched under this tile's arithmetic
        double2 abn = lds_v2f64(sb);
        unsigned idxn = lds_u32(sb + 16u);
#pragma unroll 1
        for (int m0 = 0; m0 < n; m0 += 8) {
            const bool valid = m0 + g < n;
            const double tx = abn.x, tq = abn.y;
            const unsigned idx = idxn;
            const unsigned sn = sb + 32u * (unsigned)(m0 + 8 < kEvBatch ? m0 + 8 : 0);     // (the tile after the last is never used)
            abn = lds_v2f64(sn); idxn = lds_u32(sn + 16u);
            // pass 2 of the luminosity: this query's row of pass 1 in the A-operand layout (flavour 4 s + t), fetched
            // under the contraction; lane t = 3 of step 2 gets the scale column
            double a0 = 0.0, a1 = 0.0, a2 = 0.0;
            if (MODE == kModeLumiSecond && valid) {
                const double *fr = A.f1 + (chunk_base + idx) * kNFP + t;
                a0 = __ldcs(fr); a1 = __ldcs(fr + 4); a2 = __ldcs(fr + 8);
            }
            const double wx = weight_eval(kx, tx);
            const double wq0 = weight_eval(kq, tq);
            const double wq1 = __shfl_xor_sync(0xffffffffu, wq0, 1);
            const double wq2 = __shfl_xor_sync(0xffffffffu, wq0, 2);
            const double wq3 = __shfl_xor_sync(0xffffffffu, wq0, 3);
            Acc d = {0.0, 0.0, 0.0, 0.0};
            kstep(d, wq0 * wx, make_double2(fb0, fc0));
            kstep(d, wq1 * wx, make_double2(fb1, fc1));
            kstep(d, wq2 * wx, make_double2(fb2, fc2));
            kstep(d, wq3 * wx, make_double2(fb3, fc3));
            if (MODE == kModeRows) {
                if (FAST) {
                    if (valid) {
                        char *rp = outl + (size_t)idx * ldb;
                        asm volatile("st.global.f64 [%0], %1;" ::"l"(rp), "d"(d.d00) : "memory");
                        asm volatile("st.global.f64 [%0+8], %1;" ::"l"(rp), "d"(d.d01) : "memory");
                        if (t < 2) asm volatile("st.global.f64 [%0+64], %1;" ::"l"(rp), "d"(d.d10) : "memory");
                        if (t == 0) asm volatile("st.global.f64 [%0+72], %1;" ::"l"(rp), "d"(d.d11) : "memory");
                    }
                } else if (valid) store_row(A, A.out + (chunk_base + idx) * A.ld, t, d);
            } else if (MODE == kModeLumiFirst) {
                // rows of 12 on 32-byte sectors: two stores write the three sectors whole (no zero fill needed)
                if (valid) {
                    double *rp = reinterpret_cast<double *>(outl + (size_t)idx * (unsigned)(kNFP * 8));
                    *reinterpret_cast<double2 *>(rp) = make_double2(d.d00, d.d01);
                    if (t == 0) *reinterpret_cast<double2 *>(rp + 8) = make_double2(d.d10, d.d11);
                    if (t == 1) *reinterpret_cast<double2 *>(rp + 8) = make_double2(d.d10, lds_f64(sb + 32u * (unsigned)m0 + 24u));
                }
            } else {
                // G[q][j] = sum_i f1[q][i] C[i][j] by 6 more DMMAs, then the dot with this row and the scale
                Acc gq = {0.0, 0.0, 0.0, 0.0};
                kstep(gq, a0, make_double2(cf0x, cf0y));
                kstep(gq, a1, make_double2(cf1x, cf1y));
                kstep(gq, t == 3 ? 0.0 : a2, make_double2(cf2x, cf2y));
                double dot = fma(d.d00, gq.d00, fma(d.d01, gq.d01, fma(d.d10, gq.d10, d.d11 * gq.d11)));
                dot += __shfl_xor_sync(0xffffffffu, dot, 1);
                dot += __shfl_xor_sync(0xffffffffu, dot, 2);
                const double scale = __shfl_sync(0xffffffffu, a2, lane | 3);
                if (valid && t == 0) {
                    double v = scale * dot;
                    if (v != v && a0 != a0) { v = qnan(); if (A.count_err) ++err_local; }   // the x1 parton was invalid (C-10): counted once
                    A.out[chunk_base + idx] = v;
                }
            }
        }
        __syncwarp();                                           // the stage is free for the copies after next
    }
    cp_async_wait<0>();                                         // the empty groups behind the last batch
}

// ---- E units: the lists (extrapolation classes, bin overflow), one query per lane -----------------
// flavour pair p (columns 2p, 2p+1) of a node row; rows are 96 B = 6 pairs, the 12th column is a zero pad
__device__ __forceinline__ double2 ldpair(const double *__restrict__ row, int p) { return __ldg(reinterpret_cast<const double2 *>(row) + p); }

// the row of one list entry into `v[12]`.  Warp-uniform `list`; lanes differ in their cells.
//   kListLowQ  (C-9):  a = t_x, b = r;  anchors: row Q2min and the tabulated row at 1.01 Q2min, x cell `cell`
//   kListHighQ (C-8):  a = t_x, b = theta_q;  anchors: rows last-1 and last, x cell `cell`
//   kListLowX  (C-7):  a = theta_x, b = t_q;  anchors: columns X_0 and X_1 on the 4 rows of Q2 cell `cell`
//   corners (L1744): the x rule on both Q2 anchors, then the Q2 rule
//   kListOvf: a = t_x, b = t_q, cell = i | jg << 16: the full 16-node sum
__device__ __noinline__ void list_row(const StreamArgs &A, const double *__restrict__ Vm, const double *__restrict__ RPm, int list,
                                      double a, double b, unsigned cell, double v[kNFP])
{
    const GridDev &G = A.G;
    const int nx = G.nx, last = G.nqtot - 1;
    const size_t rs = (size_t)nx * kNFP;                       // doubles per Q2 row
    if (list == kListLowQ || list == kListHighQ) {
        const int i = (int)cell;
        double wx[4];
        hermite_weights(a, G.cx[i], wx);
        const double *r0 = list == kListLowQ ? Vm : Vm + (size_t)(last - 1) * rs;
        const double *r1 = list == kListLowQ ? RPm : Vm + (size_t)last * rs;
        const double lnr = list == kListLowQ ? s3_log(b) : 0.0;
        int xn[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) xn[k] = xnode(i, k, nx) * kNFP;
#pragma unroll
        for (int p = 0; p < 6; ++p) {
            double2 e0 = make_double2(0.0, 0.0), e1 = e0;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double2 u0 = ldpair(r0 + xn[k], p), u1 = ldpair(r1 + xn[k], p);
                e0.x = fma(wx[k], u0.x, e0.x); e0.y = fma(wx[k], u0.y, e0.y);
                e1.x = fma(wx[k], u1.x, e1.x); e1.y = fma(wx[k], u1.y, e1.y);
            }
            if (list == kListLowQ) { v[2 * p] = s3_lowq(e0.x, e1.x, b, lnr); v[2 * p + 1] = p < 5 ? s3_lowq(e0.y, e1.y, b, lnr) : 0.0; }
            else { v[2 * p] = s3_two(e0.x, e1.x, b); v[2 * p + 1] = p < 5 ? s3_two(e0.y, e1.y, b) : 0.0; }
        }
    } else if (list == kListLowX) {
        const int jg = (int)cell;
        const CellTab cq = G.cq[jg];
        double wq[4];
        hermite_weights(b, cq, wq);
        size_t qn[4];
        qn[0] = (size_t)((cq.aL == 1.0) ? jg : jg - 1) * rs; qn[1] = (size_t)jg * rs; qn[2] = (size_t)(jg + 1) * rs;
        qn[3] = (size_t)((cq.aR == 1.0) ? jg + 1 : jg + 2) * rs;
#pragma unroll
        for (int p = 0; p < 6; ++p) {
            double2 e0 = make_double2(0.0, 0.0), e1 = e0;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const double2 u0 = ldpair(Vm + qn[k], p), u1 = ldpair(Vm + qn[k] + kNFP, p);
                e0.x = fma(wq[k], u0.x, e0.x); e0.y = fma(wq[k], u0.y, e0.y);
                e1.x = fma(wq[k], u1.x, e1.x); e1.y = fma(wq[k], u1.y, e1.y);
            }
            v[2 * p] = s3_two(e0.x, e1.x, a); v[2 * p + 1] = p < 5 ? s3_two(e0.y, e1.y, a) : 0.0;
        }
    } else if (list == kListLowXLowQ || list == kListLowXHighQ) {
        const bool lq = list == kListLowXLowQ;
        const double *r0 = lq ? Vm : Vm + (size_t)(last - 1) * rs;
        const double *r1 = lq ? RPm : Vm + (size_t)last * rs;
        const double lnr = lq ? s3_log(b) : 0.0;
#pragma unroll
        for (int p = 0; p < 6; ++p) {
            const double2 u00 = ldpair(r0, p), u01 = ldpair(r0 + kNFP, p), u10 = ldpair(r1, p), u11 = ldpair(r1 + kNFP, p);
            const double lox = s3_two(u00.x, u01.x, a), hix = s3_two(u10.x, u11.x, a);
            v[2 * p] = lq ? s3_lowq(lox, hix, b, lnr) : s3_two(lox, hix, b);
            if (p < 5) {
                const double loy = s3_two(u00.y, u01.y, a), hiy = s3_two(u10.y, u11.y, a);
                v[2 * p + 1] = lq ? s3_lowq(loy, hiy, b, lnr) : s3_two(loy, hiy, b);
            } else v[2 * p + 1] = 0.0;
        }
    } else {
        const int i = (int)(cell & 0xffffu), jg = (int)(cell >> 16);
        const CellTab cq = G.cq[jg];
        double wx[4], wq[4];
        hermite_weights(a, G.cx[i], wx);
        hermite_weights(b, cq, wq);
        size_t qn[4];
        qn[0] = (size_t)((cq.aL == 1.0) ? jg : jg - 1) * rs; qn[1] = (size_t)jg * rs; qn[2] = (size_t)(jg + 1) * rs;
        qn[3] = (size_t)((cq.aR == 1.0) ? jg + 1 : jg + 2) * rs;
        int xn[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) xn[k] = xnode(i, k, nx) * kNFP;
#pragma unroll
        for (int p = 0; p < 6; ++p) {
            double2 acc = make_double2(0.0, 0.0);
#pragma unroll
            for (int bq = 0; bq < 4; ++bq) {
                double2 rb = make_double2(0.0, 0.0);
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const double2 u = ldpair(Vm + qn[bq] + xn[k], p);
                    rb.x = fma(wx[k], u.x, rb.x); rb.y = fma(wx[k], u.y, rb.y);
                }
                acc.x = fma(wq[bq], rb.x, acc.x); acc.y = fma(wq[bq], rb.y, acc.y);
            }
            v[2 * p] = acc.x; v[2 * p + 1] = acc.y;
        }
    }
}

// claims batches of 32 entries from the chunk's lists until they are drained
// pass 2 of the luminosity for a list entry: w/(x1 x2) sum_ij f1_i C_ij f2_j with C broadcast from shared memory
__device__ __noinline__ double list_lumi(const double *__restrict__ fr, unsigned sC, const double v[kNFP], bool &x1_invalid)
{
    double f1[kNFP];
#pragma unroll
    for (int p = 0; p < 6; ++p) { const double2 u = __ldcs(reinterpret_cast<const double2 *>(fr) + p); f1[2 * p] = u.x; f1[2 * p + 1] = u.y; }
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < kNF; ++i) {
        double row = 0.0;
#pragma unroll
        for (int j = 0; j < kNF; ++j) row = fma(lds_f64(sC + (unsigned)(i * 128 + 8 * j)), v[j], row);
        acc = fma(f1[i], row, acc);
    }
    x1_invalid = f1[0] != f1[0];
    return f1[11] * acc;
}

template <int MODE>
__device__ __forceinline__ void e_unit(const StreamArgs &A, const double *__restrict__ Vm, const double *__restrict__ RPm, int slot,
                                       long long chunk_base, unsigned sC, unsigned long long &err_local)
{
    const StreamDev &B = A.B;
    const int lane = threadIdx.x & 31;
    unsigned *lcount = A.W.counts + (size_t)slot * (B.nbins + 32) + B.nbins, *lcursor = lcount + kNumLists;
    const Payload *lists = A.W.lists + (size_t)slot * kNumLists * A.chunk;
    // lanes 0..5 hold the lists' lengths and claim for their list
    unsigned len = 0, claim = 0;
    if (lane < kNumLists) {
        len = ldcg_u32(lcount + lane);
        if (lane == kListOvf && len > (unsigned)A.chunk) len = (unsigned)A.chunk;
        claim = len ? atomicAdd(lcursor + lane, (unsigned)kS3Batch) : 0u;
    }
    for (;;) {
        const unsigned open = __ballot_sync(0xffffffffu, lane < kNumLists && claim < len);
        if (open == 0u) break;
        const int list = __ffs(open) - 1;
        const unsigned first = __shfl_sync(0xffffffffu, claim, list), n = __shfl_sync(0xffffffffu, len, list);
        if (lane == list) claim = atomicAdd(lcursor + lane, (unsigned)kS3Batch);      // the next claim travels under this batch
        const bool active = first + lane < n;
        double a = 0.5, b = 0.5;
        unsigned idx = 0, cell = 0;
        double pad = 0.0;
        if (active) {
            const Payload *e = lists + (size_t)list * A.chunk + first + lane;
            const double2 ab = __ldcg(reinterpret_cast<const double2 *>(e));
            const uint2 ic = __ldcg(reinterpret_cast<const uint2 *>(e) + 2);
            a = ab.x; b = ab.y; idx = ic.x; cell = ic.y;
            if (MODE == kModeLumiFirst) pad = __ldcg(reinterpret_cast<const double *>(e) + 3);
        }
        double v[kNFP];
        list_row(A, Vm, RPm, list, a, b, cell, v);
        if (MODE == kModeLumiFirst) {
            if (active) {
                double2 *o = reinterpret_cast<double2 *>(A.out + (chunk_base + idx) * kNFP);
                v[11] = pad;
#pragma unroll
                for (int p = 0; p < 6; ++p) o[p] = make_double2(v[2 * p], v[2 * p + 1]);
            }
        } else if (MODE == kModeLumiSecond) {
            if (active) {
                bool bad;
                double r = list_lumi(A.f1 + (chunk_base + idx) * kNFP, sC, v, bad);
                if (bad) { r = qnan(); if (A.count_err) ++err_local; }                     // the x1 parton was invalid (C-10): counted once
                A.out[chunk_base + idx] = r;
            }
        } else if (active) {
            double *o = A.out + (chunk_base + idx) * A.ld;
            if (A.identity) {
#pragma unroll
                for (int f = 0; f < kNF; ++f) o[f] = v[f];
            } else {
                for (int p = 0; p < A.cm.n; ++p) {
                    const int c = A.cm.col[p];
                    double w = 0.0;
#pragma unroll
                    for (int f = 0; f < kNF; ++f) w = c == f ? v[f] : w;
                    o[p] = w;
                }
            }
        }
    }
}

// ---- the persistent kernel -----------------------------------------------------------------------
// dynamic shared memory: [x knots | Q2 knots | x cell tables | Q2 cell tables | lutx | lutq | per-warp stages]
__host__ __device__ inline size_t s3_table_bytes(int nx, int nqt, int nbx, int nbq)
{
    size_t b = sizeof(double) * (size_t)(nx + nqt) + sizeof(CellTab) * (size_t)(nx + nqt) + 2u * (size_t)(nbx + nbq);
    return (b + 31) / 32 * 32 + 64;                      // + alignment slack of the 16-byte aligned cell tables
}
__device__ __forceinline__ StreamTab s3_stage_tables(const GridDev &G, const StreamDev &B, unsigned char *smem, int nthreads)
{
    double *s_xk = reinterpret_cast<double *>(smem);
    double *s_qk = s_xk + G.nx;
    double *s_cx = s_qk + G.nqtot + ((G.nx + G.nqtot) & 1);      // 16-byte aligned
    double *s_cq = s_cx + 6 * G.nx;
    unsigned short *s_lx = reinterpret_cast<unsigned short *>(s_cq + 6 * G.nqtot);
    unsigned short *s_lq = s_lx + B.nbx;
    for (int k = threadIdx.x; k < G.nx; k += nthreads) s_xk[k] = G.xk[k];
    for (int k = threadIdx.x; k < G.nqtot; k += nthreads) s_qk[k] = G.qk[k];
    for (int k = threadIdx.x; k < 6 * B.ncx; k += nthreads) s_cx[k] = reinterpret_cast<const double *>(G.cx)[k];
    for (int k = threadIdx.x; k < 6 * G.nqtot; k += nthreads) s_cq[k] = reinterpret_cast<const double *>(G.cq)[k];
    for (int k = threadIdx.x; k < B.nbx; k += nthreads) s_lx[k] = B.lutx[k];
    for (int k = threadIdx.x; k < B.nbq; k += nthreads) s_lq[k] = B.lutq[k];
    StreamTab T;
    T.xk = (unsigned)__cvta_generic_to_shared(s_xk); T.qk = (unsigned)__cvta_generic_to_shared(s_qk);
    T.cx = (unsigned)__cvta_generic_to_shared(s_cx); T.cq = (unsigned)__cvta_generic_to_shared(s_cq);
    T.lutx = (unsigned)__cvta_generic_to_shared(s_lx); T.lutq = (unsigned)__cvta_generic_to_shared(s_lq);
    return T;
}

// pdf_locate on this path: the search the evaluation kernel runs, exported (ix, iq local to the sub-grid)
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
        double xe = x[e], qe = q2[e];
        apply_extrapolation(G, xe, qe);
        const Located L = s3_locate(G, B, T, xe, qe, xminb, xmaxb, qminb, qmaxb);
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

template <int MODE, bool FAST, bool OPT>
__device__ __forceinline__ void stream_body(const StreamArgs &A)
{
    extern __shared__ __align__(32) unsigned char smem_raw[];
    const StreamTab T = s3_stage_tables(A.G, A.B, smem_raw, kS3Threads);
    const unsigned stage0 = (unsigned)__cvta_generic_to_shared(smem_raw) + (unsigned)s3_table_bytes(A.G.nx, A.G.nqtot, A.B.nbx, A.B.nbq);
    __syncthreads();                                   // the only CTA barrier: every warp works alone from here on
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned sbuf = ((stage0 + 31u) & ~31u) + (unsigned)(warp * kStageBytes);
    const unsigned sC = ((stage0 + 31u) & ~31u) + (unsigned)(kS3Warps * kStageBytes);       // the coupling table (pass 2)
    if (MODE == kModeLumiSecond) {
        for (int k = threadIdx.x; k < kCoupBytes / 8; k += kS3Threads)
            asm volatile("st.shared.f64 [%0], %1;" ::"r"(sC + 8u * k), "d"(__ldg(A.coup + k)) : "memory");
        __syncthreads();
    }

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

    // A ticket is fetched when the warp is free to start it, not earlier: a prefetched ticket sits unstarted behind
    // the holder's current item and its waits, which doubles the window of unfinished tickets that the lag and the
    // ring have to cover (measured: with prefetch B units waited 29 us on average even at lag 3).
    for (;;) {
        unsigned long long t = 0;
        if (lane == 0) t = atomicAdd(ctrl, 1ULL);
        t = __shfl_sync(0xffffffffu, t, 0);
        if (t >= total) break;
        // ticket order, lag L = kS3Lag rounds:  round r = [A(r) tiles | E(r-L), B(r-L) units]
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
        unsigned long long *a_done = ctrl + kCtrlSlot0 + slot * kCtrlSlotStride, *b_fin = a_done + 16, *b_done = a_done + 32;
        long long chunk_base = c * A.chunk, chunk_end = chunk_base + A.chunk;
        if (chunk_end > A.n) chunk_end = A.n;
        const double *V = A.G.V, *RP = B.rowplus;
        if (A.ctab) {                                              // a-8: the chunk is a piece of one member's run
            const int4 ce = __ldg(reinterpret_cast<const int4 *>(A.ctab) + c);
            chunk_base = ce.x; chunk_end = (long long)ce.x + ce.y;
            V += (size_t)ce.z * A.G.memstride;
            RP += (size_t)ce.z * A.G.nx * kNFP;
        }
        if (isA) {
            // the ring slot must have been drained by the units of chunk c - kS3Ring before this tile touches its bins
            if (gen) wait_for(b_done, gen * TB);
            a_tile<MODE, OPT>(A, T, slot, chunk_base, chunk_end, sub, err_local);
            warp_release_red(a_done, 1ULL);
        } else {
            wait_for(a_done, (gen + 1) * TA);                      // every tile of A(c) has been released
            const long long row_base = A.orig ? 0 : chunk_base;    // member axis: the payload's index is the row itself
            if (sub < B.ne) e_unit<MODE>(A, V, RP, slot, row_base, sC, err_local);   // list units first: their queries are the expensive ones
            else {
                const int v = sub - B.ne;
                const int i = v / B.ng, grp = v - i * B.ng;
                b_unit<MODE, FAST>(A, T, V, slot, row_base, i, grp * B.fku, min(B.nqt, (grp + 1) * B.fku), sbuf, sC, err_local);
            }
            const unsigned long long old = warp_count_add(b_fin, 1ULL);
            if (old + 1 == (gen + 1) * TB) {                       // last unit of the chunk: the slot's counters are reset for the ring
                unsigned *cz = A.W.counts + (size_t)slot * (B.nbins + 32);
                for (int k = lane; k < B.nbins + 32; k += 32) cz[k] = 0u;
                warp_release_add(b_done, TB);
            }
        }
    }
    if (err_local) atomicAdd(A.G.err_count, err_local);
}

// k_pdf_stream: rows of the grid's own 11 columns in order (any leading dimension below 2^29 doubles); k_pdf_stream_cols:
// any column list (pid subsets, repeated or unknown pids)
__global__ void __launch_bounds__(kS3Threads, PDF_S3_MINB) k_pdf_stream(const __grid_constant__ StreamArgs A) { stream_body<kModeRows, true, false>(A); }
__global__ void __launch_bounds__(kS3Threads, PDF_S3_MINB) k_pdf_stream_cols(const __grid_constant__ StreamArgs A) { stream_body<kModeRows, false, false>(A); }
__global__ void __launch_bounds__(kS3Threads, PDF_S3_MINB) k_lumi_first(const __grid_constant__ StreamArgs A) { stream_body<kModeLumiFirst, false, false>(A); }
__global__ void __launch_bounds__(kS3Threads, PDF_S3_MINB) k_lumi_second(const __grid_constant__ StreamArgs A) { stream_body<kModeLumiSecond, false, false>(A); }
// the same with pdf_xfxq's Q -> Q2 and the extrapolation options of L1720 applied where an A tile loads its queries
__global__ void __launch_bounds__(kS3Threads, PDF_S3_MINB) k_pdf_stream_opt(const __grid_constant__ StreamArgs A) { stream_body<kModeRows, false, true>(A); }
__global__ void __launch_bounds__(kS3Threads, PDF_S3_MINB) k_lumi_first_opt(const __grid_constant__ StreamArgs A) { stream_body<kModeLumiFirst, false, true>(A); }
__global__ void __launch_bounds__(kS3Threads, PDF_S3_MINB) k_lumi_second_opt(const __grid_constant__ StreamArgs A) { stream_body<kModeLumiSecond, false, true>(A); }

__host__ __device__ inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace pdfg

#include "pdf_members.cuh"
#include "pdf_stream_host.cuh"
