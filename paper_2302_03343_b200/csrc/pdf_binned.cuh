// pdf_binned.cuh -- the binned, warp-coherent evaluation path (PDF_PATH_BINNED), version 2.
//
// Why: a query needs a 4x4 stencil x 11 flavours = 1408 B of grid data.  Gathered per lane that
// is >= 12 clk/query/SM of L1 / shared-memory bandwidth, 2.5x the HBM and FP64 budgets, so the
// lanes of a warp must share a cell: its values then come from shared memory as tensor-pipe
// fragments (interior cells) or broadcast operands (LDS.128 with one address: 1.5 clk).  With ~10^4 cells that needs a sort domain of >= 10^5
// queries, which no CTA holds on chip: queries are binned through L2 in chunks.
//
// What the machine dictates (measured on this B200):
//   * one global atomic + one scattered store per query costs a whole roofline budget
//       -> A items sort their tile by COARSE key (the x-cell) in shared memory, reserve one run
//          per (tile, key) with a single global atomic, and store each 32-byte payload as one
//          whole sector (STG.256);
//   * unaligned 88-byte rows scattered into untouched memory reach 0.9 TB/s (partial sectors)
//       -> A items first ZERO-FILL the output rows of their tile with coalesced stores; the later
//          scattered row stores of B then merge into valid L2-resident sectors (2.7 ms -> in
//          budget), and every line still leaves L2 for HBM once.
//
// How: ONE persistent kernel per call, CTAs pull tickets in the order (lag kLag = 3 rounds)
//      round r = [ A(r) tiles | B(r-3) items ]
//   A(c), one item per 2048 queries of chunk c: read x,q2 (coalesced), classify, locate the cell (a thread
//      takes its queries through the steps in groups of 2, so that loads and logarithms overlap),
//      t_x,t_q (the two logs), coarse/fine key, tile-local counting sort by coarse key, payload
//      stores; zero-fill of the tile's output rows.
//   B(c), one item per coarse key: copy the key's payloads and its 4 grid columns (4 x nq x 96 B)
//      to shared memory, counting-sort by FINE key (the Q2 cell or the extrapolation class), then
//      warps take batches of <= 32 same-cell queries.  Interior cells: FP64 mma.sync (DMMA m8n8k4)
//      tiles of 8 queries x 8 flavours over the 16 nodes, rows stored straight from the accumulator
//      fragments.  Extrapolation classes: one query per lane with broadcast LDS.128 operands.
// B(c) waits (acquire-spin by one whole warp) until every tile of A(c) has been released; by
// ticket order those tiles were claimed three rounds earlier, so the wait is normally zero and
// cannot deadlock (all CTAs are co-resident; a ticket only waits on lower tickets).  Bins live in
// a ring of kRing chunk slots.  Queries that do not fit their bin (capacity per chunk and key) go
// to an overflow list that the generic per-thread code evaluates: correctness never depends on
// the distribution.
#pragma once
#include "pdf_common.cuh"
#include "pdf_generic.cuh"

namespace pdfg {

#ifndef PDF_BINTHREADS
#define PDF_BINTHREADS 256
#endif
constexpr int kBinThreads = PDF_BINTHREADS;   // CTA size of the persistent kernel
constexpr int kBinWarps = kBinThreads / 32;
#ifndef PDF_TILEQ
#define PDF_TILEQ 8
#endif
#ifndef PDF_MINB
#define PDF_MINB 2
#endif
#ifndef PDF_LAG
#define PDF_LAG 3
#endif
constexpr int kTileQ = PDF_TILEQ;                     // queries per thread in an A item
constexpr int kTileA = kBinThreads * kTileQ;  // 2048 queries per A item (1024: 10.76, 1536: 10.26, 2048: 10.22, 3072: 10.21 ms)
constexpr int kOvfItems = 4;                  // B items per chunk that drain the overflow list
constexpr int kLag = PDF_LAG;                       // B(c) tickets follow A(c) tickets by this many rounds
#ifndef PDF_RING_EXTRA
#define PDF_RING_EXTRA 4
#endif
constexpr int kRing = kLag + PDF_RING_EXTRA;  // chunk slots in flight: A(c) reuses the slot of B(c-kRing), issued >= 2 rounds earlier
constexpr int kLowXBands = 16;                // coarse keys of low-x queries with Q2 inside: bands of Q2 cells
constexpr int kCornerSplit = 8;               // coarse keys per corner class (low-x and low-Q / high-Q): their rows cost
                                              // ~100 transcendental calls, one item of 650 of them held its ring slot 130 us
constexpr int kLowXSplit = kLowXBands + 2 * kCornerSplit;
constexpr int kLutSize = 1024;                // search-acceleration buckets per axis
constexpr int kNF = 11, kNFP = 12;            // the fast path is specialised for 11 flavours (pad 12)
constexpr int kMaxCK = 1024;                  // coarse keys (x cells + kLowXSplit) the path supports
constexpr int kMaxFK = 96;                    // fine keys (Q2 knots + 2)
#ifndef PDF_MAXCAP
#define PDF_MAXCAP 2048
#endif
constexpr int kMaxCap = PDF_MAXCAP;                 // payloads of one (chunk, coarse key) held in shared memory

struct __align__(32) Payload {                // one sector
    double a, b;                              // class-dependent abscissae (t_x,t_q / theta / r)
    unsigned idx;                             // query index inside its chunk
    unsigned fk;                              // fine key
    double pad;
};

// geometry of the key space; host copy in BinnedPlan, device copy passed by value
struct BinDev {
    int ncx, nqt, nck, nfk;                   // x cells, Q2 knots, coarse keys, fine keys
    int jgplus;                               // cell (global lower-knot index) of 1.01*Q2min
    double tqplus;                            // and its t_q  (C-9)
    int nitems;                               // B items per chunk, overflow items included
    const short *lutx, *lutq;                 // [kLutSize] start guesses of the knot search
    double lutx_scale, lutq_scale;            // buckets per unit of ln x / ln Q2
};

struct BinnedPlan {
    bool usable = false;
    BinDev dev{};
    short *d_lutx = nullptr, *d_lutq = nullptr;
    double *d_plus = nullptr;                 // scratch of k_q2plus
    int max_ctas = 0;                         // co-resident CTAs of the persistent kernel
    long long default_chunk = 352 * 1024;     // measured (C2, n = 1e8): 192k 12.2, 256k 11.2, 320k 11.1, 352k 10.95, 384k 11.1 ms;
                                              // 352k/195 cells + 4.6 sigma is what one shared-memory segment (kMaxCap) holds
};

struct BinWorkspace {                         // carved out of the caller's workspace
    unsigned long long *ctrl;                 // [0] ticket; then per ring slot: a_done, b_fin, b_done
    unsigned *counts;                         // [kRing][nck]
    unsigned *ovf_count;                      // [kRing]
    Payload *bins;                            // [kRing][nck][cap]
    Payload *ovf;                             // [kRing][chunk]  (raw x, q2)
};

inline long long binned_chunk(const BinnedPlan &p, long long n, long long chunk_opt)
{
    long long c = chunk_opt > 0 ? chunk_opt : p.default_chunk;
    c = (c + kTileA - 1) / kTileA * kTileA;
    long long need = (n + kTileA - 1) / kTileA * kTileA;
    if (need < kTileA) need = kTileA;
    return c < need ? c : need;
}

// shared-memory segment of a B item: a uniform cloud puts chunk/ncx queries on an x cell (1344 at
// 256k and 195 cells, 1848 at the default 352k); 1.125x that + 96, capped at kMaxCap, lets such a bin go
// through in one segment
inline int binned_scap(const BinnedPlan &p, long long chunk)
{
    long long c = chunk / (p.dev.ncx > 0 ? p.dev.ncx : 1);
    c = c + c / 8 + 96;
    c = (c + 31) / 32 * 32;
    if (c > kMaxCap) c = kMaxCap;
    return (int)c;
}
// bin capacity in the workspace: 4x the uniform share, so that narrower clouds (configs[4] covers
// 2/3 of the x range; VEGAS-like peaks) still bin; beyond it queries overflow to the generic path
inline int binned_cap(const BinnedPlan &p, long long chunk)
{
    long long c = 4 * (chunk / (p.dev.ncx > 0 ? p.dev.ncx : 1)) + 256;
    c = (c + 31) / 32 * 32;
    if (c > chunk) c = chunk;
    if (c < binned_scap(p, chunk)) c = binned_scap(p, chunk);
    return (int)c;
}

__host__ __device__ inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

inline size_t binned_workspace_bytes(const BinnedPlan &p, long long n, long long chunk_opt)
{
    if (!p.usable) return 0;
    long long chunk = binned_chunk(p, n, chunk_opt);
    int cap = binned_cap(p, chunk);
    size_t b = 4096;                                                    // ctrl
    b += align_up(sizeof(unsigned) * (size_t)kRing * p.dev.nck, 256);
    b += 256;                                                           // ovf_count
    b += align_up(sizeof(Payload) * (size_t)kRing * p.dev.nck * cap, 256);
    b += align_up(sizeof(Payload) * (size_t)kRing * chunk, 256);
    return b + 256;
}

inline void binned_carve(const BinnedPlan &p, void *ws, long long chunk, int cap, BinWorkspace &w)
{
    char *c = (char *)align_up((size_t)ws, 256);
    w.ctrl = (unsigned long long *)c; c += 4096;
    w.counts = (unsigned *)c; c += align_up(sizeof(unsigned) * (size_t)kRing * p.dev.nck, 256);
    w.ovf_count = (unsigned *)c; c += 256;
    w.bins = (Payload *)c; c += align_up(sizeof(Payload) * (size_t)kRing * p.dev.nck * cap, 256);
    w.ovf = (Payload *)c;
    (void)chunk;
}

}  // namespace pdfg

#include "pdf_binned_kernel.cuh"
#include "pdf_members.cuh"
#include "pdf_binned_host.cuh"
