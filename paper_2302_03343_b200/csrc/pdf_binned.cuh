// pdf_binned.cuh -- the binned, warp-coherent evaluation path (PDF_PATH_BINNED).
//
// Why: a query needs a 4x4 stencil x 11 flavours = 1408 B of grid data.  With unsorted queries
// every lane gathers its own stencil and the L1/L2 request rate, not HBM or the FP64 pipe, bounds
// the kernel (the direct path sits at ~1 % of the HBM roofline).  Here queries are first binned
// by cell, so that the 32 lanes of a warp share ONE stencil: each 16-byte load of grid data is a
// single broadcast wavefront that serves 32 queries.
//
// How (B200-first): ONE persistent kernel per call, one CTA slot per SM x occupancy, pulling
// work items from a global ticket counter.  The n queries are cut in chunks small enough that a
// chunk's bins (32 B/query) and its scattered output rows stay in the 126 MB L2, so HBM sees
// ~16 B/query in and 88 B/query out and nothing else.  Two item kinds alternate in ticket order
//      A(c):  read x,q2 of a tile of chunk c (coalesced), classify, locate the cell, compute
//             t_x,t_q (the two logs), claim a slot in the cell's bin (L2 atomic), write payload
//      B(c):  for a group of 32 cells: warps take batches of 32 payloads of one cell, build the
//             Hermite weights, run the 16-node x 11-flavour FMA sum with broadcast loads,
//             transpose through shared memory and write whole 88-byte rows
// in the order A(0) A(1) B(0) A(2) B(1) ...  B(c) waits (acquire-spin on a counter) until every
// tile of A(c) has been released; by ticket order those tiles were claimed a whole stage earlier,
// so the wait is normally zero and can never deadlock (all CTAs are co-resident; a ticket only
// ever waits on lower tickets).  Bins live in a ring of R chunk slots.
// Extrapolation classes (SURVEY a-5) get their own keys, so a warp is class-uniform.
// Queries that do not fit their bin (capacity CAP per chunk) go to an overflow list that the
// generic per-thread code evaluates; correctness never depends on the distribution.
#pragma once
#include "pdf_common.cuh"
#include "pdf_generic.cuh"

namespace pdfg {

constexpr int kBinThreads = 256;              // CTA size of the persistent kernel
constexpr int kBinWarps = kBinThreads / 32;
constexpr int kTileQ = 8;                     // queries per thread in an A item
constexpr int kTileA = kBinThreads * kTileQ;  // 2048 queries per A item
constexpr int kKeysPerItem = 32;              // keys per B item (one per lane in the prologue scan)
constexpr int kOvfItems = 8;                  // B items per chunk that drain the overflow list
constexpr int kRing = 3;                      // chunk slots in flight
constexpr int kCornerSub = 4;                 // sub-keys of each corner class (spreads heavy math)
constexpr int kLutSize = 1024;                // search-acceleration buckets per axis
constexpr int kNF = 11, kNFP = 12;            // the fast path is specialised for 11 flavours (pad 12)

struct __align__(32) Payload {                // one sector
    double a, b;                              // class-dependent abscissae (t_x,t_q / theta / r)
    unsigned idx;                             // query index inside its chunk
    unsigned pad0;
    double pad1;
};

struct BinItem { int key_begin, key_end; };  // key_begin < 0: overflow item number -key_begin-1

// geometry of the key space and the work list; host copy in BinnedPlan, device copy in BinDev
struct BinDev {
    int ncx, nqt, nkeys;
    int k_lowx, k_highq, k_lowq, k_ll, k_lh;  // first key of each class (interior starts at 0)
    int jgplus;                               // cell (global lower-knot index) of 1.01*Q2min
    double tqplus;                            // and its t_q  (C-9)
    int nitems;                               // B items per chunk, overflow items included
    const BinItem *items;                     // [nitems]
    const short *lutx, *lutq;                 // [kLutSize] start guesses of the knot search
    double lutx_scale, lutq_scale;            // buckets per unit of ln x / ln Q2
};

struct BinnedPlan {
    bool usable = false;
    BinDev dev{};
    BinItem *d_items = nullptr;
    short *d_lutx = nullptr, *d_lutq = nullptr;
    double *d_plus = nullptr;                 // scratch of k_q2plus
    int max_ctas = 0;                         // co-resident CTAs of the persistent kernel
    long long default_chunk = 1 << 19;
};

struct BinWorkspace {                         // carved out of the caller's workspace
    unsigned long long *ctrl;                 // [0] ticket, [1] error count; then per ring slot: a_done, b_done
    unsigned *counts;                         // [kRing][nkeys]
    unsigned *ovf_count;                      // [kRing]
    Payload *bins;                            // [kRing][nkeys][cap]
    Payload *ovf;                             // [kRing][chunk]
};

inline long long binned_chunk(const BinnedPlan &p, long long n, long long chunk_opt)
{
    long long c = chunk_opt > 0 ? chunk_opt : p.default_chunk;
    c = (c + kTileA - 1) / kTileA * kTileA;
    long long need = (n + kTileA - 1) / kTileA * kTileA;
    if (need < kTileA) need = kTileA;
    return c < need ? c : need;
}

inline int binned_cap(long long chunk)
{
    // bin capacity per chunk: a uniform cloud puts ~chunk/9000 queries in a cell of the LHAPDF-shaped
    // grid (58 at 512k); 4x that (min 32, max 256) keeps overflow to genuinely skewed inputs
    long long c = chunk / 2048;
    if (c < 32) c = 32;
    if (c > 256) c = 256;
    return (int)c;
}

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

inline size_t binned_workspace_bytes(const BinnedPlan &p, long long n, long long chunk_opt)
{
    if (!p.usable) return 0;
    long long chunk = binned_chunk(p, n, chunk_opt);
    int cap = binned_cap(chunk);
    size_t b = 4096;                                                    // ctrl
    b += align_up(sizeof(unsigned) * (size_t)kRing * p.dev.nkeys, 256);
    b += 256;                                                           // ovf_count
    b += align_up(sizeof(Payload) * (size_t)kRing * p.dev.nkeys * cap, 256);
    b += align_up(sizeof(Payload) * (size_t)kRing * chunk, 256);
    return b + 256;
}

inline void binned_carve(const BinnedPlan &p, void *ws, long long chunk, int cap, BinWorkspace &w)
{
    char *c = (char *)align_up((size_t)ws, 256);
    w.ctrl = (unsigned long long *)c; c += 4096;
    w.counts = (unsigned *)c; c += align_up(sizeof(unsigned) * (size_t)kRing * p.dev.nkeys, 256);
    w.ovf_count = (unsigned *)c; c += 256;
    w.bins = (Payload *)c; c += align_up(sizeof(Payload) * (size_t)kRing * p.dev.nkeys * cap, 256);
    w.ovf = (Payload *)c;
    (void)chunk;
}

}  // namespace pdfg

#include "pdf_binned_kernel.cuh"
#include "pdf_binned_host.cuh"
