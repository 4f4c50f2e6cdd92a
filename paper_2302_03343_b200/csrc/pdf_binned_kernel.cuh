// pdf_binned_kernel.cuh -- device code of the persistent binned kernel: helpers and A items
// (see pdf_binned.cuh for the design).
#pragma once

#ifdef PDF_CHECKS
#include <assert.h>
#endif

namespace pdfg {

#ifdef PDF_CHECKS
#define PDF_ASSERT(c) assert(c)
#else
#define PDF_ASSERT(c) ((void)0)
#endif

// phase clocks of thread 0 (development builds only, -DPDF_PHASES): ctrl[256 + k] += cycles
#ifdef PDF_PHASES
#define PH_DECL long long ph_t = clock64()
#define PH(k) do { if (threadIdx.x == 0) { long long ph_n = clock64(); atomicAdd(A.W.ctrl + 256 + (k), (unsigned long long)(ph_n - ph_t)); ph_t = ph_n; } } while (0)
#else
#define PH_DECL ((void)0)
#define PH(k) ((void)0)
#endif

struct StreamArgs {
    GridDev G;
    BinDev B;
    ColMap cm;
    BinWorkspace W;
    const double *x, *q2;      // a-2..a-5 inputs (pdf_xfxq2)
    double *out;
    long long n, ld;
    long long chunk;           // queries per chunk (multiple of kTileA)
    int nchunks, ta, cap;      // chunks, A items per chunk, bin capacity per (chunk, coarse key)
    int scap;                  // payloads a B item holds in shared memory at a time (segment size)
    int identity;              // 1: requested columns == the grid's 11 columns in order
    int zfill;                 // 1: rows are contiguous (ld == npid): A items zero-fill their tile of `out`
    int count_err;             // 1: invalid queries bump the grid's error counter (0 inside pdf_lumi)
    // member axis (a-8, pdf_members.cuh): the queries arrive sorted by member and every chunk lies
    // inside one member's run; ctab[c] = {first query, queries, member, 0}, *nchunks_dev chunks.
    // Null for the plain path (chunk c = queries [c*chunk, (c+1)*chunk), member 0).
    const int *ctab;
    const int *nchunks_dev;
};

// ---- small device helpers ----------------------------------------------------------------------
// CTA barrier of this kernel.  The shared-memory traffic around it is issued through inline PTX
// (st.shared / atom.shared / ld.shared with explicit shared-window addresses); without the block
// fence a warp was observed to read counters after the barrier that the other warps' atom.shared
// had not finished updating (cold launches, 80-register builds).  The fence makes every prior
// shared-memory operation of the warp performed before it arrives; cost: one MEMBAR.CTA.
__device__ __forceinline__ void cta_sync()
{
    __threadfence_block();
    __syncwarp();
    __syncthreads();
}

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long *p)
{
    unsigned long long v;
#ifdef PDF_RELAXED_POLL
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
#else
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
#endif
    return v;
}

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned *p)
{
    unsigned v;
#ifdef PDF_RELAXED_POLL
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
#else
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
#endif
    return v;
}

// called by all 32 lanes of one warp (converged): lane 0's view decides, so the warp leaves the loop together
__device__ __forceinline__ void wait_counter(const unsigned long long *p, unsigned long long target)
{
    unsigned ns = 32;
    for (;;) {
        unsigned long long v = ld_acquire_u64(p);
        v = __shfl_sync(0xffffffffu, v, 0);
        if (v >= target) break;
        __nanosleep(ns);
        if (ns < 1024) ns <<= 1;
    }
}

// one payload = one 32-byte sector, stored whole (STG.256): never a partial-sector write
__device__ __forceinline__ void store_payload(Payload *dst, double a, double b, unsigned idx, unsigned fk)
{
    double w2 = __hiloint2double((int)fk, (int)idx);       // low word idx, high word fk
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(dst), "d"(a), "d"(b), "d"(w2), "d"(0.0) : "memory");
}

// knot search from a LUT guess; exact for any knots (walks to the C-4 cell from wherever it starts)
__device__ __forceinline__ int search_cell(const double *__restrict__ k, int m, double v, int guess)
{
    int c = guess;
    while (c > 0 && k[c] > v) --c;
    while (c < m - 2 && k[c + 1] <= v) ++c;
    return c;
}
__device__ __forceinline__ int search_last_le(const double *__restrict__ k, int m, double v, int guess)
{
    int g = guess;
    while (g > 0 && k[g] > v) --g;
    while (g < m - 1 && k[g + 1] <= v) ++g;
    return g;
}

// shared memory of the persistent kernel: tables staged once per CTA + a region that A and B
// items use in turn
struct SmemTables {       // 32-bit shared-window addresses
    unsigned xk, qk;
    unsigned lutx, lutq;
};
// explicit shared-window accessors (32-bit addresses): the compiler cannot prove the address space
// of pointers that travel through structs and would emit generic loads
__device__ __forceinline__ double lds_f64(unsigned a) { double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ unsigned lds_u32(unsigned a) { unsigned v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v; }
__device__ __forceinline__ int lds_s16(unsigned a) { short v; asm volatile("ld.shared.s16 %0, [%1];" : "=h"(v) : "r"(a) : "memory"); return (int)v; }
__device__ __forceinline__ double2 lds_v2f64(unsigned a)
{
    double2 v; asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a) : "memory"); return v;
}
__device__ __forceinline__ uint4 lds_v4u32(unsigned a)
{
    uint4 v; asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory"); return v;
}
__device__ __forceinline__ void sts_u32(unsigned a, unsigned v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts_f64(unsigned a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
__device__ __forceinline__ void sts_v2f64(unsigned a, double x, double y)
{
    asm volatile("st.shared.v2.f64 [%0], {%1,%2};" ::"r"(a), "d"(x), "d"(y) : "memory");
}
__device__ __forceinline__ void sts_v4u32(unsigned a, unsigned x, unsigned y, unsigned z, unsigned w)
{
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
__device__ __forceinline__ unsigned atoms_add(unsigned a, unsigned v)
{
    unsigned r; asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(r) : "r"(a), "r"(v) : "memory"); return r;
}

// zero-fill rows [r0, r1) of `out` (contiguous rows, ld doubles each) with coalesced stores, so
// that the scattered row stores of B land in valid, L2-resident sectors.  The work is cut in
// `nslice` slices that the A loop issues between queries: the stores drain under the logarithms.
struct ZeroFill {
    double2 *p2; long long n2; double *head, *tail;
};
__device__ __forceinline__ ZeroFill zero_fill_plan(double *out, long long ld, long long r0, long long r1)
{
    ZeroFill z{nullptr, 0, nullptr, nullptr};
    double *p = out + r0 * ld, *e = out + r1 * ld;
    if (p >= e) return z;
    if ((reinterpret_cast<size_t>(p) & 8) != 0) { z.head = p; ++p; }
    z.n2 = (e - p) >> 1;
    z.p2 = reinterpret_cast<double2 *>(p);
    if ((e - p) & 1) z.tail = e - 1;
    return z;
}
__device__ __forceinline__ void zero_fill_slice(const ZeroFill &z, int slice, int nslice)
{
    const long long per = (z.n2 + nslice - 1) / nslice;
    long long k0 = per * slice, k1 = k0 + per;
    if (k1 > z.n2) k1 = z.n2;
    for (long long k = k0 + threadIdx.x; k < k1; k += kBinThreads) z.p2[k] = make_double2(0.0, 0.0);
    if (slice == 0 && threadIdx.x == 0) { if (z.head) *z.head = 0.0; if (z.tail) *z.tail = 0.0; }
}

// ---- A item: classify, locate, t_x / t_q, tile-local sort by coarse key, payload stores ---------
// Per query only (x, q2) live in registers across the loop; the payload (a, b, idx, fk) and the
// (coarse key, rank) pair are parked in shared memory until the tile's runs have been reserved.
#ifndef PDF_AGRP
#define PDF_AGRP 2
#endif
constexpr int kGrp = PDF_AGRP;         // queries of a thread that go through the A item's steps together
                                       // (1024-query tiles: 1: 11.67, 2: 10.93, 4: 10.77 ms; 2048-query tiles: 2: 10.22, 4: 10.54 ms)
static_assert(kTileQ % kGrp == 0, "kTileQ must be a multiple of kGrp");

struct ASmem {            // 32-bit shared-window addresses
    unsigned cnt;         // unsigned [nck] queries of this tile per coarse key
    unsigned base;        // unsigned [nck] first slot of the tile's run in the key's bin
    unsigned pay;         // uint4 [kTileA][2] payloads in query order; .w of the second word = ck<<16 | rank
};

__device__ __forceinline__ void a_item(const StreamArgs &A, const SmemTables &T, const ASmem &S, int slot,
                                       long long chunk_base, long long chunk_end, int tile, unsigned long long *err_local,
                                       const unsigned long long *ring_free, unsigned long long ring_target)
{
    const GridDev &G = A.G;
    const BinDev &B = A.B;
    unsigned *counts = A.W.counts + (size_t)slot * B.nck;
    Payload *bins = A.W.bins + (size_t)slot * B.nck * A.cap;
    Payload *ovf = A.W.ovf + (size_t)slot * A.chunk;
    unsigned *ovf_count = A.W.ovf_count + slot;
    const unsigned s_xk = T.xk, s_qk = T.qk, s_lx = T.lutx, s_lq = T.lutq;
    const unsigned s_cnt = S.cnt, s_base = S.base, s_pay = S.pay;
    const int nx = G.nx, nqt = G.nqtot;
    const double xmin = lds_f64(s_xk), xmax = lds_f64(s_xk + 8u * (nx - 1));
    const double qmin = lds_f64(s_qk), qmax = lds_f64(s_qk + 8u * (nqt - 1));
    const double u0 = __ldg(G.uk), s0 = __ldg(G.sk);

    PH_DECL;
    for (int k = threadIdx.x; k < B.nck; k += kBinThreads) sts_u32(s_cnt + 4u * k, 0u);

    const long long t0 = chunk_base + (long long)tile * kTileA;
    long long t1 = t0 + kTileA;
    if (t1 > chunk_end) t1 = chunk_end;
    ZeroFill zf = zero_fill_plan(A.out, A.ld, t0, A.zfill ? t1 : t0);
    cta_sync();

    // The thread's kTileQ queries go through the steps together, so that the independent loads and
    // logarithms of one step overlap (the shared-memory accessors are ordered asm statements: only
    // what is issued before the first use runs concurrently).
    // in groups of kGrp (a rolled loop over the groups keeps the code small)
#pragma unroll 1
    for (int g0 = 0; g0 < kTileQ; g0 += kGrp) {
    double xv[kGrp], qv[kGrp], lx[kGrp], lq[kGrp];
    int gi[kGrp], gj[kGrp];
    unsigned st[kGrp];                                           // 0: not a query, 1: invalid, 2: valid
#pragma unroll
    for (int q = 0; q < kGrp; ++q) {
        const long long e = t0 + (g0 + q) * kBinThreads + threadIdx.x;
        xv[q] = 1.0; qv[q] = 1.0;
        if (e < t1) { xv[q] = __ldcs(A.x + e); qv[q] = __ldcs(A.q2 + e); }
    }
    PH(21);
    // The ring slot must have been drained by B(c - kRing) before this tile touches its bins (after the
    // next barrier); polled here, under the loads.  The whole warp polls (same address): a lane that
    // spins alone would reach the barrier apart from its warp, and bar.sync counts such a warp twice.
    if (g0 == 0 && threadIdx.x < 32 && ring_target) wait_counter(ring_free, ring_target);
    PH(11);
    zero_fill_slice(zf, (g0 / kGrp) * 4 + 0, 4 * (kTileQ / kGrp));
    PH(22);
#pragma unroll
    for (int q = 0; q < kGrp; ++q) {
        const long long e = t0 + (g0 + q) * kBinThreads + threadIdx.x;
        st[q] = e < t1 ? ((!(finite_pos(xv[q]) && finite_pos(qv[q])) || xv[q] > xmax) ? 1u : 2u) : 0u;   // C-10
        lx[q] = 0.0; lq[q] = 0.0;
        if (st[q] == 2u) { lx[q] = log(xv[q]); lq[q] = log(qv[q]); }
    }
    PH(23);
    zero_fill_slice(zf, (g0 / kGrp) * 4 + 1, 4 * (kTileQ / kGrp));
    PH(22);
    // start guesses of both searches (buckets clamped: always a valid table entry)
#pragma unroll
    for (int q = 0; q < kGrp; ++q) {
        int bx = (int)((lx[q] - u0) * B.lutx_scale), bq = (int)((lq[q] - s0) * B.lutq_scale);
        bx = bx < 0 ? 0 : (bx >= kLutSize ? kLutSize - 1 : bx);
        bq = bq < 0 ? 0 : (bq >= kLutSize ? kLutSize - 1 : bq);
        gi[q] = lds_s16(s_lx + 2u * bx);
        gj[q] = lds_s16(s_lq + 2u * bq);
    }
    // The guess is the cell at the lower edge of the bucket and buckets are finer than cells, so the
    // query lies <= 1 knot (x) or <= 2 knots (Q2: a threshold is two equal knots) above it: branch-free
    // steps on knots loaded together, a check of the C-4 condition on the raw values, and the exact
    // walk only where the check fails (coarser tables, rounding of the bucket index).
    {
        double xa[kGrp], xb[kGrp], xc[kGrp], qa[kGrp], qb[kGrp], qc[kGrp], qd[kGrp];
#pragma unroll
        for (int q = 0; q < kGrp; ++q) {
            const int c = gi[q], g = gj[q];
            xa[q] = lds_f64(s_xk + 8u * c);
            xb[q] = lds_f64(s_xk + 8u * min(c + 1, nx - 1));
            xc[q] = lds_f64(s_xk + 8u * min(c + 2, nx - 1));
            qa[q] = lds_f64(s_qk + 8u * g);
            qb[q] = lds_f64(s_qk + 8u * min(g + 1, nqt - 1));
            qc[q] = lds_f64(s_qk + 8u * min(g + 2, nqt - 1));
            qd[q] = lds_f64(s_qk + 8u * min(g + 3, nqt - 1));
        }
        bool fix = false;
#pragma unroll
        for (int q = 0; q < kGrp; ++q) {
            const double x = xv[q], q2 = qv[q];
            int c = gi[q];
            const bool ux = c < nx - 2 && xb[q] <= x;              // x cells: [0, nx-2]
            c += ux;
            const double xlo = ux ? xb[q] : xa[q], xhi = ux ? xc[q] : xb[q];
            const bool okx = xlo <= x && (c >= nx - 2 || x < xhi);
            gi[q] = c;
            int g = gj[q];                                         // last knot <= q2: [0, nqt-1]
            const bool u1 = g < nqt - 1 && qb[q] <= q2;
            g += u1;
            double lo = u1 ? qb[q] : qa[q], hi = u1 ? qc[q] : qb[q];
            const double nx2 = u1 ? qd[q] : qc[q];
            const bool u2 = g < nqt - 1 && hi <= q2;
            g += u2;
            lo = u2 ? hi : lo; hi = u2 ? nx2 : hi;
            const bool okq = lo <= q2 && (g >= nqt - 1 || q2 < hi);
            gj[q] = g;
            fix |= st[q] == 2u && ((!(x < xmin) && !okx) || (!(q2 < qmin) && !okq));
        }
        if (fix) {
#pragma unroll
            for (int q = 0; q < kGrp; ++q) {
                const double x = xv[q], q2 = qv[q];
                if (st[q] != 2u) continue;
                if (!(x < xmin)) {
                    int c = gi[q];
                    while (c > 0 && lds_f64(s_xk + 8u * c) > x) --c;
                    while (c < nx - 2 && lds_f64(s_xk + 8u * (c + 1)) <= x) ++c;
                    gi[q] = c;
                }
                if (!(q2 < qmin)) {
                    int g = gj[q];
                    while (g > 0 && lds_f64(s_qk + 8u * g) > q2) --g;
                    while (g < nqt - 1 && lds_f64(s_qk + 8u * (g + 1)) <= q2) ++g;
                    gj[q] = g;
                }
            }
        }
    }
    PH(24);
    zero_fill_slice(zf, (g0 / kGrp) * 4 + 2, 4 * (kTileQ / kGrp));
    PH(22);
    // cell constants (L1-resident tables) and the knots above, all in flight
    {
        int adj[kGrp];
#pragma unroll
        for (int q = 0; q < kGrp; ++q) adj[q] = (int)__ldg(G.cell_adj + gj[q]);   // last knot of a sub-grid -> its last cell
        double2 ci[kGrp], cj[kGrp];
        double kx1[kGrp], kq1[kGrp];
#pragma unroll
        for (int q = 0; q < kGrp; ++q) {
            gj[q] -= adj[q];
            ci[q] = __ldg(reinterpret_cast<const double2 *>(G.cx + gi[q]));          // lo_log, inv_d
            cj[q] = __ldg(reinterpret_cast<const double2 *>(G.cq + gj[q]));
            kx1[q] = lds_f64(s_xk + 8u * (gi[q] + 1));
            kq1[q] = lds_f64(s_qk + 8u * (gj[q] + 1));
        }
        // the extrapolation abscissae through reciprocals (one division each per item instead of per query)
        const double inv_du0 = 1.0 / (__ldg(G.uk + 1) - u0);
        const double sA = __ldg(G.sk + nqt - 2), inv_ds = 1.0 / (__ldg(G.sk + nqt - 1) - sA), inv_qmin = 1.0 / qmin;
#pragma unroll
        for (int q = 0; q < kGrp; ++q) {
            const double x = xv[q], q2 = qv[q];
            const bool lowx = x < xmin, lowq = q2 < qmin, highq = q2 > qmax;
            const double ta = lowx ? (lx[q] - u0) * inv_du0                           // theta_x (C-7)
                                   : (x == kx1[q]) ? 1.0 : (lx[q] - ci[q].x) * ci[q].y;
            const double tb = lowq ? q2 * inv_qmin                                    // r (C-9)
                            : highq ? (lq[q] - sA) * inv_ds                           // theta_q (C-8)
                                    : (q2 == kq1[q]) ? 1.0 : (lq[q] - cj[q].x) * cj[q].y;
            lx[q] = ta; lq[q] = tb;
        }
    }
    PH(25);
    zero_fill_slice(zf, (g0 / kGrp) * 4 + 3, 4 * (kTileQ / kGrp));
    PH(22);
#pragma unroll
    for (int q = 0; q < kGrp; ++q) {
        const int ql = (g0 + q) * kBinThreads + threadIdx.x;             // query index inside the tile
        const double x = xv[q], q2 = qv[q];
        const bool lowx = x < xmin, lowq = q2 < qmin, highq = q2 > qmax;
        unsigned tag = st[q] == 0u ? 0xffffffffu : 0xfffffffeu;
        unsigned fk = 0;
        if (st[q] == 2u) {
            const int jg = gj[q];
            fk = lowq ? (unsigned)nqt : highq ? (unsigned)nqt + 1u : (unsigned)jg;
            unsigned ck = (unsigned)gi[q];
            if (lowx)       // low-x classes: one coarse key per band of Q2 cells, so that their batches fill up;
                            // the corners, whose rows are the most expensive, are dealt over kCornerSplit keys each
                ck = (unsigned)B.ncx + (lowq ? (unsigned)kLowXBands + (threadIdx.x & (kCornerSplit - 1))
                                             : highq ? (unsigned)(kLowXBands + kCornerSplit) + (threadIdx.x & (kCornerSplit - 1))
                                                     : (unsigned)(jg * kLowXBands) / (unsigned)nqt);
            PDF_ASSERT(ck < (unsigned)B.nck && fk < (unsigned)B.nfk);
            const unsigned rank = atoms_add(s_cnt + 4u * ck, 1u);
            tag = (ck << 16) | rank;
        }
        const unsigned pa = s_pay + 32u * ql;
        sts_v2f64(pa, lx[q], lq[q]);
        sts_v4u32(pa + 16u, (unsigned)(t0 + ql - chunk_base), fk, 0u, tag);
    }
    }
    PH(26);
    cta_sync();
    PH(8);
    for (int k = threadIdx.x; k < B.nck; k += kBinThreads) {       // one global atomic per (tile, key)
        unsigned c = lds_u32(s_cnt + 4u * k);
        sts_u32(s_base + 4u * k, c ? atomicAdd(counts + k, c) : 0u);
    }
    cta_sync();
    PH(9);
#pragma unroll 1
    for (int q = 0; q < kTileQ; ++q) {
        const int ql = q * kBinThreads + threadIdx.x;
        const unsigned pa = s_pay + 32u * ql;
        const uint4 w1 = lds_v4u32(pa + 16u);
        if (w1.w == 0xffffffffu) continue;
        if (w1.w == 0xfffffffeu) {
            double *o = A.out + (t0 + ql) * A.ld;
            for (int p = 0; p < A.cm.n; ++p) o[p] = qnan();
            if (A.count_err) ++*err_local;
            continue;
        }
        const double2 ab = lds_v2f64(pa);
        const unsigned ck = w1.w >> 16, rank = w1.w & 0xffffu;
        PDF_ASSERT(ck < (unsigned)B.nck);
        const unsigned pos = lds_u32(s_base + 4u * ck) + rank;
        if (pos < (unsigned)A.cap) store_payload(bins + (size_t)ck * A.cap + pos, ab.x, ab.y, w1.x, w1.y);
        else {                                                     // bin full: raw query to the overflow list
            unsigned o = atomicAdd(ovf_count, 1u);
            store_payload(ovf + o, __ldg(A.x + t0 + ql), __ldg(A.q2 + t0 + ql), w1.x, 0u);
        }
    }
    PH(10);
}

}  // namespace pdfg

#include "pdf_binned_eval.cuh"
