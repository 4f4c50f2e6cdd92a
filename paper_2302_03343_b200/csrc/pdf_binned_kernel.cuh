// pdf_binned_kernel.cuh -- device code of the persistent binned kernel: helpers and A items
// (see pdf_binned.cuh for the design).
#pragma once

namespace pdfg {

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
    int identity;              // 1: requested columns == the grid's 11 columns in order
    int zfill;                 // 1: rows are contiguous (ld == npid): A items zero-fill their tile of `out`
};

// ---- small device helpers ----------------------------------------------------------------------
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long *p)
{
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void wait_counter(const unsigned long long *p, unsigned long long target)
{
    unsigned ns = 32;
    while (ld_acquire_u64(p) < target) {
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
struct SmemTables {
    const double *xk, *qk;
    const short *lutx, *lutq;
};
struct ASmem {
    unsigned *cnt;        // [nck] queries of this tile per coarse key
    unsigned *base;       // [nck] first slot of the tile's run in the key's bin
};

// zero-fill rows [r0, r1) of `out` (contiguous rows, ld doubles each) with coalesced stores, so
// that the scattered row stores of B land in valid, L2-resident sectors
__device__ __forceinline__ void zero_fill_rows(double *out, long long ld, long long r0, long long r1)
{
    double *p = out + r0 * ld, *e = out + r1 * ld;
    if (p >= e) return;
    if ((reinterpret_cast<size_t>(p) & 8) != 0) { if (threadIdx.x == 0) *p = 0.0; ++p; }
    long long n2 = (e - p) >> 1;
    double2 *p2 = reinterpret_cast<double2 *>(p);
    for (long long k = threadIdx.x; k < n2; k += kBinThreads) p2[k] = make_double2(0.0, 0.0);
    if (((e - p) & 1) && threadIdx.x == 0) e[-1] = 0.0;
}

// ---- A item: classify, locate, t_x / t_q, tile-local sort by coarse key, payload stores ---------
__device__ __forceinline__ void a_item(const StreamArgs &A, const SmemTables &T, const ASmem &S, int slot,
                                       long long chunk_base, int tile, unsigned long long *err_local)
{
    const GridDev &G = A.G;
    const BinDev &B = A.B;
    unsigned *counts = A.W.counts + (size_t)slot * B.nck;
    Payload *bins = A.W.bins + (size_t)slot * B.nck * A.cap;
    Payload *ovf = A.W.ovf + (size_t)slot * A.chunk;
    unsigned *ovf_count = A.W.ovf_count + slot;
    const double xmin = T.xk[0], xmax = T.xk[G.nx - 1], qmin = T.qk[0], qmax = T.qk[G.nqtot - 1];
    const double u0 = __ldg(G.uk), s0 = __ldg(G.sk);

    for (int k = threadIdx.x; k < B.nck; k += kBinThreads) S.cnt[k] = 0u;

    const long long t0 = chunk_base + (long long)tile * kTileA;
    long long t1 = t0 + kTileA;
    if (t1 > A.n) t1 = A.n;
    if (t1 > chunk_base + A.chunk) t1 = chunk_base + A.chunk;
    double xv[kTileQ], qv[kTileQ];
    const long long e0 = t0 + threadIdx.x;
#pragma unroll
    for (int q = 0; q < kTileQ; ++q) {
        long long e = e0 + q * kBinThreads;
        bool in = e < t1;
        xv[q] = in ? __ldcs(A.x + e) : -1.0;      // streaming: read once
        qv[q] = in ? __ldcs(A.q2 + e) : -1.0;
    }
    if (A.zfill) zero_fill_rows(A.out, A.ld, t0, t1);
    __syncthreads();

    int ck[kTileQ];
    unsigned fkv[kTileQ], rank[kTileQ];
    double pa[kTileQ], pb[kTileQ];
#pragma unroll
    for (int q = 0; q < kTileQ; ++q) {
        long long e = e0 + q * kBinThreads;
        double x = xv[q], q2 = qv[q];
        ck[q] = -1; rank[q] = 0; fkv[q] = 0; pa[q] = 0.0; pb[q] = 0.0;
        if (e >= t1) continue;
        if (!(finite_pos(x) && finite_pos(q2)) || x > xmax) { ck[q] = -2; continue; }       // C-10
        bool lowx = x < xmin, lowq = q2 < qmin, highq = q2 > qmax;
        double lx = log(x), lq = log(q2);
        int i = 0, jg = 0;
        double ta, tb;
        if (!lowx) {
            int b = (int)((lx - u0) * B.lutx_scale);
            b = b < 0 ? 0 : (b >= kLutSize ? kLutSize - 1 : b);
            i = search_cell(T.xk, G.nx, x, T.lutx[b]);
            CellTab c = G.cx[i];
            ta = (x == T.xk[i + 1]) ? 1.0 : (lx - c.lo_log) * c.inv_d;
        } else {
            ta = (lx - u0) / (__ldg(G.uk + 1) - u0);              // theta_x (C-7)
        }
        if (!lowq && !highq) {
            int b = (int)((lq - s0) * B.lutq_scale);
            b = b < 0 ? 0 : (b >= kLutSize ? kLutSize - 1 : b);
            int g = search_last_le(T.qk, G.nqtot, q2, T.lutq[b]);
            int k = __ldg(G.sub_of + g);
            int q0 = __ldg(G.qoff + k), q1 = __ldg(G.qoff + k + 1);
            int j = g - q0;
            if (j > q1 - q0 - 2) j = q1 - q0 - 2;
            jg = q0 + j;
            CellTab c = G.cq[jg];
            tb = (q2 == T.qk[jg + 1]) ? 1.0 : (lq - c.lo_log) * c.inv_d;
        } else if (highq) {
            int last = G.nqtot - 1;
            tb = (lq - __ldg(G.sk + last - 1)) / (__ldg(G.sk + last) - __ldg(G.sk + last - 1));   // theta_q (C-8)
        } else {
            tb = q2 / qmin;                                        // r (C-9)
        }
        unsigned idx = (unsigned)(e - chunk_base);
        ck[q] = lowx ? B.ncx + (int)(idx & (kLowXSplit - 1)) : i;
        fkv[q] = lowq ? (unsigned)B.nqt : highq ? (unsigned)B.nqt + 1u : (unsigned)jg;
        pa[q] = ta; pb[q] = tb;
        rank[q] = atomicAdd(S.cnt + ck[q], 1u);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < B.nck; k += kBinThreads) {       // one global atomic per (tile, key)
        unsigned c = S.cnt[k];
        S.base[k] = c ? atomicAdd(counts + k, c) : 0u;
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < kTileQ; ++q) {
        long long e = e0 + q * kBinThreads;
        if (ck[q] >= 0) {
            unsigned idx = (unsigned)(e - chunk_base);
            unsigned pos = S.base[ck[q]] + rank[q];
            if (pos < (unsigned)A.cap) store_payload(bins + (size_t)ck[q] * A.cap + pos, pa[q], pb[q], idx, fkv[q]);
            else {                                                 // bin full: raw query to the overflow list
                unsigned o = atomicAdd(ovf_count, 1u);
                store_payload(ovf + o, xv[q], qv[q], idx, 0u);
            }
        } else if (ck[q] == -2) {
            double *o = A.out + e * A.ld;
            for (int p = 0; p < A.cm.n; ++p) o[p] = qnan();
            ++*err_local;
        }
    }
}

}  // namespace pdfg

#include "pdf_binned_eval.cuh"
