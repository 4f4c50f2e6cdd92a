// pdf_binned_eval.cuh -- B items (warp-coherent evaluation from shared memory) and the
// persistent kernel itself.
#pragma once

namespace pdfg {

// The 4 grid columns of a coarse key, staged in shared memory as sV[jg][slot a][12 doubles]:
// the 4 x-nodes of a Q2 row are 384 contiguous bytes.  Every lane of a warp passes the SAME
// address: each LDS.128 is one broadcast (1.5 clk) that serves 32 queries.
// sV is addressed in the shared window (32-bit address) with explicit ld.shared: the compiler
// cannot prove the address space of a pointer that travels through a struct
__device__ __forceinline__ double2 lds_d2(unsigned addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

__device__ __forceinline__ void node_fma_s(unsigned p, double w, double acc[kNF])
{
    double2 v0 = lds_d2(p), v1 = lds_d2(p + 16), v2 = lds_d2(p + 32), v3 = lds_d2(p + 48), v4 = lds_d2(p + 64),
            v5 = lds_d2(p + 80);
    acc[0] = fma(w, v0.x, acc[0]); acc[1] = fma(w, v0.y, acc[1]);
    acc[2] = fma(w, v1.x, acc[2]); acc[3] = fma(w, v1.y, acc[3]);
    acc[4] = fma(w, v2.x, acc[4]); acc[5] = fma(w, v2.y, acc[5]);
    acc[6] = fma(w, v3.x, acc[6]); acc[7] = fma(w, v3.y, acc[7]);
    acc[8] = fma(w, v4.x, acc[8]); acc[9] = fma(w, v4.y, acc[9]);
    acc[10] = fma(w, v5.x, acc[10]);
}

__device__ __forceinline__ unsigned snode(unsigned sV, int jrow, int slot)
{
    return sV + (unsigned)((jrow * 4 + slot) * kNFP * 8);
}

struct AxisNodes { int n[4]; };
__device__ __forceinline__ AxisNodes q_nodes(const CellTab &c, int jg)
{
    AxisNodes a; a.n[0] = (c.aL == 1.0) ? jg : jg - 1; a.n[1] = jg; a.n[2] = jg + 1; a.n[3] = (c.aR == 1.0) ? jg + 1 : jg + 2;
    return a;
}

__device__ __forceinline__ void zero_acc(double acc[kNF])
{
#pragma unroll
    for (int f = 0; f < kNF; ++f) acc[f] = 0.0;
}

// C-6: 16-node tensor sum in cell (i, jg); the x-nodes i-1..i+2 (clamped) sit in slots 0..3
__device__ __forceinline__ void eval_interior_s(const GridDev &G, unsigned sV, int i, int jg, double tx, double tq,
                                                double acc[kNF])
{
    CellTab cq = G.cq[jg];
    double wx[4], wq[4];
    hermite_weights(tx, G.cx[i], wx);
    hermite_weights(tq, cq, wq);
    AxisNodes qn = q_nodes(cq, jg);
    zero_acc(acc);
#pragma unroll
    for (int b = 0; b < 4; ++b)
#pragma unroll
        for (int a = 0; a < 4; ++a) node_fma_s(snode(sV, qn.n[b], a), wq[b] * wx[a], acc);
}

// sum_b wq[b] V[slot][rows of cell jg]  (x fixed on a knot column)
__device__ __forceinline__ void eval_column_s(const GridDev &G, unsigned sV, int slot, int jg, double tq, double acc[kNF])
{
    CellTab cq = G.cq[jg];
    double wq[4];
    hermite_weights(tq, cq, wq);
    AxisNodes qn = q_nodes(cq, jg);
    zero_acc(acc);
#pragma unroll
    for (int b = 0; b < 4; ++b) node_fma_s(snode(sV, qn.n[b], slot), wq[b], acc);
}

// sum_a wx[a] V[slots of cell i][row]  (Q2 fixed on a knot row)
__device__ __forceinline__ void eval_row_s(const GridDev &G, unsigned sV, int i, int jrow, double tx, double acc[kNF])
{
    double wx[4];
    hermite_weights(tx, G.cx[i], wx);
    zero_acc(acc);
#pragma unroll
    for (int a = 0; a < 4; ++a) node_fma_s(snode(sV, jrow, a), wx[a], acc);
}

__device__ __forceinline__ void load_node_s(unsigned sV, int jrow, int slot, double acc[kNF])
{
    zero_acc(acc);
    node_fma_s(snode(sV, jrow, slot), 1.0, acc);
}

// extrapolation classes (a-5).  Warp-uniform branches: a batch holds one (coarse, fine) key.
// In an in-range-x unit the slots hold the x-nodes of cell i; in a low-x unit slot 0 / 1 hold
// the knot columns X_0 / X_1 (C-7).
__device__ __noinline__ void eval_extrap_s(const GridDev &G, const BinDev &B, unsigned sV, bool lowx_unit, int i,
                                           int fk, double pa, double pb, double acc[kNF])
{
    double e0[kNF], e1[kNF];
    const int last = G.nqtot - 1;
    if (!lowx_unit) {
        if (fk == B.nqt) {                                 // low-Q (C-9): pa = t_x, pb = r
            eval_row_s(G, sV, i, 0, pa, e0);
            eval_interior_s(G, sV, i, B.jgplus, pa, B.tqplus, e1);
            const double lnr = log(pb);
#pragma unroll
            for (int f = 0; f < kNF; ++f) acc[f] = lowq_continue_ln(e0[f], e1[f], pb, lnr);
        } else {                                           // high-Q (C-8): pa = t_x, pb = theta_q
            eval_row_s(G, sV, i, last - 1, pa, e0);
            eval_row_s(G, sV, i, last, pa, e1);
#pragma unroll
            for (int f = 0; f < kNF; ++f) acc[f] = continue_two(e0[f], e1[f], pb);
        }
        return;
    }
    if (fk < B.nqt) {                                      // low-x (C-7): pa = theta_x, pb = t_q
        eval_column_s(G, sV, 0, fk, pb, e0);
        eval_column_s(G, sV, 1, fk, pb, e1);
#pragma unroll
        for (int f = 0; f < kNF; ++f) acc[f] = continue_two(e0[f], e1[f], pa);
    } else if (fk == B.nqt) {                              // low-x & low-Q (L1744): x rule, then Q rule
        double e2[kNF], e3[kNF];
        const double lnr = log(pb);
        load_node_s(sV, 0, 0, e0); load_node_s(sV, 0, 1, e1);
        eval_column_s(G, sV, 0, B.jgplus, B.tqplus, e2); eval_column_s(G, sV, 1, B.jgplus, B.tqplus, e3);
#pragma unroll
        for (int f = 0; f < kNF; ++f)
            acc[f] = lowq_continue_ln(continue_two(e0[f], e1[f], pa), continue_two(e2[f], e3[f], pa), pb, lnr);
    } else {                                               // low-x & high-Q
        double e2[kNF], e3[kNF];
        load_node_s(sV, last - 1, 0, e0); load_node_s(sV, last - 1, 1, e1);
        load_node_s(sV, last, 0, e2); load_node_s(sV, last, 1, e3);
#pragma unroll
        for (int f = 0; f < kNF; ++f)
            acc[f] = continue_two(continue_two(e0[f], e1[f], pa), continue_two(e2[f], e3[f], pa), pb);
    }
}

// overflow list: raw queries evaluated by the generic per-thread code (rare; register-capped)
__device__ __noinline__ void ovf_item(const StreamArgs &A, int slot, long long chunk_base, int part)
{
    unsigned cnt = __ldcg(A.W.ovf_count + slot);
    const Payload *ovf = A.W.ovf + (size_t)slot * A.chunk;
    for (unsigned e = part * kBinThreads + threadIdx.x; e < cnt; e += kOvfItems * kBinThreads) {
        double2 ab = __ldcg(reinterpret_cast<const double2 *>(ovf + e));
        uint2 ii = __ldcg(reinterpret_cast<const uint2 *>(ovf + e) + 2);
        QueryPlan P;
        make_plan(A.G, ab.x, ab.y, P);
        double *o = A.out + (chunk_base + ii.x) * A.ld;
        for (int p = 0; p < A.cm.n; ++p) {
            int c = A.cm.col[p];
            o[p] = c < 0 ? 0.0 : plan_value(A.G, A.G.V, P, c);
        }
    }
}

struct BSmem {
    uint4 *sP;            // [cap] payloads (2 x uint4 each)
    double *sV;           // [nqt][4][12]
    double *stage;        // [kBinWarps][32*kNF]
    unsigned long long *sptr; // [kBinWarps][32] output row pointers of the staged batch
    int *fcnt;            // [nfk]
    int *foff;            // [nfk+1]
    int *bstart;          // [nfk+1]
    int *next;            // [1] batch queue of the item
    unsigned short *order;// [cap]
};

// ---- B item: one coarse key of one chunk ------------------------------------------------------
__device__ __forceinline__ void b_item(const StreamArgs &A, const BSmem &S, int slot, long long chunk_base, int item)
{
    const BinDev &B = A.B;
    const GridDev &G = A.G;
    if (item >= B.nck) { ovf_item(A, slot, chunk_base, item - B.nck); return; }
    const int ck = item;
    unsigned *counts = A.W.counts + (size_t)slot * B.nck;
    unsigned cnt_u = __ldcg(counts + ck);
    if (cnt_u == 0u) return;                               // uniform over the CTA
    const int cnt = cnt_u > (unsigned)A.cap ? A.cap : (int)cnt_u;
    const uint4 *bin = reinterpret_cast<const uint4 *>(A.W.bins + ((size_t)slot * B.nck + ck) * A.cap);
    const bool lowx_unit = ck >= B.ncx;
    const int i = lowx_unit ? 0 : ck;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned sPa = (unsigned)__cvta_generic_to_shared(S.sP), sVa = (unsigned)__cvta_generic_to_shared(S.sV);
    const unsigned fcnt = (unsigned)__cvta_generic_to_shared(S.fcnt), foff = (unsigned)__cvta_generic_to_shared(S.foff);
    const unsigned bstart = (unsigned)__cvta_generic_to_shared(S.bstart), order = (unsigned)__cvta_generic_to_shared(S.order);
    const unsigned nexta = (unsigned)__cvta_generic_to_shared(S.next);
    const unsigned stage = (unsigned)__cvta_generic_to_shared(S.stage) + (unsigned)warp * (32 * kNF * 8);
    const unsigned sptr = (unsigned)__cvta_generic_to_shared(S.sptr) + (unsigned)warp * (32 * 8);

    // stage payloads (coalesced) and the key's 4 grid columns
    for (int e = threadIdx.x; e < cnt * 2; e += kBinThreads) {
        uint4 v = __ldcg(bin + e);
        sts_v4u32(sPa + 16u * e, v.x, v.y, v.z, v.w);
    }
    {
        int c0, c1, c2, c3;
        if (lowx_unit) { c0 = 0; c1 = 1; c2 = 0; c3 = 1; }
        else { c0 = i > 0 ? i - 1 : i; c1 = i; c2 = i + 1; c3 = i + 2 < G.nx ? i + 2 : i + 1; }
        const double2 *V2 = reinterpret_cast<const double2 *>(G.V);
        const int tot = G.nqtot * 24;                      // double2 units: rows x 4 slots x 6
        for (int e = threadIdx.x; e < tot; e += kBinThreads) {
            int jg = e / 24, r = e - jg * 24, a = r / 6, p = r - a * 6;
            int col = a == 0 ? c0 : a == 1 ? c1 : a == 2 ? c2 : c3;
            double2 v = __ldg(V2 + ((size_t)jg * G.nx + col) * 6 + p);
            sts_v2f64(sVa + 16u * e, v.x, v.y);
        }
    }
    for (int k = threadIdx.x; k < B.nfk; k += kBinThreads) sts_u32(fcnt + 4u * k, 0u);
    if (threadIdx.x == 0) sts_u32(nexta, 0u);
    __syncthreads();
    // counting sort by fine key: rank kept in the payload's spare word
    for (int e = threadIdx.x; e < cnt; e += kBinThreads) {
        unsigned fk = lds_u32(sPa + 32u * e + 20u);
        unsigned r = atoms_add(fcnt + 4u * fk, 1u);
        sts_u32(sPa + 32u * e + 24u, r);
    }
    __syncthreads();
    if (warp == 0) {                                       // exclusive scans: slots and 32-query batches per key
        int carry_o = 0, carry_b = 0;
        for (int k0 = 0; k0 < B.nfk; k0 += 32) {
            int k = k0 + lane;
            int c = k < B.nfk ? (int)lds_u32(fcnt + 4u * k) : 0;
            int nb = (c + 31) >> 5;
            int so = c, sb = nb;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                int vo = __shfl_up_sync(0xffffffffu, so, d), vb = __shfl_up_sync(0xffffffffu, sb, d);
                if (lane >= d) { so += vo; sb += vb; }
            }
            if (k < B.nfk) { sts_u32(foff + 4u * k, (unsigned)(carry_o + so - c)); sts_u32(bstart + 4u * k, (unsigned)(carry_b + sb - nb)); }
            carry_o += __shfl_sync(0xffffffffu, so, 31);
            carry_b += __shfl_sync(0xffffffffu, sb, 31);
        }
        if (lane == 0) { sts_u32(foff + 4u * B.nfk, (unsigned)carry_o); sts_u32(bstart + 4u * B.nfk, (unsigned)carry_b); }
    }
    __syncthreads();
    for (int e = threadIdx.x; e < cnt; e += kBinThreads) {
        uint2 w = make_uint2(lds_u32(sPa + 32u * e + 20u), lds_u32(sPa + 32u * e + 24u));
        unsigned pos = lds_u32(foff + 4u * w.x) + w.y;
        asm volatile("st.shared.u16 [%0], %1;" ::"r"(order + 2u * pos), "h"((unsigned short)e) : "memory");
    }
    __syncthreads();

    const int total = (int)lds_u32(bstart + 4u * B.nfk);
    for (;;) {
        int fb = 0;
        if (lane == 0) fb = (int)atoms_add(nexta, 1u);     // batches are handed out dynamically,
        fb = __shfl_sync(0xffffffffu, fb, 0);              // last keys first: the extrapolation classes
        if (fb >= total) break;                            // (long, few lanes) must not form the tail
        fb = total - 1 - fb;
        int lo = 0, hi = B.nfk;                            // largest k with bstart[k] <= fb
        while (hi - lo > 1) {
            int mid = (lo + hi) >> 1;
            if ((int)lds_u32(bstart + 4u * mid) <= fb) lo = mid; else hi = mid;
        }
        const int fk = lo, kcnt = (int)lds_u32(fcnt + 4u * fk);
        const int first = (fb - (int)lds_u32(bstart + 4u * fk)) * 32;
        const int nact = min(32, kcnt - first);
        const bool active = lane < nact;
        double pa = 0.0, pb = 0.0;
        unsigned idx = 0;
        if (active) {
            unsigned short e16;
            asm volatile("ld.shared.u16 %0, [%1];" : "=h"(e16) : "r"(order + 2u * (lds_u32(foff + 4u * fk) + first + lane)));
            const unsigned pe = sPa + 32u * e16;
            double2 ab = lds_v2f64(pe);
            pa = ab.x; pb = ab.y;
            idx = lds_u32(pe + 16u);
        }
        double acc[kNF];
        if (!lowx_unit && fk < B.nqt) eval_interior_s(G, sVa, i, fk, pa, pb, acc);
        else eval_extrap_s(G, B, sVa, lowx_unit, i, fk, pa, pb, acc);
        // transpose through shared memory so that whole rows leave in contiguous pieces
#pragma unroll
        for (int f = 0; f < kNF; ++f) sts_f64(stage + 8u * (lane * kNF + f), acc[f]);
        {
            unsigned long long rp = reinterpret_cast<unsigned long long>(A.out + (chunk_base + idx) * A.ld);
            asm volatile("st.shared.u64 [%0], %1;" ::"r"(sptr + 8u * lane), "l"(rp) : "memory");
        }
        __syncwarp();
        if (A.identity) {
            const int tot = nact * kNF;
#pragma unroll
            for (int itx = 0; itx < kNF; ++itx) {
                int e = itx * 32 + lane;
                if (e < tot) {
                    int r = (e * 745) >> 13, p = e - r * kNF;          // e / 11 for e < 352
                    unsigned long long rp;
                    asm volatile("ld.shared.u64 %0, [%1];" : "=l"(rp) : "r"(sptr + 8u * r));
                    reinterpret_cast<double *>(rp)[p] = lds_f64(stage + 8u * e);
                }
            }
        } else {
            const int np = A.cm.n, tot = nact * np;
            for (int e = lane; e < tot; e += 32) {
                int r = e / np, p = e - r * np, c = A.cm.col[p];
                unsigned long long rp;
                asm volatile("ld.shared.u64 %0, [%1];" : "=l"(rp) : "r"(sptr + 8u * r));
                reinterpret_cast<double *>(rp)[p] = c < 0 ? 0.0 : lds_f64(stage + 8u * (r * kNF + c));
            }
        }
        __syncwarp();
    }
    __syncthreads();
    if (threadIdx.x == 0) counts[ck] = 0u;                 // the bin is empty again for the ring
}

// ---- the persistent kernel -----------------------------------------------------------------------
// dynamic shared memory: [knots | LUTs | item region]; the item region is used by A items as
// (cnt, base) and by B items as (payloads, columns, stage, sort tables)
__host__ __device__ inline size_t bsmem_item_bytes(int nqt, int nck, int nfk, int cap)
{
    size_t b = (size_t)cap * 32;                                        // sP
    b += (size_t)nqt * 4 * kNFP * sizeof(double);                       // sV
    b += (size_t)kBinWarps * 32 * kNF * sizeof(double);                 // stage
    b += (size_t)kBinWarps * 32 * sizeof(unsigned long long);           // sptr
    b += (size_t)(3 * nfk + 8) * sizeof(int);                           // fcnt, foff, bstart, next
    b += ((size_t)cap * sizeof(unsigned short) + 15) / 16 * 16;         // order
    size_t a = (size_t)kTileA * 32 + (size_t)2 * nck * sizeof(unsigned); // A items: payloads, cnt, base
    return (b > a ? b : a) + 32;
}

__global__ void __launch_bounds__(kBinThreads, 2) k_pdf_stream(const __grid_constant__ StreamArgs A)
{
    extern __shared__ __align__(32) unsigned char smem_raw[];
    double *s_xk = reinterpret_cast<double *>(smem_raw);
    double *s_qk = s_xk + A.G.nx;
    short *s_lutx = reinterpret_cast<short *>(s_qk + A.G.nqtot);
    short *s_lutq = s_lutx + kLutSize;
    unsigned char *region = reinterpret_cast<unsigned char *>(s_lutq + kLutSize);
    region = reinterpret_cast<unsigned char *>((reinterpret_cast<size_t>(region) + 31) & ~(size_t)31);
    __shared__ unsigned long long s_ticket;

    for (int i = threadIdx.x; i < A.G.nx; i += kBinThreads) s_xk[i] = A.G.xk[i];
    for (int i = threadIdx.x; i < A.G.nqtot; i += kBinThreads) s_qk[i] = A.G.qk[i];
    for (int i = threadIdx.x; i < kLutSize; i += kBinThreads) { s_lutx[i] = A.B.lutx[i]; s_lutq[i] = A.B.lutq[i]; }
    __syncthreads();
    SmemTables T{s_xk, s_qk, s_lutx, s_lutq};
    ASmem SA;
    SA.pay = reinterpret_cast<uint4 *>(region);
    SA.cnt = reinterpret_cast<unsigned *>(region + (size_t)kTileA * 32);
    SA.base = SA.cnt + A.B.nck;
    BSmem SB;
    SB.sP = reinterpret_cast<uint4 *>(region);
    SB.sV = reinterpret_cast<double *>(region + (size_t)A.cap * 32);
    SB.stage = SB.sV + (size_t)A.G.nqtot * 4 * kNFP;
    SB.sptr = reinterpret_cast<unsigned long long *>(SB.stage + kBinWarps * 32 * kNF);
    SB.fcnt = reinterpret_cast<int *>(SB.sptr + kBinWarps * 32);
    SB.foff = SB.fcnt + A.B.nfk + 1;
    SB.bstart = SB.foff + A.B.nfk + 1;
    SB.next = SB.bstart + A.B.nfk + 2;
    SB.order = reinterpret_cast<unsigned short *>(SB.next + 2);

    unsigned long long *ctrl = A.W.ctrl;
    const unsigned long long TA = A.ta, TB = A.B.nitems, per = TA + TB;
    const unsigned long long total = (unsigned long long)A.nchunks * per;
    unsigned long long err_local = 0;

    // the next ticket is fetched while the current item runs (a global atomic is ~1 us)
    unsigned long long next_t = 0;
    if (threadIdx.x == 0) next_t = atomicAdd(ctrl, 1ULL);
    for (;;) {
        if (threadIdx.x == 0) s_ticket = next_t;
        __syncthreads();
        const unsigned long long t = s_ticket;
        __syncthreads();
        if (t >= total) break;
        if (threadIdx.x == 0) next_t = atomicAdd(ctrl, 1ULL);      // consumed at the top of the next round
        // ticket order, lag L = kLag rounds:  round r = [A(r) tiles | B(r-L) items]; B(c) is handed out
        // L rounds after A(c), so its tiles were claimed >= L waves earlier and the wait below is ~never taken
        bool isA; long long c; int sub;
        {
            const unsigned long long RA = (unsigned long long)(A.nchunks < kLag ? A.nchunks : kLag);   // A-only rounds
            const unsigned long long F = (unsigned long long)A.nchunks - RA;                             // full rounds
            if (t < RA * TA) { isA = true; c = (long long)(t / TA); sub = (int)(t % TA); }
            else {
                unsigned long long tp = t - RA * TA;
                if (tp < F * per) {
                    unsigned long long round = RA + tp / per, w = tp % per;
                    isA = w < TA;
                    c = isA ? (long long)round : (long long)(round - RA);
                    sub = (int)(isA ? w : w - TA);
                } else {
                    unsigned long long tq = tp - F * per;
                    isA = false; c = (long long)(F + tq / TB); sub = (int)(tq % TB);
                }
            }
        }
        const int slot = (int)(c % kRing);
        const unsigned long long gen = (unsigned long long)(c / kRing);
        unsigned long long *a_done = ctrl + 8 + slot * 4, *b_fin = a_done + 1, *b_done = a_done + 2;
        const long long chunk_base = c * A.chunk;
        if (isA) {
            if (threadIdx.x == 0 && gen > 0) wait_counter(b_done, gen * TB);   // ring slot drained
            __syncthreads();
            a_item(A, T, SA, slot, chunk_base, sub, &err_local);
            __threadfence();
            __syncthreads();
            if (threadIdx.x == 0) atomicAdd(a_done, 1ULL);
        } else {
            if (threadIdx.x == 0) wait_counter(a_done, (gen + 1) * TA);        // every tile of A(c) released
            __syncthreads();
            b_item(A, SB, slot, chunk_base, sub);
            __threadfence();
            __syncthreads();
            if (threadIdx.x == 0) {
                unsigned long long old = atomicAdd(b_fin, 1ULL);
                if (old + 1 == (gen + 1) * TB) {                               // last item of the chunk
                    A.W.ovf_count[slot] = 0u;
                    __threadfence();
                    atomicAdd(b_done, TB);
                }
            }
        }
    }
    if (err_local) atomicAdd(A.G.err_count, err_local);
}

}  // namespace pdfg
