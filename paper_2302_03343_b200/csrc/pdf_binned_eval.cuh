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
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
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
__device__ __noinline__ void ovf_item(const StreamArgs &A, const double *V, int slot, long long chunk_base, int part)
{
    unsigned cnt = ld_acquire_u32(A.W.ovf_count + slot);
    const Payload *ovf = A.W.ovf + (size_t)slot * A.chunk;
    for (unsigned e = part * kBinThreads + threadIdx.x; e < cnt; e += kOvfItems * kBinThreads) {
        double2 ab = __ldcg(reinterpret_cast<const double2 *>(ovf + e));
        uint2 ii = __ldcg(reinterpret_cast<const uint2 *>(ovf + e) + 2);
        QueryPlan P;
        make_plan(A.G, ab.x, ab.y, P);
        double *o = A.out + (chunk_base + ii.x) * A.ld;
        for (int p = 0; p < A.cm.n; ++p) {
            int c = A.cm.col[p];
            o[p] = c < 0 ? 0.0 : plan_value(A.G, V, P, c);
        }
    }
}

// ---- interior cells on the FP64 tensor pipe (DMMA m8n8k4) ---------------------------------------
// A batch is one cell: out[q][f] = sum_n W[q][n] V[n][f] is a (queries x 16 nodes) x (16 nodes x 11
// flavours) contraction.  As mma.sync.m8n8k4 tiles (8 queries x 8 flavours, k = 4 nodes) the cell's
// values are read ONCE per batch, 8 doubles per lane, instead of 192 broadcast doubles per lane;
// DMMA runs on the same FP64 pipe as DFMA, so this buys operand traffic and
// instruction count, not flops.  Lane (g = lane/4, t = lane%4) serves query g of the 8-query tile.
// Step r of 4 uses Q2-row (t ^ r) and x-node t:  A[g][t] = wq_g[t^r] wx_g[t],  B[t][n] = V[row t^r][node t][n].
__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
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

// 16-byte asynchronous copy global -> shared through L2 (LDGSTS): bins are written by other SMs
__device__ __forceinline__ void cp_async16(unsigned saddr, const void *g)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(saddr), "l"(g) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// queries per batch of an interior cell = 1 << kCellBatchShift (a batch is a loop over 8-query DMMA
// tiles; its prologue -- cell constants, node rows, the cell's 8 values per lane -- is paid once)
#ifndef PDF_CELLBATCH_SHIFT
#define PDF_CELLBATCH_SHIFT 6
#endif
constexpr int kCellBatchShift = PDF_CELLBATCH_SHIFT;
static_assert(kCellBatchShift >= 5 && kCellBatchShift <= 7, "batch descriptor holds <= 255 queries");

struct BSmem {            // 32-bit shared-window addresses
    unsigned sP;          // uint4 [cap][2] payloads
    unsigned sV;          // double [nqt][4][12]
    unsigned bkey;        // u32 [cap/32 + nfk] descriptor of every batch (<= 32 queries, interior cells <= 1 << kCellBatchShift): fine key | queries << 8 | first slot in `order` << 16
    unsigned fcnt;        // int [nfk]
    unsigned foff;        // int [nfk+1]
    unsigned bstart;      // int [nfk+1]
    unsigned next;        // int [2] batch queue of the item; the item's count
    unsigned order;       // u16 [cap]
};

// ---- B item: one coarse key of one chunk ------------------------------------------------------
__device__ __forceinline__ void b_item(const StreamArgs &A, const BSmem &S, const double *V, int slot, long long chunk_base, int item,
                                       const unsigned long long *a_done, unsigned long long a_target)
{
    const BinDev &B = A.B;
    const GridDev &G = A.G;
    // every tile of A(c) must have been released; one whole warp polls (see a_item)
    if (item >= B.nck) {
        if (threadIdx.x < 32) wait_counter(a_done, a_target);
        cta_sync();
        ovf_item(A, V, slot, chunk_base, item - B.nck);
        return;
    }
    const int ck = B.nck - 1 - item;                       // low-x keys first: the long items must not end the round
    PH_DECL;
    unsigned *counts = A.W.counts + (size_t)slot * B.nck;
    const bool lowx_unit = ck >= B.ncx;
    const int i = lowx_unit ? 0 : ck;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned sPa = S.sP, sVa = S.sV, fcnt = S.fcnt, foff = S.foff, bstart = S.bstart, order = S.order;
    const unsigned nexta = S.next, bkey = S.bkey;

    // stage the key's 4 grid columns: asynchronous copies (no registers, all in flight at once) that
    // run under the count read below
    {
        int c0, c1, c2, c3;
        if (lowx_unit) { c0 = 0; c1 = 1; c2 = 0; c3 = 1; }
        else { c0 = i > 0 ? i - 1 : i; c1 = i; c2 = i + 1; c3 = i + 2 < G.nx ? i + 2 : i + 1; }
        const double2 *V2 = reinterpret_cast<const double2 *>(V);
        const int tot = G.nqtot * 24;                      // double2 units: rows x 4 slots x 6
        for (int e = threadIdx.x; e < tot; e += kBinThreads) {
            int jg = e / 24, r = e - jg * 24, a = r / 6, p = r - a * 6;
            int col = a == 0 ? c0 : a == 1 ? c1 : a == 2 ? c2 : c3;
            cp_async16(sVa + 16u * e, V2 + ((size_t)jg * G.nx + col) * 6 + p);
        }
    }
    // one thread reads the count and the CTA takes that value: every later branch and barrier count
    // of the item depends on it, so it must be the same in all 256 threads
    if (threadIdx.x < 32) {
        wait_counter(a_done, a_target);
        if (threadIdx.x == 0) sts_u32(nexta + 4u, ld_acquire_u32(counts + ck));
    }
    cta_sync();
    const unsigned cnt_u = lds_u32(nexta + 4u);                // not written again before the item's last barrier
    PH(0);
    if (cnt_u == 0u) { cp_async_wait_all(); cta_sync(); return; }
    const int cnt_all = cnt_u > (unsigned)A.cap ? A.cap : (int)cnt_u;
    const char *bin = reinterpret_cast<const char *>(A.W.bins + ((size_t)slot * B.nck + ck) * A.cap);
    // the bin is processed in segments of at most A.scap payloads (what fits in shared memory)
    for (int s0 = 0; s0 < cnt_all; s0 += A.scap) {
    const int cnt = min(A.scap, cnt_all - s0);
    if (s0) cta_sync();                               // the previous segment's batches are done
    for (int e = threadIdx.x; e < cnt * 2; e += kBinThreads) cp_async16(sPa + 16u * e, bin + 16 * (size_t)(2 * s0 + e));
    cp_async_wait_all();
    for (int k = threadIdx.x; k < B.nfk; k += kBinThreads) sts_u32(fcnt + 4u * k, 0u);
    if (threadIdx.x == 0) sts_u32(nexta, 0u);
    cta_sync();
    PH(1);
    // counting sort by fine key: rank kept in the payload's spare word
    for (int e = threadIdx.x; e < cnt; e += kBinThreads) {
        unsigned fk = lds_u32(sPa + 32u * e + 20u);
        PDF_ASSERT(fk < (unsigned)B.nfk);
        unsigned r = atoms_add(fcnt + 4u * fk, 1u);
        sts_u32(sPa + 32u * e + 24u, r);
    }
    cta_sync();
    PH(2);
    if (warp == 0) {                                       // exclusive scans: slots and 32-query batches per key
        int carry_o = 0, carry_b = 0;
        for (int k0 = 0; k0 < B.nfk; k0 += 32) {
            int k = k0 + lane;
            int c = k < B.nfk ? (int)lds_u32(fcnt + 4u * k) : 0;
            const int bsh = (!lowx_unit && k < B.nqt) ? kCellBatchShift : 5;   // interior cells: DMMA tiles, longer batches
            int nb = (c + (1 << bsh) - 1) >> bsh;
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
        __syncwarp();
        for (int k = lane; k < B.nfk; k += 32) {           // batch descriptors
            const int b0 = (int)lds_u32(bstart + 4u * k), b1 = (int)lds_u32(bstart + 4u * (k + 1));
            const int c = (int)lds_u32(fcnt + 4u * k), fo = (int)lds_u32(foff + 4u * k);
            const int bmax = 1 << ((!lowx_unit && k < B.nqt) ? kCellBatchShift : 5);
            for (int bb = b0; bb < b1; ++bb) {
                const int first = (bb - b0) * bmax;
                sts_u32(bkey + 4u * (unsigned)bb, (unsigned)k | ((unsigned)min(bmax, c - first) << 8) | ((unsigned)(fo + first) << 16));
            }
        }
    }
    cta_sync();
    PH(3);
    for (int e = threadIdx.x; e < cnt; e += kBinThreads) {
        uint2 w = make_uint2(lds_u32(sPa + 32u * e + 20u), lds_u32(sPa + 32u * e + 24u));
        unsigned pos = lds_u32(foff + 4u * w.x) + w.y;
        PDF_ASSERT(w.x < (unsigned)B.nfk && pos < (unsigned)cnt);
        asm volatile("st.shared.u16 [%0], %1;" ::"r"(order + 2u * pos), "h"((unsigned short)e) : "memory");
    }
    cta_sync();
    PH(4);

    const int total = (int)lds_u32(bstart + 4u * B.nfk);
    const WCoef kx = weight_coef(G.cx[i], lane & 3);       // x-axis weight of this lane's node, fixed for the unit
    for (;;) {
        int fb = 0;
        if (lane == 0) fb = (int)atoms_add(nexta, 1u);     // batches are handed out dynamically,
        fb = __shfl_sync(0xffffffffu, fb, 0);              // last keys first: the extrapolation classes
        if (fb >= total) break;                            // (long, few lanes) must not form the tail
        fb = total - 1 - fb;
        const unsigned desc = lds_u32(bkey + 4u * (unsigned)fb);
        const int fk = (int)(desc & 0xffu), nact = (int)((desc >> 8) & 0xffu);
        PDF_ASSERT(fk < B.nfk && fb >= 0 && fb < A.scap / 32 + B.nfk && nact >= 1 && nact <= (1 << kCellBatchShift));
        const unsigned ord0 = order + 2u * (desc >> 16);
        if (!lowx_unit && fk < B.nqt) {
            // ---- interior cell (i, fk): DMMA tiles of 8 queries ----
            const int g = lane >> 2, t = lane & 3;
            const CellTab cq = G.cq[fk];
            const WCoef kq = weight_coef(cq, t);
            const int edge_lo = cq.aL == 1.0 ? 1 : 0, edge_hi = cq.aR == 1.0 ? 1 : 0;   // one-sided ends of a sub-grid (q_nodes)
            double b0[4], b1[4];
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const int tr = t ^ r;
                const int row = fk - 1 + tr + (tr == 0 ? edge_lo : 0) - (tr == 3 ? edge_hi : 0);
                const unsigned pn = snode(sVa, row, t);
                b0[r] = lds_f64(pn + 8u * g);
                b1[r] = g < 4 ? lds_f64(pn + 8u * (8 + g)) : 0.0;
            }
            // the next tile's abscissae are fetched (two dependent shared-memory loads) under this tile's arithmetic
            double txn = 0.0, tqn = 0.0;
            unsigned idxn = 0;
            bool vn = g < nact;
            if (vn) {
                unsigned short e16;
                asm volatile("ld.shared.u16 %0, [%1];" : "=h"(e16) : "r"(ord0 + 2u * g) : "memory");
                PDF_ASSERT(e16 < cnt);
                const unsigned pe = sPa + 32u * e16;
                const double2 ab = lds_v2f64(pe);
                txn = ab.x; tqn = ab.y;
                idxn = lds_u32(pe + 16u);
            }
            for (int m0 = 0; m0 < nact; m0 += 8) {
                const bool valid = vn;
                const double tx = txn, tq = tqn;
                const unsigned idx = idxn;
                {
                    const int qi = m0 + 8 + g;
                    vn = qi < nact;
                    txn = 0.0; tqn = 0.0;
                    if (vn) {
                        unsigned short e16;
                        asm volatile("ld.shared.u16 %0, [%1];" : "=h"(e16) : "r"(ord0 + 2u * qi) : "memory");
                        PDF_ASSERT(e16 < cnt);
                        const unsigned pe = sPa + 32u * e16;
                        const double2 ab = lds_v2f64(pe);
                        txn = ab.x; tqn = ab.y;
                        idxn = lds_u32(pe + 16u);
                    }
                }
                const double wx = valid ? weight_eval(kx, tx) : 0.0;
                const double wq0 = weight_eval(kq, tq);
                const double wq1 = __shfl_xor_sync(0xffffffffu, wq0, 1);
                const double wq2 = __shfl_xor_sync(0xffffffffu, wq0, 2);
                const double wq3 = __shfl_xor_sync(0xffffffffu, wq0, 3);
                double d00 = 0.0, d01 = 0.0, d10 = 0.0, d11 = 0.0;
                const double a0 = wq0 * wx, a1 = wq1 * wx, a2 = wq2 * wx, a3 = wq3 * wx;
                dmma884(d00, d01, a0, b0[0]); dmma884(d10, d11, a0, b1[0]);
                dmma884(d00, d01, a1, b0[1]); dmma884(d10, d11, a1, b1[1]);
                dmma884(d00, d01, a2, b0[2]); dmma884(d10, d11, a2, b1[2]);
                dmma884(d00, d01, a3, b0[3]); dmma884(d10, d11, a3, b1[3]);
                if (valid) {                               // lane holds flavours 2t, 2t+1, 8+2t, 9+2t of its query
                    PDF_ASSERT(chunk_base + idx < A.n);
                    double *rp = A.out + (chunk_base + idx) * A.ld;
                    if (A.identity) {
                        rp[2 * t] = d00; rp[2 * t + 1] = d01;
                        if (t < 2) rp[8 + 2 * t] = d10;
                        if (t == 0) rp[9] = d11;
                    } else {
                        for (int p = 0; p < A.cm.n; ++p) {
                            const int c = A.cm.col[p];
                            if (c < 0) { if (t == 0) rp[p] = 0.0; continue; }
                            if (((c & 7) >> 1) == t) rp[p] = (c & 8) ? ((c & 1) ? d11 : d10) : ((c & 1) ? d01 : d00);
                        }
                    }
                }
            }
            continue;
        }
        // ---- extrapolation classes: one query per lane, broadcast operands ----
        const bool active = lane < nact;
        double pa = 0.0, pb = 0.0;
        unsigned idx = 0;
        if (active) {
            unsigned short e16;
            asm volatile("ld.shared.u16 %0, [%1];" : "=h"(e16) : "r"(ord0 + 2u * lane) : "memory");
            const unsigned pe = sPa + 32u * e16;
            double2 ab = lds_v2f64(pe);
            pa = ab.x; pb = ab.y;
            idx = lds_u32(pe + 16u);
        }
        double acc[kNF];
        eval_extrap_s(G, B, sVa, lowx_unit, i, fk, pa, pb, acc);
        if (active) {                                      // 5 % of the queries: one row per lane
            double *rp = A.out + (chunk_base + idx) * A.ld;
            if (A.identity) {
#pragma unroll
                for (int f = 0; f < kNF; ++f) rp[f] = acc[f];
            } else {
                for (int p = 0; p < A.cm.n; ++p) {
                    const int c = A.cm.col[p];
                    double v = 0.0;
#pragma unroll
                    for (int f = 0; f < kNF; ++f) v = c == f ? acc[f] : v;
                    rp[p] = v;
                }
            }
        }
        __syncwarp();
    }
    if (threadIdx.x == 0) { PH(5); }
    __syncwarp();
    cta_sync();
    PH(6);
    }   // segments
    cta_sync();
    if (threadIdx.x == 0) counts[ck] = 0u;                 // the bin is empty again for the ring
}

// ---- the persistent kernel -----------------------------------------------------------------------
// dynamic shared memory: [knots | LUTs | item region]; the item region is used by A items as
// (cnt, base) and by B items as (payloads, columns, stage, sort tables)
__host__ __device__ inline size_t bsmem_item_bytes(int nqt, int nck, int nfk, int cap)
{
    size_t b = (size_t)cap * 32;                                        // sP
    b += (size_t)nqt * 4 * kNFP * sizeof(double);                       // sV
    b += ((size_t)(cap / 32 + nfk) * 4 + 15) / 16 * 16;                 // bkey (batch descriptors)
    b += (size_t)(3 * nfk + 8) * sizeof(int);                           // fcnt, foff, bstart, next
    b += ((size_t)cap * sizeof(unsigned short) + 15) / 16 * 16;         // order
    size_t a = (size_t)kTileA * 32 + (size_t)2 * nck * sizeof(unsigned); // A items: payloads, cnt, base
    return (b > a ? b : a) + 32;
}

__global__ void __launch_bounds__(kBinThreads, PDF_MINB) k_pdf_stream(const __grid_constant__ StreamArgs A)
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
    cta_sync();
    const unsigned region_a = (unsigned)__cvta_generic_to_shared(region);   // everything below derives from this one address
    const unsigned tables_a = (unsigned)__cvta_generic_to_shared(smem_raw);

    unsigned long long *ctrl = A.W.ctrl;
    const unsigned long long TA = A.ta, TB = A.B.nitems, per = TA + TB;
    const int nchunks = A.ctab ? __ldg(A.nchunks_dev) : A.nchunks;
    const unsigned long long total = (unsigned long long)nchunks * per;
    unsigned long long err_local = 0;

    // the next ticket is fetched while the current item runs (a global atomic is ~1 us)
    unsigned long long next_t = 0;
    if (threadIdx.x == 0) next_t = atomicAdd(ctrl, 1ULL);
    for (;;) {
        if (threadIdx.x == 0) s_ticket = next_t;
        cta_sync();
        const unsigned long long t = s_ticket;
        cta_sync();
        if (t >= total) break;
        if (threadIdx.x == 0) next_t = atomicAdd(ctrl, 1ULL);      // consumed at the top of the next round
        // ticket order, lag L = kLag rounds:  round r = [A(r) tiles | B(r-L) items]; B(c) is handed out
        // L rounds after A(c), so its tiles were claimed >= L waves earlier and the wait below is ~never taken
        bool isA; long long c; int sub;
        {
            const unsigned long long RA = (unsigned long long)(nchunks < kLag ? nchunks : kLag);   // A-only rounds
            const unsigned long long F = (unsigned long long)nchunks - RA;                             // full rounds
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
        long long chunk_base = c * A.chunk, chunk_end = chunk_base + A.chunk;
        if (chunk_end > A.n) chunk_end = A.n;
        const double *V = A.G.V;
        if (A.ctab) {                                              // a-8: the chunk is a piece of one member's run
            const int4 ce = __ldg(reinterpret_cast<const int4 *>(A.ctab) + c);
            chunk_base = ce.x; chunk_end = (long long)ce.x + ce.y;
            V += (size_t)ce.z * A.G.memstride;
        }
        if (isA) {
            // (the wait for the ring slot is inside the item, under its loads)
#ifdef PDF_PHASES
            long long ph_t;
#endif
            SmemTables T;
            T.xk = tables_a; T.qk = T.xk + 8u * A.G.nx; T.lutx = T.qk + 8u * A.G.nqtot; T.lutq = T.lutx + 2u * kLutSize;
            ASmem SA;
            SA.pay = region_a; SA.cnt = region_a + (unsigned)kTileA * 32u; SA.base = SA.cnt + 4u * A.B.nck;
            a_item(A, T, SA, slot, chunk_base, chunk_end, sub, &err_local, b_done, gen * TB);
#ifdef PDF_PHASES
            ph_t = clock64();
#endif
            // release: the barrier orders every thread's stores before thread 0's gpu-scope fence, and the
            // fence is cumulative (the pattern of a grid-wide barrier: bar.sync; one thread fences and signals)
            cta_sync();
            PH(20);
            if (threadIdx.x == 0) { __threadfence(); atomicAdd(a_done, 1ULL); }
        } else {
#ifdef PDF_PHASES
            long long bt0 = clock64();
#endif
            BSmem SB;
            SB.sP = region_a;
            SB.sV = region_a + (unsigned)A.scap * 32u;
            SB.fcnt = SB.sV + (unsigned)A.G.nqtot * (4u * kNFP * 8u);
            SB.foff = SB.fcnt + 4u * (A.B.nfk + 1);
            SB.bstart = SB.foff + 4u * (A.B.nfk + 1);
            SB.next = SB.bstart + 4u * (A.B.nfk + 2);
            SB.order = SB.next + 8u;
            SB.bkey = SB.order + 2u * ((A.scap + 7) & ~7);
            b_item(A, SB, V, slot, chunk_base, sub, a_done, (gen + 1) * TA);
#ifdef PDF_PHASES
            if (threadIdx.x == 0) {
                unsigned long long dt = (unsigned long long)(clock64() - bt0);
                atomicMax(A.W.ctrl + 256 + 16, dt);
                if (dt > 100000ULL) atomicAdd(A.W.ctrl + 256 + 17, 1ULL);
                if (dt > 200000ULL) atomicAdd(A.W.ctrl + 256 + 18, 1ULL);
                if (dt > 200000ULL) A.W.ctrl[256 + 19] = (unsigned long long)sub;
            }
            long long ph_t = clock64();
#endif
            cta_sync();
            PH(7);
            if (threadIdx.x == 0) {
                __threadfence();
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
