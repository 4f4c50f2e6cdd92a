// pdf_binned_eval.cuh -- B items (warp-coherent evaluation) and the persistent kernel itself.
#pragma once

namespace pdfg {

// acc[f] += w * V[node][f] for the 11 flavours of one node row (12 doubles, 16-byte aligned).
// Every lane passes the SAME address: each 16-byte load is one broadcast wavefront for 32 queries.
__device__ __forceinline__ void node_fma(const double *__restrict__ p, double w, double acc[kNF])
{
    double2 v0 = ldg_nc_d2(p), v1 = ldg_nc_d2(p + 2), v2 = ldg_nc_d2(p + 4);
    double2 v3 = ldg_nc_d2(p + 6), v4 = ldg_nc_d2(p + 8), v5 = ldg_nc_d2(p + 10);
    acc[0] = fma(w, v0.x, acc[0]); acc[1] = fma(w, v0.y, acc[1]);
    acc[2] = fma(w, v1.x, acc[2]); acc[3] = fma(w, v1.y, acc[3]);
    acc[4] = fma(w, v2.x, acc[4]); acc[5] = fma(w, v2.y, acc[5]);
    acc[6] = fma(w, v3.x, acc[6]); acc[7] = fma(w, v3.y, acc[7]);
    acc[8] = fma(w, v4.x, acc[8]); acc[9] = fma(w, v4.y, acc[9]);
    acc[10] = fma(w, v5.x, acc[10]);
}

__device__ __forceinline__ const double *node_ptr(const GridDev &G, int jrow, int icol)
{
    return G.V + ((size_t)jrow * G.nx + icol) * kNFP;
}

struct AxisNodes { int n[4]; };
__device__ __forceinline__ AxisNodes x_nodes(const GridDev &G, int i)
{
    AxisNodes a; a.n[0] = i > 0 ? i - 1 : i; a.n[1] = i; a.n[2] = i + 1; a.n[3] = i + 2 < G.nx ? i + 2 : i + 1;
    return a;
}
__device__ __forceinline__ AxisNodes q_nodes(const CellTab &c, int jg)
{
    AxisNodes a; a.n[0] = (c.aL == 1.0) ? jg : jg - 1; a.n[1] = jg; a.n[2] = jg + 1; a.n[3] = (c.aR == 1.0) ? jg + 1 : jg + 2;
    return a;
}

// C-6: 16-node tensor sum in cell (i, jg)
__device__ __forceinline__ void eval_interior(const GridDev &G, int i, int jg, double tx, double tq, double acc[kNF])
{
    CellTab cq = G.cq[jg];
    double wx[4], wq[4];
    hermite_weights(tx, G.cx[i], wx);
    hermite_weights(tq, cq, wq);
    AxisNodes xn = x_nodes(G, i), qn = q_nodes(cq, jg);
#pragma unroll
    for (int f = 0; f < kNF; ++f) acc[f] = 0.0;
#pragma unroll
    for (int b = 0; b < 4; ++b)
#pragma unroll
        for (int a = 0; a < 4; ++a) node_fma(node_ptr(G, qn.n[b], xn.n[a]), wq[b] * wx[a], acc);
}

// sum_b wq[b] V[col][rows of cell jg]  (x fixed on a knot column)
__device__ __forceinline__ void eval_column(const GridDev &G, int col, int jg, double tq, double acc[kNF])
{
    CellTab cq = G.cq[jg];
    double wq[4];
    hermite_weights(tq, cq, wq);
    AxisNodes qn = q_nodes(cq, jg);
#pragma unroll
    for (int f = 0; f < kNF; ++f) acc[f] = 0.0;
#pragma unroll
    for (int b = 0; b < 4; ++b) node_fma(node_ptr(G, qn.n[b], col), wq[b], acc);
}

// sum_a wx[a] V[cols of cell i][row]  (Q2 fixed on a knot row)
__device__ __forceinline__ void eval_row(const GridDev &G, int i, int jrow, double tx, double acc[kNF])
{
    double wx[4];
    hermite_weights(tx, G.cx[i], wx);
    AxisNodes xn = x_nodes(G, i);
#pragma unroll
    for (int f = 0; f < kNF; ++f) acc[f] = 0.0;
#pragma unroll
    for (int a = 0; a < 4; ++a) node_fma(node_ptr(G, jrow, xn.n[a]), wx[a], acc);
}

__device__ __forceinline__ void load_node(const GridDev &G, int jrow, int icol, double acc[kNF])
{
#pragma unroll
    for (int f = 0; f < kNF; ++f) acc[f] = 0.0;
    node_fma(node_ptr(G, jrow, icol), 1.0, acc);
}

// class dispatch: key -> values of the 11 flavours for payload (a, b).  Warp-uniform branches.
__device__ __noinline__ void eval_extrap(const GridDev &G, const BinDev &B, int key, double pa, double pb, double acc[kNF])
{
    double e0[kNF], e1[kNF];
    int last = G.nqtot - 1;
    if (key >= B.k_lh) {                                   // low-x & high-Q (L1744): x rule, then Q rule
        double e2[kNF], e3[kNF];
        load_node(G, last - 1, 0, e0); load_node(G, last - 1, 1, e1);
        load_node(G, last, 0, e2); load_node(G, last, 1, e3);
#pragma unroll
        for (int f = 0; f < kNF; ++f)
            acc[f] = continue_two(continue_two(e0[f], e1[f], pa), continue_two(e2[f], e3[f], pa), pb);
    } else if (key >= B.k_ll) {                            // low-x & low-Q
        double e2[kNF], e3[kNF];
        load_node(G, 0, 0, e0); load_node(G, 0, 1, e1);
        eval_column(G, 0, B.jgplus, B.tqplus, e2); eval_column(G, 1, B.jgplus, B.tqplus, e3);
#pragma unroll
        for (int f = 0; f < kNF; ++f)
            acc[f] = lowq_continue(continue_two(e0[f], e1[f], pa), continue_two(e2[f], e3[f], pa), pb);
    } else if (key >= B.k_lowq) {                          // low-Q (C-9): pa = t_x, pb = r
        int i = key - B.k_lowq;
        eval_row(G, i, 0, pa, e0);
        eval_interior(G, i, B.jgplus, pa, B.tqplus, e1);
#pragma unroll
        for (int f = 0; f < kNF; ++f) acc[f] = lowq_continue(e0[f], e1[f], pb);
    } else if (key >= B.k_highq) {                         // high-Q (C-8): pa = t_x, pb = theta_q
        int i = key - B.k_highq;
        eval_row(G, i, last - 1, pa, e0);
        eval_row(G, i, last, pa, e1);
#pragma unroll
        for (int f = 0; f < kNF; ++f) acc[f] = continue_two(e0[f], e1[f], pb);
    } else {                                               // low-x (C-7): pa = theta_x, pb = t_q
        int jg = key - B.k_lowx;
        eval_column(G, 0, jg, pb, e0);
        eval_column(G, 1, jg, pb, e1);
#pragma unroll
        for (int f = 0; f < kNF; ++f) acc[f] = continue_two(e0[f], e1[f], pa);
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
    double *stage;        // [kBinWarps][32*kNF]
    unsigned *sidx;       // [kBinWarps][32]
    int *bstart;          // [kKeysPerItem+1]
    int *cnt;             // [kKeysPerItem]
};

__device__ __forceinline__ void b_item(const StreamArgs &A, const BSmem &S, int slot, long long chunk_base, int item)
{
    const BinDev &B = A.B;
    BinItem it = B.items[item];
    if (it.key_begin < 0) { ovf_item(A, slot, chunk_base, -it.key_begin - 1); return; }
    unsigned *counts = A.W.counts + (size_t)slot * B.nkeys;
    const Payload *bins = A.W.bins + (size_t)slot * B.nkeys * A.cap;
    const int nk = it.key_end - it.key_begin;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (warp == 0) {                                       // batches per key, prefix-summed
        unsigned c = lane < nk ? __ldcg(counts + it.key_begin + lane) : 0u;
        if (c > (unsigned)A.cap) c = A.cap;
        int nb = (int)((c + 31) >> 5), incl = nb;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { int v = __shfl_up_sync(0xffffffffu, incl, d); if (lane >= d) incl += v; }
        if (lane < nk) { S.cnt[lane] = (int)c; S.bstart[lane + 1] = incl; }
        if (lane == 0) S.bstart[0] = 0;
    }
    __syncthreads();
    const int total = S.bstart[nk];
    double *stage = S.stage + warp * (32 * kNF);
    unsigned *sidx = S.sidx + warp * 32;
    int k = 0;
    for (int fb = warp; fb < total; fb += kBinWarps) {
        while (S.bstart[k + 1] <= fb) ++k;
        const int key = it.key_begin + k, cnt = S.cnt[k];
        const int lslot = (fb - S.bstart[k]) * 32 + lane;
        const bool active = lslot < cnt;
        const int nact = min(32, cnt - (fb - S.bstart[k]) * 32);
        double pa = 0.0, pb = 0.0;
        unsigned idx = 0;
        if (active) {
            const Payload *src = bins + (size_t)key * A.cap + lslot;
            double2 ab = __ldcg(reinterpret_cast<const double2 *>(src));
            uint2 ii = __ldcg(reinterpret_cast<const uint2 *>(src) + 2);
            pa = ab.x; pb = ab.y; idx = ii.x;
        }
        double acc[kNF];
        if (key < B.k_lowx) {
            int jg = key / B.ncx, i = key - jg * B.ncx;
            eval_interior(A.G, i, jg, pa, pb, acc);
        } else {
            eval_extrap(A.G, B, key, pa, pb, acc);
        }
        // transpose through shared memory so that whole 88-byte rows leave in coalesced stores
#pragma unroll
        for (int f = 0; f < kNF; ++f) stage[lane * kNF + f] = acc[f];
        sidx[lane] = idx;
        __syncwarp();
        if (A.identity) {
            const int tot = nact * kNF;
#pragma unroll
            for (int itx = 0; itx < kNF; ++itx) {
                int e = itx * 32 + lane;
                if (e < tot) {
                    int r = e / kNF, p = e - r * kNF;
                    A.out[(chunk_base + sidx[r]) * A.ld + p] = stage[e];
                }
            }
        } else {
            const int np = A.cm.n, tot = nact * np;
            for (int e = lane; e < tot; e += 32) {
                int r = e / np, p = e - r * np, c = A.cm.col[p];
                A.out[(chunk_base + sidx[r]) * A.ld + p] = c < 0 ? 0.0 : stage[r * kNF + c];
            }
        }
        __syncwarp();
    }
    __syncthreads();
    if (threadIdx.x < nk) counts[it.key_begin + threadIdx.x] = 0u;   // bins are empty again for the ring
}

// ---- the persistent kernel -----------------------------------------------------------------------
__global__ void __launch_bounds__(kBinThreads, 2) k_pdf_stream(const __grid_constant__ StreamArgs A)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *s_xk = reinterpret_cast<double *>(smem_raw);
    double *s_qk = s_xk + A.G.nx;
    double *s_stage = s_qk + A.G.nqtot;
    unsigned *s_idx = reinterpret_cast<unsigned *>(s_stage + kBinWarps * 32 * kNF);
    int *s_bstart = reinterpret_cast<int *>(s_idx + kBinWarps * 32);
    int *s_cnt = s_bstart + kKeysPerItem + 1;
    short *s_lutx = reinterpret_cast<short *>(s_cnt + kKeysPerItem + 1);
    short *s_lutq = s_lutx + kLutSize;
    __shared__ unsigned long long s_ticket;

    for (int i = threadIdx.x; i < A.G.nx; i += kBinThreads) s_xk[i] = A.G.xk[i];
    for (int i = threadIdx.x; i < A.G.nqtot; i += kBinThreads) s_qk[i] = A.G.qk[i];
    for (int i = threadIdx.x; i < kLutSize; i += kBinThreads) { s_lutx[i] = A.B.lutx[i]; s_lutq[i] = A.B.lutq[i]; }
    __syncthreads();
    SmemTables T{s_xk, s_qk, s_lutx, s_lutq};
    BSmem S{s_stage, s_idx, s_bstart, s_cnt};

    unsigned long long *ctrl = A.W.ctrl;
    const unsigned long long TA = A.ta, TB = A.B.nitems, per = TA + TB;
    const unsigned long long total = (unsigned long long)A.nchunks * per;
    unsigned long long err_local = 0;

    for (;;) {
        if (threadIdx.x == 0) s_ticket = atomicAdd(ctrl, 1ULL);
        __syncthreads();
        const unsigned long long t = s_ticket;
        __syncthreads();
        if (t >= total) break;
        // ticket order: A(0) | A(1) B(0) | A(2) B(1) | ... | B(last)
        bool isA; long long c; int sub;
        if (t < TA) { isA = true; c = 0; sub = (int)t; }
        else {
            unsigned long long tp = t - TA, round = 1 + tp / per, w = tp % per;
            if ((long long)round < A.nchunks) { isA = w < TA; c = isA ? (long long)round : (long long)round - 1; sub = (int)(isA ? w : w - TA); }
            else { isA = false; c = A.nchunks - 1; sub = (int)w; if (w >= TB) continue; }
        }
        const int slot = (int)(c % kRing);
        const unsigned long long gen = (unsigned long long)(c / kRing);
        unsigned long long *a_done = ctrl + 8 + slot * 4, *b_fin = a_done + 1, *b_done = a_done + 2;
        const long long chunk_base = c * A.chunk;
        if (isA) {
            if (threadIdx.x == 0 && gen > 0) wait_counter(b_done, gen * TB);   // ring slot drained
            __syncthreads();
            a_item(A, T, slot, chunk_base, sub, &err_local);
            __threadfence();
            __syncthreads();
            if (threadIdx.x == 0) atomicAdd(a_done, 1ULL);
        } else {
            if (threadIdx.x == 0) wait_counter(a_done, (gen + 1) * TA);        // every tile of A(c) released
            __syncthreads();
            b_item(A, S, slot, chunk_base, sub);
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
