// pdf_binned_host.cuh -- host side of the binned path: key geometry, work list, launch.
#pragma once
#include <cmath>
#include <vector>

namespace pdfg {

constexpr long long kAutoMinN = 1 << 15;      // PDF_PATH_AUTO: below this the direct path is used
constexpr long long kMemberMinPer = 1 << 14;  // PDF_PATH_AUTO with member ids: queries per member below which the direct path is used

// cell and t_q of 1.01*Q2min with the device log (C-9); res = {jg, t, in_range}
__global__ void k_q2plus(GridDev G, double *res)
{
    if (threadIdx.x || blockIdx.x) return;
    double q = G.q2plus;
    if (q > G.qk[G.nqtot - 1]) { res[2] = 0.0; return; }
    int j, jg;
    q_locate(G, q, j, jg);
    res[0] = (double)jg;
    res[1] = (q == G.qk[jg + 1]) ? 1.0 : (log(q) - G.cq[jg].lo_log) * G.cq[jg].inv_d;
    res[2] = 1.0;
}

inline void binned_plan_free(BinnedPlan &p)
{
    cudaFree(p.d_lutx); cudaFree(p.d_lutq); cudaFree(p.d_plus);
    p.d_lutx = p.d_lutq = nullptr; p.d_plus = nullptr; p.usable = false;
}

inline size_t binned_smem_bytes(int nx, int nqtot, int nck, int nfk, int cap)
{
    return sizeof(double) * (nx + nqtot) + sizeof(short) * 2 * kLutSize + 64 + bsmem_item_bytes(nqtot, nck, nfk, cap);
}

// builds LUTs and the key geometry; leaves usable = false when the grid does not fit the
// specialised path (then every call takes the direct path)
inline int binned_plan_init(BinnedPlan &p, const GridDev &G, const std::vector<double> &xk,
                            const std::vector<double> &qk, const std::vector<int> &qoff)
{
    p.usable = false;
    const int nx = G.nx, nqt = G.nqtot;
    if (G.nflav != kNF || G.nfp != kNFP) return 0;
    if (nx - 1 + kLowXSplit > kMaxCK || nqt + 2 > kMaxFK || nx < 2) return 0;
    BinDev &d = p.dev;
    d.ncx = nx - 1; d.nqt = nqt;
    d.nck = d.ncx + kLowXSplit;
    d.nfk = nqt + 2;
    d.nitems = d.nck + kOvfItems;

    // search LUTs: bucket b covers ln v in [l0 + b/scale, l0 + (b+1)/scale); entry = a cell at its lower edge
    auto make_lut = [](const std::vector<double> &k, bool last_le, double &scale, std::vector<short> &lut) {
        const int m = (int)k.size();
        double l0 = std::log(k.front()), l1 = std::log(k.back());
        scale = kLutSize / (l1 - l0) * (1.0 - 1e-12);
        lut.resize(kLutSize);
        int c = 0;
        for (int b = 0; b < kLutSize; ++b) {
            double edge = std::exp(l0 + b / scale);
            int lim = last_le ? m - 1 : m - 2;
            while (c < lim && k[c + 1] <= edge) ++c;
            lut[b] = (short)c;
        }
    };
    std::vector<short> lx, lq;
    make_lut(xk, false, d.lutx_scale, lx);
    make_lut(qk, true, d.lutq_scale, lq);

    if (cudaMalloc((void **)&p.d_lutx, sizeof(short) * kLutSize) != cudaSuccess) return PDF_ENOMEM;
    if (cudaMalloc((void **)&p.d_lutq, sizeof(short) * kLutSize) != cudaSuccess) return PDF_ENOMEM;
    if (cudaMalloc((void **)&p.d_plus, sizeof(double) * 4) != cudaSuccess) return PDF_ENOMEM;
    cudaMemcpy(p.d_lutx, lx.data(), sizeof(short) * kLutSize, cudaMemcpyHostToDevice);
    cudaMemcpy(p.d_lutq, lq.data(), sizeof(short) * kLutSize, cudaMemcpyHostToDevice);
    k_q2plus<<<1, 32>>>(G, p.d_plus);
    double res[3] = {0, 0, 0};
    if (cudaMemcpy(res, p.d_plus, sizeof res, cudaMemcpyDeviceToHost) != cudaSuccess) return PDF_ECUDA;
    if (res[2] != 1.0) return 0;                           // 1.01*Q2min beyond the grid: direct path only
    d.jgplus = (int)res[0]; d.tqplus = res[1];
    d.lutx = p.d_lutx; d.lutq = p.d_lutq;

    // largest shared-memory footprint (cap = kMaxCap) must fit one CTA; the launch computes the real one
    size_t smem_max = binned_smem_bytes(nx, nqt, d.nck, d.nfk, kMaxCap);
    if (smem_max > 200 * 1024) return 0;
    if (cudaFuncSetAttribute(k_pdf_stream, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max) != cudaSuccess) return 0;
    (void)qoff;
    p.usable = true;
    return 0;
}

inline bool binned_qualifies(const BinnedPlan &p, const ColMap &, const int *member) { return p.usable && !member; }
inline bool binned_members_qualifies(const BinnedPlan &p, const GridDev &G, const int *member)
{
    return p.usable && member && G.nmem > 1 && G.nmem <= kMemMax;
}
// ---- luminosity on top of the binned path ------------------------------------------------------
// pdf_lumi in slices of kLumiSlice events: xf(x1,Q2) and xf(x2,Q2) of the slice by two runs of the
// persistent binned kernel into two scratch arrays, then k_lumi_combine reduces the 11 x 11 coupling
// per event in registers.  The per-flavour values of a slice make one round trip through the
// scratch (L2 / HBM); the fused single-kernel form is k_lumi_direct (PDF_PATH_DIRECT).
constexpr long long kLumiSlice = 1LL << 24;   // 2^22: 30.4 ms, 2^23: 29.0 ms, 2^24: 28.1 ms per 1e8 events (fewer pipeline ramps)

struct CouplingParam { double c[kNF * kNF]; };            // passed by value: constant-bank operands

__global__ void __launch_bounds__(256)
k_lumi_combine(const __grid_constant__ CouplingParam C, long long n, const double *__restrict__ f1,
               const double *__restrict__ f2, const double *__restrict__ x1, const double *__restrict__ x2,
               const double *__restrict__ w, double *__restrict__ out, unsigned long long *err_count)
{
    long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    const double a = __ldcs(x1 + e), b = __ldcs(x2 + e);
    double h[kNF];
    const double inv_b = 1.0 / b, inv_a = 1.0 / a;
#pragma unroll
    for (int j = 0; j < kNF; ++j) h[j] = __ldcs(f2 + e * kNF + j) * inv_b;
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < kNF; ++i) {
        double row = 0.0;
#pragma unroll
        for (int j = 0; j < kNF; ++j) row = fma(C.c[i * kNF + j], h[j], row);
        acc = fma(__ldcs(f1 + e * kNF + i) * inv_a, row, acc);
    }
    const double v = __ldcs(w + e) * acc;
    if (!(finite_pos(a) && finite_pos(b)) || v != v) {
        // an invalid parton made its whole row NaN (C-10); the event counts once
        if (isnan(__ldcs(f1 + e * kNF)) || isnan(__ldcs(f2 + e * kNF))) { atomicAdd(err_count, 1ULL); out[e] = qnan(); return; }
    }
    out[e] = v;
}

inline bool binned_lumi_qualifies(const BinnedPlan &p) { return p.usable; }
// two scratch arrays of min(n, kLumiSlice) rows
inline size_t binned_lumi_scratch_bytes(const BinnedPlan &p, long long n)
{
    const long long slice = n < kLumiSlice ? n : kLumiSlice;
    return p.usable ? (size_t)2 * slice * kNF * sizeof(double) + 512 : 0;
}

// one memset + one persistent kernel for the whole call
template <typename Scope>
inline int binned_xfxq2(const GridDev &G, const BinnedPlan &p, const ColMap &cm, long long n, const double *x,
                        const double *q2, double *out, long long ld, void *ws, size_t ws_bytes, long long chunk_opt,
                        cudaStream_t s, int count_err = 1, const int *ctab = nullptr, const int *nchunks_dev = nullptr)
{
    if (binned_workspace_bytes(p, n, chunk_opt) > ws_bytes) return PDF_EWORKSPACE;
    StreamArgs A;
    A.ctab = ctab; A.nchunks_dev = nchunks_dev;
    A.G = G; A.B = p.dev; A.cm = cm;
    A.chunk = binned_chunk(p, n, chunk_opt);
    A.cap = binned_cap(p, A.chunk);
    A.scap = binned_scap(p, A.chunk);
    binned_carve(p, ws, A.chunk, A.cap, A.W);
    A.x = x; A.q2 = q2; A.out = out; A.n = n; A.ld = ld;
    A.nchunks = (int)((n + A.chunk - 1) / A.chunk);
    A.ta = (int)(A.chunk / kTileA);
    A.identity = cm.n == kNF;
    for (int f = 0; f < kNF && A.identity; ++f) A.identity = cm.col[f] == f;
    A.zfill = (ld == cm.n) ? 1 : 0;
    A.count_err = count_err;
#ifdef PDF_NOZFILL
    A.zfill = 0;
#endif
    size_t zero_bytes = (size_t)((char *)A.W.bins - (char *)A.W.ctrl);      // ctrl + counts + ovf_count
    if (cudaMemsetAsync(A.W.ctrl, 0, zero_bytes, s) != cudaSuccess) return PDF_ECUDA;
    size_t smem = binned_smem_bytes(G.nx, G.nqtot, p.dev.nck, p.dev.nfk, A.scap);
    int per_sm = 0, dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_pdf_stream, kBinThreads, smem) != cudaSuccess || per_sm < 1)
        return PDF_ECUDA;
    unsigned long long max_ctas = (unsigned long long)per_sm * sms;         // all CTAs must be co-resident
    // with a chunk table the chunk count is on the device: the launch takes its upper bound
    const long long nch = ctab ? member_max_chunks(n, A.chunk, G.nmem) : (long long)A.nchunks;
    unsigned long long tickets = (unsigned long long)nch * (A.ta + p.dev.nitems);
    unsigned grid = (unsigned)(tickets < max_ctas ? tickets : max_ctas);
    {
        Scope sc(s, "k_pdf_stream");
        k_pdf_stream<<<grid, kBinThreads, smem, s>>>(A);
    }
    return cudaGetLastError() == cudaSuccess ? PDF_OK : PDF_ECUDA;
}

// a-8 on the binned path (pdf_members.cuh): per slice, partition by member, one persistent-kernel
// run over the chunk table into the sorted scratch rows, gather back to query order
inline size_t binned_members_bytes(const BinnedPlan &p, const GridDev &G, long long n, long long chunk_opt, int npid)
{
    if (!p.usable || G.nmem < 2 || G.nmem > kMemMax) return 0;
    const long long slice = member_slice(n);
    const long long chunk = binned_chunk(p, slice, chunk_opt);
    return binned_workspace_bytes(p, slice, chunk_opt) + member_scratch_bytes(slice, chunk, G.nmem, npid) + 256;
}

template <typename Scope>
inline int binned_members(const GridDev &G, const BinnedPlan &p, const ColMap &cm, long long n, const double *x,
                          const double *q2, const int *member, double *out, long long ld, void *ws, size_t ws_bytes,
                          long long chunk_opt, cudaStream_t s)
{
    if (binned_members_bytes(p, G, n, chunk_opt, cm.n) > ws_bytes) return PDF_EWORKSPACE;
    const long long slice = member_slice(n);
    const long long chunk = binned_chunk(p, slice, chunk_opt);
    const size_t ws_x = binned_workspace_bytes(p, slice, chunk_opt);
    MemberWs M;
    member_carve((char *)ws + ws_x, slice, chunk, G.nmem, M);
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const size_t hsm = sizeof(unsigned) * (size_t)G.nmem;
    if (cudaFuncSetAttribute(k_member_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)member_scatter_smem(G.nmem)) != cudaSuccess)
        return PDF_ECUDA;
    for (long long off = 0; off < n; off += slice) {
        const long long m = n - off < slice ? n - off : slice;
        if (cudaMemsetAsync(M.hist, 0, hsm, s) != cudaSuccess) return PDF_ECUDA;
        {
            Scope sc(s, "k_member_hist");
            long long want = (m + 2047) / 2048;
            k_member_hist<<<(unsigned)(want < sms * 8 ? want : sms * 8), 256, hsm, s>>>(member + off, m, G.nmem, M.hist);
        }
        {
            Scope sc(s, "k_member_plan");
            k_member_plan<<<1, 256, hsm, s>>>(M.hist, G.nmem, (int)chunk, M.cursor, M.ctab, M.nchunks);
        }
        {
            Scope sc(s, "k_member_scatter");
            k_member_scatter<<<(unsigned)((m + kMemScatThreads * kMemTileQ - 1) / (kMemScatThreads * kMemTileQ)), kMemScatThreads, member_scatter_smem(G.nmem), s>>>(
                x + off, q2 + off, member + off, m, G.nmem, M.cursor, M.xs, M.q2s, M.inv);
        }
        int rc = binned_xfxq2<Scope>(G, p, cm, m, M.xs, M.q2s, M.tmp, cm.n, ws, ws_x, chunk_opt, s, 1, M.ctab, M.nchunks);
        if (rc) return rc;
        {
            Scope sc(s, "k_member_gather");
            long long want = (m + 255) / 256;
            k_member_gather<<<(unsigned)(want < sms * 16 ? want : sms * 16), 256, 0, s>>>(M.tmp, M.inv, m, cm.n, out + off * ld, ld,
                                                                                       G.err_count);
        }
    }
    return cudaGetLastError() == cudaSuccess ? PDF_OK : PDF_ECUDA;
}

template <typename Scope>
inline int binned_lumi(const GridDev &G, const BinnedPlan &p, const double *hostC, long long n, const double *x1,
                       const double *x2, const double *q2, const double *w, double *out, void *ws, size_t ws_bytes,
                       long long chunk_opt, cudaStream_t s)
{
    const long long slice = n < kLumiSlice ? n : kLumiSlice;
    const size_t ws_x = binned_workspace_bytes(p, slice, chunk_opt);
    if (ws_x + binned_lumi_scratch_bytes(p, n) > ws_bytes) return PDF_EWORKSPACE;
    double *f1 = reinterpret_cast<double *>(align_up((size_t)ws + ws_x, 256));
    double *f2 = f1 + slice * kNF;
    ColMap cm; cm.n = kNF;
    for (int f = 0; f < kNF; ++f) cm.col[f] = f;
    CouplingParam C;
    for (int k = 0; k < kNF * kNF; ++k) C.c[k] = hostC[k];
    for (long long off = 0; off < n; off += slice) {
        const long long m = n - off < slice ? n - off : slice;
        int rc = binned_xfxq2<Scope>(G, p, cm, m, x1 + off, q2 + off, f1, kNF, ws, ws_x, chunk_opt, s, 0);
        if (rc) return rc;
        rc = binned_xfxq2<Scope>(G, p, cm, m, x2 + off, q2 + off, f2, kNF, ws, ws_x, chunk_opt, s, 0);
        if (rc) return rc;
        {
            Scope sc(s, "k_lumi_combine");
            k_lumi_combine<<<(unsigned)((m + 255) / 256), 256, 0, s>>>(C, m, f1, f2, x1 + off, x2 + off, w + off, out + off,
                                                                      G.err_count);
        }
    }
    return cudaGetLastError() == cudaSuccess ? PDF_OK : PDF_ECUDA;
}

}  // namespace pdfg
