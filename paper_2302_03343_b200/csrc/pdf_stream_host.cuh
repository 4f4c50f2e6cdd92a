// pdf_stream_host.cuh -- host side of the binned path: key geometry, search tables, workspace, launch.
#pragma once
#include <cmath>
#include <cstdio>
#include <cstring>
#include <vector>

namespace pdfg {

constexpr long long kAutoMinN = 1 << 15;      // PDF_PATH_AUTO: below this the direct path is used
constexpr long long kMemberMinPer = 1 << 14;  // PDF_PATH_AUTO with member ids: queries per member below which the direct path is used

struct StreamPlan {
    bool usable = false;
    StreamDev dev{};
    unsigned short *d_lutx = nullptr, *d_lutq = nullptr;
    double *d_rowplus = nullptr;              // [nmem][nx][12] values at 1.01*Q2min (C-9's second anchor row)
    double *d_coup = nullptr;                 // [12][16] zero-padded coupling of the call in flight (pass 2 of pdf_lumi)
    double *d_plus = nullptr;                 // scratch of k_q2plus
    int ncells_q = 1;                         // Q2 cells (knots - sub-grids)
    bool locate_ok = false;                   // the search tables exist (pdf_locate can run this path's search)

    long long default_chunk = 256 * 1024;
};

// cell and t_q of 1.01*Q2min with the device log (C-9); res = {jg, t, in_range}
__global__ void k_q2plus(GridDev G, double *res)
{
    if (threadIdx.x || blockIdx.x) return;
    double q = G.q2plus;
    if (q > G.qk[G.nqtot - 1]) { res[2] = 0.0; return; }
    int j, jg;
    q_locate(G, q, j, jg);
    res[0] = (double)jg;
    res[1] = (q == G.qk[jg + 1]) ? 1.0 : (pdf_log(q) - G.cq[jg].lo_log) * G.cq[jg].inv_d;
    res[2] = 1.0;
}

// a-1 for C-9: the grid's values at Q2 = 1.01 Q2min for every member and x knot, RP[m][ix][f] =
// sum_b wq_b V[m][row_b][ix][f] with the 4 node weights of cell jgplus at tqplus (the Q2 direction of the
// second anchor of eq. 3.4 does not depend on the query, so it is tabulated once per grid)
__global__ void k_rowplus(GridDev G, int jgplus, double tqplus, double *__restrict__ rp)
{
    const size_t per = (size_t)G.nx * G.nfp;
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= per * G.nmem) return;
    const int m = (int)(e / per);
    const size_t r = e % per;
    Point1D qp;
    q_point_cell(G, jgplus, tqplus, qp);
    const double *Vm = G.V + (size_t)m * G.memstride;
    double acc = 0.0;
#pragma unroll
    for (int b = 0; b < 4; ++b) acc = fma(qp.w[b], Vm[(size_t)qp.idx[b] * per + r], acc);
    rp[e] = acc;
}

inline void stream_plan_free(StreamPlan &p)
{
    cudaFree(p.d_lutx); cudaFree(p.d_lutq); cudaFree(p.d_rowplus); cudaFree(p.d_plus); cudaFree(p.d_coup); p.d_coup = nullptr;
    p.d_lutx = p.d_lutq = nullptr; p.d_rowplus = nullptr; p.d_plus = nullptr; p.usable = false; p.locate_ok = false;
}

// search table of one knot line: bucket = (high word of v >> shift) - base; entry = the largest c <= lim with
// k[c] <= the bucket's lower edge (0 if none).  The widest bucket that keeps the table within kS3LutMax entries.
inline void make_search_table(const std::vector<double> &k, int lim, int &shift, int &base, std::vector<unsigned short> &lut)
{
    auto hi = [](double v) { long long b; std::memcpy(&b, &v, 8); return (int)(b >> 32); };
    const int h0 = hi(k.front()), h1 = hi(k.back());
    shift = 12;                                         // 8 mantissa bits: 256 buckets per binade
    while (shift < 31 && ((h1 >> shift) - (h0 >> shift) + 1) > kS3LutMax) ++shift;
    base = h0 >> shift;
    const int nb = (h1 >> shift) - base + 1;
    lut.resize(nb);
    int c = 0;
    for (int b = 0; b < nb; ++b) {
        const long long eb = ((long long)(base + b) << shift) << 32;
        double edge;
        std::memcpy(&edge, &eb, 8);
        while (c < lim && k[c + 1] <= edge) ++c;
        lut[b] = (unsigned short)c;
    }
}

inline long long stream_chunk(const StreamPlan &p, long long n, long long chunk_opt)
{
    long long c = chunk_opt > 0 ? chunk_opt : p.default_chunk;
    c = (c + kS3TileA - 1) / kS3TileA * kS3TileA;
    long long need = (n + kS3TileA - 1) / kS3TileA * kS3TileA;
    if (need < kS3TileA) need = kS3TileA;
    return c < need ? c : need;
}

// per-chunk geometry: a cell bin holds 3x the uniform share + 32 (a uniform cloud is Poisson around the share;
// beyond it queries overflow to a list), one E unit per 1024 queries of the chunk
inline void stream_caps(const StreamPlan &p, long long chunk, StreamDev &d, int mode = kModeRows)
{
    d = p.dev;
    d.fku = mode == kModeLumiSecond ? kS3FkPerUnitLumi2 : kS3FkPerUnit;
    d.ng = (d.nqt + d.fku - 1) / d.fku;
    const long long per_cell = chunk / ((long long)(d.ncx > 0 ? d.ncx : 1) * (p.ncells_q > 0 ? p.ncells_q : 1));
    long long cap = (3 * per_cell + 32 + 31) / 32 * 32;
    if (cap > chunk) cap = (chunk + 31) / 32 * 32;
    d.cap = (int)cap;
    d.ne = (int)((chunk + PDF_S3_EDIV - 1) / PDF_S3_EDIV);
    d.tb = d.ne + d.ncx * d.ng;
}

inline size_t stream_workspace_bytes(const StreamPlan &p, long long n, long long chunk_opt)
{
    if (!p.usable) return 0;
    const long long chunk = stream_chunk(p, n, chunk_opt);
    StreamDev d;
    stream_caps(p, chunk, d);
    size_t b = sizeof(unsigned long long) * kCtrlWords;
    b += align_up(sizeof(unsigned) * (size_t)kS3Ring * (d.nbins + 32), 256);
    b += align_up(sizeof(Payload) * (size_t)kS3Ring * d.nbins * d.cap, 256);
    b += align_up(sizeof(Payload) * (size_t)kS3Ring * kNumLists * chunk, 256);
    return b + 256;
}

inline void stream_carve(void *ws, long long chunk, const StreamDev &d, StreamWorkspace &w)
{
    char *c = (char *)align_up((size_t)ws, 256);
    w.ctrl = (unsigned long long *)c; c += sizeof(unsigned long long) * kCtrlWords;
    w.counts = (unsigned *)c; c += align_up(sizeof(unsigned) * (size_t)kS3Ring * (d.nbins + 32), 256);
    w.bins = (Payload *)c; c += align_up(sizeof(Payload) * (size_t)kS3Ring * d.nbins * d.cap, 256);
    w.lists = (Payload *)c;
    (void)chunk;
}

inline size_t stream_smem_bytes(const GridDev &G, const StreamDev &d)
{
    return s3_table_bytes(G.nx, G.nqtot, d.nbx, d.nbq) + 32 + (size_t)kS3Warps * kStageBytes + kCoupBytes;
}

// builds the search tables and the key geometry; leaves usable = false when the grid does not fit the
// specialised path (then every call takes the direct path; pdf_last_path reports which one ran)
inline int stream_plan_init(StreamPlan &p, const GridDev &G, const std::vector<double> &xk, const std::vector<double> &qk, int nsub)
{
    p.usable = false;
    const int nx = G.nx, nqt = G.nqtot;
    if (G.nflav != kNF || G.nfp != kNFP) return 0;
    if (nx - 1 > kS3MaxCells || nqt > kS3MaxCells || nx < 2) return 0;
    StreamDev &d = p.dev;
    d.ncx = nx - 1; d.nqt = nqt;
    d.nbins = d.ncx * nqt;
    d.fku = kS3FkPerUnit; d.ng = (nqt + d.fku - 1) / d.fku;
    p.ncells_q = nqt - nsub;

    std::vector<unsigned short> lx, lq;
    make_search_table(xk, nx - 2, d.xshift, d.xbase, lx);
    make_search_table(qk, nqt - 1, d.qshift, d.qbase, lq);
    d.nbx = (int)lx.size(); d.nbq = (int)lq.size();

    if (cudaMalloc((void **)&p.d_lutx, sizeof(unsigned short) * lx.size()) != cudaSuccess) return PDF_ENOMEM;
    if (cudaMalloc((void **)&p.d_lutq, sizeof(unsigned short) * lq.size()) != cudaSuccess) return PDF_ENOMEM;
    if (cudaMalloc((void **)&p.d_plus, sizeof(double) * 4) != cudaSuccess) return PDF_ENOMEM;
    cudaMemcpy(p.d_lutx, lx.data(), sizeof(unsigned short) * lx.size(), cudaMemcpyHostToDevice);
    cudaMemcpy(p.d_lutq, lq.data(), sizeof(unsigned short) * lq.size(), cudaMemcpyHostToDevice);
    k_q2plus<<<1, 32>>>(G, p.d_plus);
    double res[3] = {0, 0, 0};
    if (cudaMemcpy(res, p.d_plus, sizeof res, cudaMemcpyDeviceToHost) != cudaSuccess) return PDF_ECUDA;
    d.lutx = p.d_lutx; d.lutq = p.d_lutq;
    // pdf_locate on this path needs only the tables
    if (cudaFuncSetAttribute(k_locate_stream, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)s3_table_bytes(nx, nqt, d.nbx, d.nbq)) != cudaSuccess) return 0;
    p.locate_ok = true;
    if (res[2] != 1.0) return 0;                           // 1.01*Q2min beyond the grid: direct path only
    d.jgplus = (int)res[0]; d.tqplus = res[1];
    const size_t nrp = (size_t)G.nmem * nx * kNFP;
    if (cudaMalloc((void **)&p.d_rowplus, sizeof(double) * nrp) != cudaSuccess) return PDF_ENOMEM;
    k_rowplus<<<(unsigned)((nrp + 255) / 256), 256>>>(G, d.jgplus, d.tqplus, p.d_rowplus);
    if (cudaDeviceSynchronize() != cudaSuccess) return PDF_ECUDA;
    d.rowplus = p.d_rowplus;
    const size_t smem = stream_smem_bytes(G, d);
    if (smem > 200 * 1024) return 0;
    if (cudaFuncSetAttribute(k_pdf_stream, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return 0;
    if (cudaFuncSetAttribute(k_pdf_stream_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return 0;
    if (cudaFuncSetAttribute(k_lumi_first, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return 0;
    if (cudaFuncSetAttribute(k_lumi_second, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return 0;
    if (cudaFuncSetAttribute(k_pdf_stream_opt, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return 0;
    if (cudaFuncSetAttribute(k_lumi_first_opt, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return 0;
    if (cudaFuncSetAttribute(k_lumi_second_opt, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return 0;
    if (cudaMalloc((void **)&p.d_coup, kCoupBytes) != cudaSuccess) return PDF_ENOMEM;
    p.usable = true;
    return 0;
}

inline bool stream_qualifies(const StreamPlan &p, const int *member) { return p.usable && !member; }
inline bool stream_members_qualifies(const StreamPlan &p, const GridDev &G, const int *member)
{
    return p.usable && member && G.nmem > 1 && G.nmem <= kMemMax;
}

// one memset + one persistent kernel for the whole call
template <typename Scope>
inline int stream_xfxq2(const GridDev &G, const StreamPlan &p, const ColMap &cm, long long n, const double *x,
                        const double *q2, double *out, long long ld, void *ws, size_t ws_bytes, long long chunk_opt,
                        cudaStream_t s, int count_err = 1, const int *ctab = nullptr, const int *nchunks_dev = nullptr,
                        int mode = kModeRows, const double *x2 = nullptr, const double *w = nullptr, const double *f1 = nullptr,
                        const unsigned *orig = nullptr, int q_is_q = 0)
{
    if (stream_workspace_bytes(p, n, chunk_opt) > ws_bytes) return PDF_EWORKSPACE;
    StreamArgs A;
    A.ctab = ctab; A.nchunks_dev = nchunks_dev;
    A.x2 = x2; A.w = w; A.f1 = f1; A.coup = p.d_coup; A.orig = orig;
    A.G = G; A.cm = cm;
    A.chunk = stream_chunk(p, n, chunk_opt);
    stream_caps(p, A.chunk, A.B, mode);
    stream_carve(ws, A.chunk, A.B, A.W);
    A.x = x; A.q2 = q2; A.out = out; A.n = n; A.ld = ld;
    A.nchunks = (int)((n + A.chunk - 1) / A.chunk);
    A.ta = (int)(A.chunk / kS3TileA);
    A.identity = cm.n == kNF;
    for (int f = 0; f < kNF && A.identity; ++f) A.identity = cm.col[f] == f;
    A.count_err = count_err;
    A.q_is_q = q_is_q;
    const size_t zero_bytes = (size_t)((char *)A.W.bins - (char *)A.W.ctrl);      // ctrl + counts
    if (cudaMemsetAsync(A.W.ctrl, 0, zero_bytes, s) != cudaSuccess) return PDF_ECUDA;
    const size_t smem = stream_smem_bytes(G, A.B);
    int per_sm = 0, dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const bool rows11 = A.identity && ld < (1LL << 29);              // the four fixed stores of b_unit (32-bit row stride in bytes)
    const bool opt = q_is_q || G.extrap != kExtrapContinuation;      // pdf_xfxq / an extrapolation option of L1720: kernels of their own
    const auto kern = opt ? (mode == kModeLumiFirst ? k_lumi_first_opt : mode == kModeLumiSecond ? k_lumi_second_opt : k_pdf_stream_opt)
                          : (mode == kModeLumiFirst ? k_lumi_first : mode == kModeLumiSecond ? k_lumi_second : rows11 ? k_pdf_stream : k_pdf_stream_cols);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kS3Threads, smem) != cudaSuccess || per_sm < 1)
        return PDF_ECUDA;
    const unsigned long long max_ctas = (unsigned long long)per_sm * sms;         // all CTAs must be co-resident
    // with a chunk table the chunk count is on the device: the launch takes its upper bound
    const long long nch = ctab ? member_max_chunks(n, A.chunk, G.nmem) : (long long)A.nchunks;
    const unsigned long long tickets = (unsigned long long)nch * (A.ta + A.B.tb);
    const unsigned long long want = (tickets + kS3Warps - 1) / kS3Warps;
    const unsigned grid = (unsigned)(want < max_ctas ? want : max_ctas);
    {
        Scope sc(s, opt ? (mode == kModeLumiFirst ? "k_lumi_first_opt" : mode == kModeLumiSecond ? "k_lumi_second_opt" : "k_pdf_stream_opt")
                        : (mode == kModeLumiFirst ? "k_lumi_first" : mode == kModeLumiSecond ? "k_lumi_second" : rows11 ? "k_pdf_stream" : "k_pdf_stream_cols"));
        kern<<<grid, kS3Threads, smem, s>>>(A);
    }
    return cudaGetLastError() == cudaSuccess ? PDF_OK : PDF_ECUDA;
}

template <typename Scope>
inline int stream_locate(const GridDev &G, const StreamPlan &p, long long n, const double *x, const double *q2,
                         int *ix, int *iq, int *isub, int *region, cudaStream_t s)
{
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long long want = (n + 255) / 256;
    const unsigned grid = (unsigned)(want < (long long)sms * 8 ? want : (long long)sms * 8);
    Scope sc(s, "k_locate_stream");
    k_locate_stream<<<grid, 256, s3_table_bytes(G.nx, G.nqtot, p.dev.nbx, p.dev.nbq), s>>>(G, p.dev, n, x, q2, ix, iq, isub, region);
    return cudaGetLastError() == cudaSuccess ? PDF_OK : PDF_ECUDA;
}

// ---- luminosity on top of the binned path (a-7) ------------------------------------------------
// pdf_lumi in slices of kLumiSlice events, two runs of the persistent kernel per slice:
//   k_lumi_first   bins the events by the cell of (x1, Q2) and writes rows [xf_0..xf_10(x1, Q2), w/(x1 x2)] of 12
//                  doubles -- whole 32-byte sectors, so no zero fill -- into the slice's scratch;
//   k_lumi_second  bins them by the cell of (x2, Q2); its epilogue reads the event's row of pass 1 straight into DMMA
//                  A-operand fragments, forms G = f1 C by 6 more DMMAs, dots it with its own accumulator fragments and
//                  writes the 8-byte result.  The 88 B / event of xf(x2) never leave the registers and there is no
//                  separate reduction kernel.
constexpr long long kLumiSlice = 1LL << 24;

inline bool stream_lumi_qualifies(const StreamPlan &p) { return p.usable; }
inline size_t stream_lumi_scratch_bytes(const StreamPlan &p, long long n)
{
    const long long slice = n < kLumiSlice ? n : kLumiSlice;
    return p.usable ? (size_t)slice * kNFP * sizeof(double) + 512 : 0;
}

template <typename Scope>
inline int stream_lumi(const GridDev &G, const StreamPlan &p, const double *hostC, long long n, const double *x1,
                       const double *x2, const double *q2, const double *w, double *out, void *ws, size_t ws_bytes,
                       long long chunk_opt, cudaStream_t s)
{
    const long long slice = n < kLumiSlice ? n : kLumiSlice;
    const size_t ws_x = stream_workspace_bytes(p, slice, chunk_opt);
    if (ws_x + stream_lumi_scratch_bytes(p, n) > ws_bytes) return PDF_EWORKSPACE;
    double *f1 = reinterpret_cast<double *>(align_up((size_t)ws + ws_x, 256));
    ColMap cm12; cm12.n = kNF;
    for (int f = 0; f < kNF; ++f) cm12.col[f] = f;
    ColMap cm1; cm1.n = 1; cm1.col[0] = 0;
    double Cp[kNFP * 16];
    for (int k = 0; k < kNFP * 16; ++k) Cp[k] = 0.0;
    for (int i = 0; i < kNF; ++i)
        for (int j = 0; j < kNF; ++j) Cp[i * 16 + j] = hostC[i * kNF + j];
    if (cudaMemcpyAsync(p.d_coup, Cp, sizeof Cp, cudaMemcpyHostToDevice, s) != cudaSuccess) return PDF_ECUDA;   // pageable source: staged before return
    for (long long off = 0; off < n; off += slice) {
        const long long m = n - off < slice ? n - off : slice;
        int rc = stream_xfxq2<Scope>(G, p, cm12, m, x1 + off, q2 + off, f1, kNFP, ws, ws_x, chunk_opt, s, 0, nullptr, nullptr,
                                     kModeLumiFirst, x2 + off, w + off, nullptr);
        if (rc) return rc;
        rc = stream_xfxq2<Scope>(G, p, cm1, m, x2 + off, q2 + off, out + off, 1, ws, ws_x, chunk_opt, s, 1, nullptr, nullptr,
                                 kModeLumiSecond, nullptr, nullptr, f1);
        if (rc) return rc;
    }
    return cudaGetLastError() == cudaSuccess ? PDF_OK : PDF_ECUDA;
}

// a-8 on the binned path (pdf_members.cuh): per slice, partition by member, then one persistent-kernel
// run over the chunk table whose rows go straight to their queries' places
inline size_t stream_members_bytes(const StreamPlan &p, const GridDev &G, long long n, long long chunk_opt, int npid)
{
    if (!p.usable || G.nmem < 2 || G.nmem > kMemMax) return 0;
    const long long slice = member_slice(n);
    const long long chunk = stream_chunk(p, slice, chunk_opt);
    return stream_workspace_bytes(p, slice, chunk_opt) + member_scratch_bytes(slice, chunk, G.nmem, npid) + 256;
}

template <typename Scope>
inline int stream_members(const GridDev &G, const StreamPlan &p, const ColMap &cm, long long n, const double *x,
                          const double *q2, const int *member, double *out, long long ld, void *ws, size_t ws_bytes,
                          long long chunk_opt, cudaStream_t s)
{
    if (stream_members_bytes(p, G, n, chunk_opt, cm.n) > ws_bytes) return PDF_EWORKSPACE;
    const long long slice = member_slice(n);
    const long long chunk = stream_chunk(p, slice, chunk_opt);
    const size_t ws_x = stream_workspace_bytes(p, slice, chunk_opt);
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
                x + off, q2 + off, member + off, m, G.nmem, M.cursor, M.xs, M.q2s, M.orig, out + off * ld, ld, cm.n, G.err_count);
        }
        int rc = stream_xfxq2<Scope>(G, p, cm, m, M.xs, M.q2s, out + off * ld, ld, ws, ws_x, chunk_opt, s, 1, M.ctab, M.nchunks,
                                     kModeRows, nullptr, nullptr, nullptr, M.orig);
        if (rc) return rc;
    }
    return cudaGetLastError() == cudaSuccess ? PDF_OK : PDF_ECUDA;
}

}  // namespace pdfg
