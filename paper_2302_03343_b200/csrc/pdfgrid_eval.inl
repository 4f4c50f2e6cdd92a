// pdfgrid_eval.inl -- evaluation entry points of the C ABI (included at the end of pdfgrid.cu).

namespace {

int build_colmap(const pdf_grid *g, const int *pids, int npid, ColMap &cm)
{
    if (!pids || npid < 1 || npid > 64) return PDF_EINVAL;
    cm.n = npid;
    for (int p = 0; p < npid; ++p) cm.col[p] = col_of_pid(g, pids[p]);
    return PDF_OK;
}

inline unsigned blocks_for(long long n, int threads) { return (unsigned)((n + threads - 1) / threads); }

// direct path in slices of < 2^31 blocks (n is long long)
int launch_direct(const pdf_grid *g, const ColMap &cm, long long n, const double *x, const double *q2,
                  const int *member, double *out, long long ld, cudaStream_t s, int q_is_q = 0)
{
    const long long slice = 1LL << 30;
    for (long long off = 0; off < n; off += slice) {
        long long m = n - off < slice ? n - off : slice;
        LaunchScope a(s, "k_xfxq2_direct");
        k_xfxq2_direct<<<blocks_for(m, 128), 128, 0, s>>>(g->d, cm, m, x + off, q2 + off,
                                                         member ? member + off : nullptr, out + off * ld, ld, q_is_q);
    }
    CK(cudaGetLastError());
    return PDF_OK;
}

int on_device(const pdf_grid *g);

// pdf_xfxq2_ex with the workspace as an argument (the *_host calls pass their own staging workspace)
int xfxq2_impl(const pdf_grid *g, void *ws, size_t ws_bytes, const int *pids, int npid, long long n, const double *x,
               const double *q2, const int *member, double *out, long long ld_out, cudaStream_t s, int q_is_q = 0)
{
    if (!g || n < 0 || ld_out < npid) return PDF_EINVAL;
    if (q_is_q && member) return PDF_EINVAL;
    ColMap cm;
    int rc = build_colmap(g, pids, npid, cm);
    if (rc) return rc;
    if (n == 0) return PDF_OK;
    if (!x || !q2 || !out) return PDF_EINVAL;
    if ((rc = on_device(g))) return rc;
    // a-8: per-query member ids on the binned path (partition by member first, pdf_members.cuh)
    if (stream_members_qualifies(g->bplan, g->d, member) && npid <= g->d.nflav) {
        const size_t need = stream_members_bytes(g->bplan, g->d, n, g->chunk, npid);
        if (g->path == PDF_PATH_BINNED) {
            if (!ws || ws_bytes < need) return PDF_EWORKSPACE;
            g->last_path = PDF_PATH_BINNED;
            return stream_members<LaunchScope>(g->d, g->bplan, cm, n, x, q2, member, out, ld_out, ws, ws_bytes, g->chunk, s);
        }
        if (g->path == PDF_PATH_AUTO && ws && ws_bytes >= need && n >= kMemberMinPer * g->d.nmem) {
            g->last_path = PDF_PATH_BINNED;
            return stream_members<LaunchScope>(g->d, g->bplan, cm, n, x, q2, member, out, ld_out, ws, ws_bytes, g->chunk, s);
        }
    }
    bool ok_binned = stream_qualifies(g->bplan, member);
    const size_t need = stream_workspace_bytes(g->bplan, n, g->chunk);      // what THIS call uses of the workspace
    bool want_binned = (g->path == PDF_PATH_BINNED) ||
                       (g->path == PDF_PATH_AUTO && ws && ok_binned && n >= kAutoMinN && ws_bytes >= need);
    if (want_binned) {
        if (!ok_binned) return PDF_EINVAL;
        if (!ws || ws_bytes < need) return PDF_EWORKSPACE;
        g->last_path = PDF_PATH_BINNED;
        return stream_xfxq2<LaunchScope>(g->d, g->bplan, cm, n, x, q2, out, ld_out, ws, ws_bytes, g->chunk, s, 1, nullptr, nullptr,
                                         kModeRows, nullptr, nullptr, nullptr, nullptr, q_is_q);
    }
    g->last_path = PDF_PATH_DIRECT;
    return launch_direct(g, cm, n, x, q2, member, out, ld_out, s, q_is_q);
}

int lumi_impl(const pdf_grid *g, void *ws, size_t ws_bytes, long long n, const double *x1, const double *x2, const double *q2,
              const double *weights, double *out, cudaStream_t s)
{
    if (!g || n < 0) return PDF_EINVAL;
    if (!g->d.C) return PDF_ESTATE;
    if (g->d.nflav > kMaxLumiFlav) return PDF_EINVAL;
    if (n == 0) return PDF_OK;
    if (!x1 || !x2 || !q2 || !weights || !out) return PDF_EINVAL;
    int rc = on_device(g);
    if (rc) return rc;
    const size_t need = stream_workspace_bytes(g->bplan, n < kLumiSlice ? n : kLumiSlice, g->chunk) +
                        stream_lumi_scratch_bytes(g->bplan, n) + 256;
    bool want_binned = stream_lumi_qualifies(g->bplan) &&
                       (g->path == PDF_PATH_BINNED || (g->path == PDF_PATH_AUTO && ws && n >= kAutoMinN &&
                                                       ws_bytes >= need));
    if (want_binned) {
        g->last_path = PDF_PATH_BINNED;
        return stream_lumi<LaunchScope>(g->d, g->bplan, g->h_C.data(), n, x1, x2, q2, weights, out, ws, ws_bytes, g->chunk, s);
    }
    g->last_path = PDF_PATH_DIRECT;
    const long long slice = 1LL << 30;
    for (long long off = 0; off < n; off += slice) {
        long long m = n - off < slice ? n - off : slice;
        LaunchScope a(s, "k_lumi_direct");
        k_lumi_direct<<<blocks_for(m, 128), 128, 0, s>>>(g->d, m, x1 + off, x2 + off, q2 + off, weights + off, out + off);
    }
    CK(cudaGetLastError());
    return PDF_OK;
}

// every evaluation call runs on the device the grid lives on
int on_device(const pdf_grid *g)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return PDF_ECUDA;
    if (dev != g->device && cudaSetDevice(g->device) != cudaSuccess) return PDF_ECUDA;
    return PDF_OK;
}

}  // namespace

extern "C" {

int pdf_xfxq2_ex(const pdf_grid *g, const int *pids, int npid, long long n, const double *x,
                 const double *q2, const int *member, double *out, long long ld_out, void *stream)
{
    if (!g) return PDF_EINVAL;
    return xfxq2_impl(g, g->ws, g->ws_bytes, pids, npid, n, x, q2, member, out, ld_out, (cudaStream_t)stream);
}

int pdf_xfxq2(const pdf_grid *g, const int *pids, int npid, long long n, const double *x,
              const double *q2, double *out, void *stream)
{
    return pdf_xfxq2_ex(g, pids, npid, n, x, q2, nullptr, out, npid, stream);
}

int pdf_xfxq(const pdf_grid *g, const int *pids, int npid, long long n, const double *x,
             const double *q, double *out, void *stream)
{
    if (!g) return PDF_EINVAL;
    return xfxq2_impl(g, g->ws, g->ws_bytes, pids, npid, n, x, q, nullptr, out, npid, (cudaStream_t)stream, 1);
}

int pdf_xfxq2_xgrid(const pdf_grid *g, const int *pids, int npid, long long npts, const double *x, const double *q2,
                    int nrep, const int *members, double *out, long long ld_out, void *stream)
{
    if (!g || npts < 0 || nrep < 0 || ld_out < npid) return PDF_EINVAL;
    ColMap cm;
    int rc = build_colmap(g, pids, npid, cm);
    if (rc) return rc;
    if (npts == 0 || nrep == 0) return PDF_OK;
    if (!x || !q2 || !out) return PDF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, g->device);
    const long long bx = (npts + kXgridThreads - 1) / kXgridThreads;
    if (bx > 0x7fffffffLL) return PDF_EINVAL;
    // member slices: one wave of co-resident CTAs (4 per SM at 128 registers), at most one slice per member
    long long by = ((long long)sms * 4) / bx;
    if (by > nrep) by = nrep;
    if (by > 65535) by = 65535;
    if (by < 1) by = 1;
    // the row-wise path: 11 value columns in rows of 12 doubles; the coalesced store also needs contiguous
    // rows and the identity column map
    const int fast11 = g->d.nflav == 11 && g->d.nfp == 12;
    bool ident = fast11 && ld_out == 11 && cm.n == 11;
    for (int k = 0; ident && k < 11; ++k) ident = cm.col[k] == k;
    if (ident && g->path != PDF_PATH_DIRECT) {   // the (member, cell)-shared form (contiguous 11-flavour rows); PDF_PATH_DIRECT keeps the per-point kernel
        const long long tiles = (npts + kXcT - 1) / kXcT, groups = ((long long)nrep + kXcMem - 1) / kXcMem;
        // worth it once (tile, member group) pairs fill the machine; measured on the Table 3.3 shape:
        // N_rep = 50: 0.037 against 0.026 ms per-point, 100: 0.040 / 0.038, 200: 0.041 / 0.054, 400: 0.066 / 0.091
        if (tiles <= 0x7fffffffLL && tiles * groups >= 2LL * sms) {
            // one wave of co-resident CTAs (4 per SM); a CTA walks the member groups in strides of the grid's
            // rows (one (tile, group) pair per CTA in several waves measured slower: 0.077 against 0.074 ms (then) at
            // N_rep = 400, every wave pays the tile's plan phase again)
            long long gy = ((long long)sms * 4) / tiles;
            if (gy > groups) gy = groups;
            if (gy > 65535) gy = 65535;
            if (gy < 1) gy = 1;
            LaunchScope a(s, "k_xfxq2_xgrid_cell");
            k_xfxq2_xgrid_cell<<<dim3((unsigned)tiles, (unsigned)gy), kXcThreads, 0, s>>>(g->d, npts, x, q2, nrep, members, out);
            CK(cudaGetLastError());
            return PDF_OK;
        }
    }
    LaunchScope a(s, "k_xfxq2_xgrid");
    k_xfxq2_xgrid<<<dim3((unsigned)bx, (unsigned)by), kXgridThreads, 0, s>>>(g->d, cm, npts, x, q2, nrep, members, out,
                                                                              ld_out, fast11, ident ? 1 : 0);
    CK(cudaGetLastError());
    return PDF_OK;
}

size_t pdf_workspace_bytes(const pdf_grid *g, long long n)
{
    if (!g || n < 0) return 0;
    size_t b = stream_workspace_bytes(g->bplan, n, g->chunk);
    if (b && g->d.C) b += stream_lumi_scratch_bytes(g->bplan, n) + 256;    // pdf_lumi slices (only once a coupling is set)
    if (g->d.nmem > 1) {                                                // a-8: member partition scratch (all flavours)
        size_t m = stream_members_bytes(g->bplan, g->d, n, g->chunk, g->d.nflav);
        if (m > b) b = m;
    }
    return b;
}

int pdf_alphas_q2(const pdf_grid *g, long long n, const double *q2, double *out, void *stream)
{
    if (!g || n < 0) return PDF_EINVAL;
    if (g->d.na < 2) return PDF_ESTATE;
    if (n == 0) return PDF_OK;
    if (!q2 || !out) return PDF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, g->device);
    long long want = (n + 255) / 256;
    unsigned grid = (unsigned)(want < (long long)sms * 8 ? want : (long long)sms * 8);
    LaunchScope a(s, "k_alphas");
    size_t smem = sizeof(double) * (2 * g->d.na + 6 * (g->d.na - 1)) + sizeof(short) * g->d.nalut + 16;
    if (smem > 48 * 1024) return PDF_EINVAL;
    k_alphas<<<grid, 256, smem, s>>>(g->d, n, q2, out);
    CK(cudaGetLastError());
    return PDF_OK;
}

int pdf_lumi(const pdf_grid *g, long long n, const double *x1, const double *x2, const double *q2,
             const double *weights, double *out, void *stream)
{
    if (!g) return PDF_EINVAL;
    return lumi_impl(g, g->ws, g->ws_bytes, n, x1, x2, q2, weights, out, (cudaStream_t)stream);
}

int pdf_locate(const pdf_grid *g, long long n, const double *x, const double *q2, int *ix,
               int *iq, int *isub, int *region, void *stream)
{
    if (!g || n < 0) return PDF_EINVAL;
    if (n == 0) return PDF_OK;
    if (!x || !q2) return PDF_EINVAL;
    int rc = on_device(g);
    if (rc) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    // the search of the path the evaluation calls take: the table-driven search of the binned kernel's A
    // tiles unless PDF_PATH_DIRECT is set (or the grid does not fit the binned path), then the binary
    // search of the direct kernels
    if (g->path != PDF_PATH_DIRECT && g->bplan.locate_ok) {
        g->last_path = PDF_PATH_BINNED;
        return stream_locate<LaunchScope>(g->d, g->bplan, n, x, q2, ix, iq, isub, region, s);
    }
    g->last_path = PDF_PATH_DIRECT;
    const long long slice = 1LL << 30;
    for (long long off = 0; off < n; off += slice) {
        long long m = n - off < slice ? n - off : slice;
        LaunchScope a(s, "k_locate");
        k_locate<<<blocks_for(m, 256), 256, 0, s>>>(g->d, m, x + off, q2 + off, ix ? ix + off : nullptr,
                                                   iq ? iq + off : nullptr, isub ? isub + off : nullptr,
                                                   region ? region + off : nullptr);
    }
    CK(cudaGetLastError());
    return PDF_OK;
}

int pdf_last_path(const pdf_grid *g)
{
    return g ? g->last_path : PDF_EINVAL;
}

int pdf_error_count(const pdf_grid *g, long long *n_invalid, void *stream)
{
    if (!g || !n_invalid) return PDF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    unsigned long long v = 0;
    CK(cudaMemcpyAsync(&v, g->d_err, sizeof v, cudaMemcpyDeviceToHost, s));
    CK(cudaMemsetAsync(g->d_err, 0, sizeof v, s));
    CK(cudaStreamSynchronize(s));
    *n_invalid = (long long)v;
    return PDF_OK;
}

int pdf_log_f64(long long n, const double *x, double *out, void *stream)
{
    if (n < 0) return PDF_EINVAL;
    if (n == 0) return PDF_OK;
    if (!x || !out) return PDF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    LaunchScope a(s, "k_log_f64");
    k_log_f64<<<blocks_for(n, 256), 256, 0, s>>>(n, x, out);
    CK(cudaGetLastError());
    return PDF_OK;
}

int pdf_measure_fp64_tflops(double *tflops, void *stream)
{
    if (!tflops) return PDF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    double *sink = nullptr;
    int rc = dev_alloc(&sink, 1);
    if (rc) return rc;
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    const int iters = 1 << 15, blocks = sms * 8, threads = 256;
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(a, s);
        { LaunchScope l(s, "k_dfma_chain"); k_dfma_chain<<<blocks, threads, 0, s>>>(sink, iters, 0.999999, 1e-9); }
        cudaEventRecord(b, s);
        cudaEventSynchronize(b);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, a, b);
        if (rep && ms < best) best = ms;
    }
    cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(sink);
    CK(cudaGetLastError());
    double flops = 2.0 * 8.0 * (double)iters * (double)blocks * threads;
    *tflops = flops / (best * 1e-3) / 1e12;
    return PDF_OK;
}

}  // extern "C"

#include "pdfgrid_host.inl"
