// pdfgrid_host.inl -- host-buffer convenience calls (the e2e path of bench.py): inputs are copied
// to the device in chunks, evaluated by the same kernels as the device-pointer calls, and copied
// back; two pipeline slots on their own streams overlap H2D, compute and D2H of adjacent chunks.

namespace {

constexpr long long kHostChunk = 1LL << 22;   // queries per slot and chunk

int stage_reserve(pdf_grid *g, HostStage &st, size_t in_doubles, size_t out_doubles, size_t ws_bytes)
{
    if (!st.stream) CK(cudaStreamCreateWithFlags(&st.stream, cudaStreamNonBlocking));
    if (st.in_doubles < in_doubles) {
        cudaFree(st.in); st.in = nullptr; st.in_doubles = 0;
        int rc = dev_alloc(&st.in, in_doubles); if (rc) return rc;
        st.in_doubles = in_doubles;
    }
    if (st.out_doubles < out_doubles) {
        cudaFree(st.out); st.out = nullptr; st.out_doubles = 0;
        int rc = dev_alloc(&st.out, out_doubles); if (rc) return rc;
        st.out_doubles = out_doubles;
    }
    if (st.ws_bytes < ws_bytes) {
        cudaFree(st.ws); st.ws = nullptr; st.ws_bytes = 0;
        char *p = nullptr;
        int rc = dev_alloc(&p, ws_bytes); if (rc) return rc;
        st.ws = p; st.ws_bytes = ws_bytes;
    }
    (void)g;
    return PDF_OK;
}

// run `body(slot, off, m)` over [0,n) in chunks alternating between the two slots
template <typename F> int host_pipeline(pdf_grid *g, long long n, F body)
{
    int rc = PDF_OK;
    int c = 0;
    for (long long off = 0; off < n && rc == PDF_OK; off += kHostChunk, ++c) {
        long long m = n - off < kHostChunk ? n - off : kHostChunk;
        rc = body(g->stage[c & 1], off, m);
    }
    for (auto &st : g->stage) if (st.stream) {
        cudaError_t e = cudaStreamSynchronize(st.stream);
        if (e != cudaSuccess && rc == PDF_OK) rc = cuda_fail(e, "host pipeline");
    }
    return rc;
}

}  // namespace

extern "C" {

int pdf_xfxq2_host(pdf_grid *g, const int *pids, int npid, long long n, const double *x,
                   const double *q2, double *out)
{
    if (!g || n < 0 || npid < 1) return PDF_EINVAL;
    if (n == 0) return PDF_OK;
    if (!x || !q2 || !out) return PDF_EINVAL;
    long long cap = n < kHostChunk ? n : kHostChunk;
    size_t wsb = pdf_workspace_bytes(g, cap);
    for (auto &st : g->stage) {
        int rc = stage_reserve(g, st, 2 * (size_t)cap, (size_t)cap * npid, wsb);
        if (rc) return rc;
    }
    int rc = host_pipeline(g, n, [&](HostStage &st, long long off, long long m) -> int {
        CK(cudaMemcpyAsync(st.in, x + off, sizeof(double) * m, cudaMemcpyHostToDevice, st.stream));
        CK(cudaMemcpyAsync(st.in + cap, q2 + off, sizeof(double) * m, cudaMemcpyHostToDevice, st.stream));
        int r = xfxq2_impl(g, st.ws, st.ws_bytes, pids, npid, m, st.in, st.in + cap, nullptr, st.out, npid, st.stream);
        if (r) return r;
        CK(cudaMemcpyAsync(out + off * npid, st.out, sizeof(double) * m * npid, cudaMemcpyDeviceToHost, st.stream));
        return PDF_OK;
    });
    return rc;
}

int pdf_alphas_q2_host(pdf_grid *g, long long n, const double *q2, double *out)
{
    if (!g || n < 0) return PDF_EINVAL;
    if (g->d.na < 2) return PDF_ESTATE;
    if (n == 0) return PDF_OK;
    if (!q2 || !out) return PDF_EINVAL;
    long long cap = n < kHostChunk ? n : kHostChunk;
    for (auto &st : g->stage) {
        int rc = stage_reserve(g, st, (size_t)cap, (size_t)cap, 0);
        if (rc) return rc;
    }
    return host_pipeline(g, n, [&](HostStage &st, long long off, long long m) -> int {
        CK(cudaMemcpyAsync(st.in, q2 + off, sizeof(double) * m, cudaMemcpyHostToDevice, st.stream));
        int r = pdf_alphas_q2(g, m, st.in, st.out, st.stream);
        if (r) return r;
        CK(cudaMemcpyAsync(out + off, st.out, sizeof(double) * m, cudaMemcpyDeviceToHost, st.stream));
        return PDF_OK;
    });
}

int pdf_lumi_host(pdf_grid *g, long long n, const double *x1, const double *x2, const double *q2,
                  const double *weights, double *out)
{
    if (!g || n < 0) return PDF_EINVAL;
    if (!g->d.C) return PDF_ESTATE;
    if (n == 0) return PDF_OK;
    if (!x1 || !x2 || !q2 || !weights || !out) return PDF_EINVAL;
    long long cap = n < kHostChunk ? n : kHostChunk;
    size_t wsb = pdf_workspace_bytes(g, cap);
    for (auto &st : g->stage) {
        int rc = stage_reserve(g, st, 4 * (size_t)cap, (size_t)cap, wsb);
        if (rc) return rc;
    }
    int rc = host_pipeline(g, n, [&](HostStage &st, long long off, long long m) -> int {
        const double *src[4] = {x1, x2, q2, weights};
        for (int a = 0; a < 4; ++a)
            CK(cudaMemcpyAsync(st.in + a * cap, src[a] + off, sizeof(double) * m, cudaMemcpyHostToDevice, st.stream));
        int r = lumi_impl(g, st.ws, st.ws_bytes, m, st.in, st.in + cap, st.in + 2 * cap, st.in + 3 * cap, st.out, st.stream);
        if (r) return r;
        CK(cudaMemcpyAsync(out + off, st.out, sizeof(double) * m, cudaMemcpyDeviceToHost, st.stream));
        return PDF_OK;
    });
    return rc;
}

}  // extern "C"
