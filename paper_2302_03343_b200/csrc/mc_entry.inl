// mc_entry.inl -- C-ABI entry points of the Monte Carlo steps around the hot path (included at the end of pdfgrid.cu)

extern "C" {

int pdf_rambo(long long nev, int npart, const double *sqrt_s, const double *masses, const double *u, double ptmin,
              double *p, double *w, void *stream)
{
    if (nev < 0 || npart < 2 || npart > kRamboMaxN) return PDF_EINVAL;
    if (nev == 0) return PDF_OK;
    if (!sqrt_s || !u || !p || !w) return PDF_EINVAL;
    RamboMasses M{};
    if (masses)
        for (int i = 0; i < npart; ++i) {
            if (!(masses[i] >= 0.0) || !std::isfinite(masses[i])) return PDF_EINVAL;
            M.m[i] = masses[i];
            if (masses[i] > 0.0) M.massive = 1;
        }
    cudaStream_t s = (cudaStream_t)stream;
    LaunchScope a(s, "k_rambo");
    k_rambo<<<blocks_for(nev, 128), 128, 0, s>>>(nev, npart, sqrt_s, M, u, ptmin, p, w);
    CK(cudaGetLastError());
    return PDF_OK;
}

int pdf_vegas_map(int ndim, int nbins, const double *edges, long long n, const double *u, double *x, double *jac,
                  int *bin, void *stream)
{
    if (ndim < 1 || nbins < 1 || n < 0 || (size_t)ndim * (nbins + 1) * sizeof(double) > 48 * 1024) return PDF_EINVAL;
    if (n == 0) return PDF_OK;
    if (!edges || !u || !x || !jac) return PDF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    int sms = 148, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long long want = (n + 255) / 256;
    LaunchScope a(s, "k_vegas_map");
    k_vegas_map<<<(unsigned)(want < (long long)sms * 8 ? want : (long long)sms * 8), 256, sizeof(double) * ndim * (nbins + 1), s>>>(
        ndim, nbins, edges, n, u, x, jac, bin);
    CK(cudaGetLastError());
    return PDF_OK;
}

int pdf_vegas_accumulate(int ndim, int nbins, long long n, const double *f, const double *jac, const int *bin,
                         double *sums, double *hist, void *stream)
{
    if (ndim < 1 || nbins < 1 || n < 0 || ((size_t)ndim * nbins + 16) * sizeof(double) > 48 * 1024) return PDF_EINVAL;
    if (!sums || (hist && !bin)) return PDF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    CK(cudaMemsetAsync(sums, 0, 2 * sizeof(double), s));
    if (hist) CK(cudaMemsetAsync(hist, 0, sizeof(double) * ndim * nbins, s));
    if (n == 0) return PDF_OK;
    if (!f || !jac) return PDF_EINVAL;
    int sms = 148, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long long want = (n + 255) / 256;
    LaunchScope a(s, "k_vegas_accumulate");
    k_vegas_accumulate<<<(unsigned)(want < (long long)sms * 4 ? want : (long long)sms * 4), 256,
                         sizeof(double) * ((size_t)ndim * nbins + 16), s>>>(ndim, nbins, n, f, jac, bin, sums, hist);
    CK(cudaGetLastError());
    return PDF_OK;
}

int pdf_vegas_estimate(long long n, const double *sums, double *res, void *stream)
{
    if (n < 2 || !sums || !res) return PDF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    LaunchScope a(s, "k_vegas_estimate");
    k_vegas_estimate<<<1, 32, 0, s>>>(n, sums, res);
    CK(cudaGetLastError());
    return PDF_OK;
}

int pdf_vegas_refine(int ndim, int nbins, const double *hist, double alpha, double *edges, double *scratch, void *stream)
{
    if (ndim < 1 || nbins < 1 || !hist || !edges || !scratch || !(alpha >= 0.0)) return PDF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    LaunchScope a(s, "k_vegas_refine");
    k_vegas_refine<<<(ndim + 31) / 32, 32, 0, s>>>(ndim, nbins, hist, alpha, edges, scratch);
    CK(cudaGetLastError());
    return PDF_OK;
}

int pdf_vegas_combine(int M, const double *E, const double *S2, double *res, void *stream)
{
    if (M < 1 || !E || !S2 || !res) return PDF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    LaunchScope a(s, "k_vegas_combine");
    k_vegas_combine<<<1, 32, 0, s>>>(M, E, S2, res);
    CK(cudaGetLastError());
    return PDF_OK;
}

int pdf_unweight(long long n, const double *w, const double *u, unsigned char *accept, void *scratch16,
                 double *wmax, long long *n_accept, void *stream)
{
    if (n < 0 || !scratch16) return PDF_EINVAL;
    if (n && (!w || !u || !accept)) return PDF_EINVAL;
    cudaStream_t s = (cudaStream_t)stream;
    unsigned long long *sc = (unsigned long long *)scratch16;
    CK(cudaMemsetAsync(sc, 0, 16, s));
    if (n) {
        int sms = 148, dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        const long long want = (n + 255) / 256;
        const unsigned grid = (unsigned)(want < (long long)sms * 8 ? want : (long long)sms * 8);
        { LaunchScope a(s, "k_weight_max"); k_weight_max<<<grid, 256, 0, s>>>(n, w, sc); }
        { LaunchScope a(s, "k_unweight"); k_unweight<<<grid, 256, 0, s>>>(n, w, u, sc, accept, sc + 1); }
        CK(cudaGetLastError());
    }
    if (wmax || n_accept) {
        unsigned long long h[2] = {0, 0};
        CK(cudaMemcpyAsync(h, sc, 16, cudaMemcpyDeviceToHost, s));
        CK(cudaStreamSynchronize(s));
        if (wmax) std::memcpy(wmax, &h[0], 8);
        if (n_accept) *n_accept = (long long)h[1];
    }
    return PDF_OK;
}

}  // extern "C"
