// pdfgrid.cu -- the C ABI of include/pdfgrid.h: handle management, grid layout (a-1), and the
// host-side dispatch of every evaluation call.  All arithmetic of the path runs in the kernels of
// pdf_generic.cuh / pdf_binned.cuh; nothing here computes a PDF value on the host.
#include "../../include/pdfgrid.h"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "pdf_common.cuh"
#include "pdf_generic.cuh"
#include "pdf_stream.cuh"
#include "mc_kernels.cuh"

using namespace pdfg;

namespace {

thread_local std::string g_last_cuda_error;
std::atomic<long long> g_launches{0};

struct ProfEntry { const char *name; cudaEvent_t a, b; };
std::mutex g_prof_mu;
bool g_prof_on = false;
std::vector<ProfEntry> g_prof;

int cuda_fail(cudaError_t e, const char *what)
{
    g_last_cuda_error = std::string(what) + ": " + cudaGetErrorString(e);
    return PDF_ECUDA;
}
#define CK(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return cuda_fail(e__, #call); } while (0)

// every kernel launch of the library goes through these two: count it, optionally time it
struct LaunchScope {
    cudaStream_t s; const char *name; ProfEntry pe{}; bool on;
    LaunchScope(cudaStream_t st, const char *nm, int launches = 1) : s(st), name(nm)
    {
        g_launches.fetch_add(launches, std::memory_order_relaxed);
        on = g_prof_on;
        if (on) { cudaEventCreate(&pe.a); cudaEventCreate(&pe.b); pe.name = nm; cudaEventRecord(pe.a, s); }
    }
    ~LaunchScope()
    {
        if (on) { cudaEventRecord(pe.b, s); std::lock_guard<std::mutex> l(g_prof_mu); g_prof.push_back(pe); }
    }
};

template <typename T> int dev_alloc(T **p, size_t n)
{
    cudaError_t e = cudaMalloc((void **)p, n * sizeof(T));
    if (e != cudaSuccess) { g_last_cuda_error = std::string("cudaMalloc: ") + cudaGetErrorString(e); return PDF_ENOMEM; }
    return PDF_OK;
}

bool finite_pos_h(double v) { return std::isfinite(v) && v > 0.0; }

struct HostStage {           // device staging of the *_host calls, one per pipeline slot
    cudaStream_t stream = nullptr;
    double *in = nullptr, *out = nullptr; void *ws = nullptr;
    size_t in_doubles = 0, out_doubles = 0, ws_bytes = 0;
};

}  // namespace

struct pdf_grid {
    GridDev d{};
    int device = 0;
    std::vector<double> xk, qk;
    std::vector<int> nq, qoff, pids;
    // owned device allocations
    double *d_xk = nullptr, *d_qk = nullptr, *d_uk = nullptr, *d_sk = nullptr, *d_V = nullptr;
    int *d_sub_of = nullptr, *d_qoff = nullptr, *d_cell_adj = nullptr;
    CellTab *d_cx = nullptr, *d_cq = nullptr, *d_ca = nullptr;
    double *d_ak = nullptr, *d_alk = nullptr, *d_av = nullptr, *d_C = nullptr, *d_acell = nullptr;
    unsigned short *d_alut = nullptr;
    unsigned long long *d_err = nullptr;
    std::vector<double> h_av, h_ak, h_C;
    // caller-owned workspace of the binned path
    void *ws = nullptr; size_t ws_bytes = 0;
    int path = PDF_PATH_AUTO;
    long long chunk = 0;      // binned-path chunk size override (0 = default)
    HostStage stage[2];
    StreamPlan bplan{};       // key geometry and search tables of the binned path (pdf_stream.cuh)
    mutable int last_path = 0;  // PDF_PATH_DIRECT / PDF_PATH_BINNED: what the last evaluation call of this handle ran
    void *noalloc_ws = nullptr; // device address of the static scratch array on this grid's device (pdf_noalloc.inl)
};

namespace {

int noalloc_setup(int device, void **ptr);   // pdf_noalloc.inl

int col_of_pid(const pdf_grid *g, int pid)
{
    if (pid == 0) pid = 21;
    for (size_t f = 0; f < g->pids.size(); ++f) if (g->pids[f] == pid) return (int)f;
    return -1;
}

void free_grid(pdf_grid *g)
{
    if (!g) return;
    cudaFree(g->d_xk); cudaFree(g->d_qk); cudaFree(g->d_uk); cudaFree(g->d_sk); cudaFree(g->d_V);
    cudaFree(g->d_sub_of); cudaFree(g->d_qoff); cudaFree(g->d_cell_adj); cudaFree(g->d_cx); cudaFree(g->d_cq); cudaFree(g->d_ca);
    cudaFree(g->d_ak); cudaFree(g->d_alk); cudaFree(g->d_av); cudaFree(g->d_C); cudaFree(g->d_err);
    cudaFree(g->d_acell); cudaFree(g->d_alut);
    stream_plan_free(g->bplan);
    for (auto &s : g->stage) {
        cudaFree(s.in); cudaFree(s.out); cudaFree(s.ws);
        if (s.stream) cudaStreamDestroy(s.stream);
    }
    delete g;
}

}  // namespace

extern "C" {

const char *pdf_status_string(int status)
{
    switch (status) {
    case PDF_OK: return "ok";
    case PDF_EINVAL: return "invalid argument";
    case PDF_ENOMEM: return "out of memory";
    case PDF_ECUDA: return "CUDA runtime error";
    case PDF_EWORKSPACE: return "workspace missing or too small";
    case PDF_ESTATE: return "required grid data not set";
    case PDF_ELIMIT: return "size beyond what the static scratch of the no-allocation entry point holds (see its max_n)";
    default: return "unknown status";
    }
}

const char *pdf_last_cuda_error(void) { return g_last_cuda_error.c_str(); }
long long pdf_launch_count(void) { return g_launches.load(); }

int pdf_profile_enable(int on)
{
    std::lock_guard<std::mutex> l(g_prof_mu);
    for (auto &p : g_prof) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
    g_prof.clear();
    g_prof_on = on != 0;
    return PDF_OK;
}

int pdf_profile_read(int max_entries, const char **names, float *ms)
{
    std::lock_guard<std::mutex> l(g_prof_mu);
    int n = 0;
    for (auto &p : g_prof) {
        if (n >= max_entries) break;
        if (cudaEventSynchronize(p.b) != cudaSuccess) break;
        float t = 0.f;
        cudaEventElapsedTime(&t, p.a, p.b);
        if (names) names[n] = p.name;
        if (ms) ms[n] = t;
        ++n;
    }
    for (auto &p : g_prof) { cudaEventDestroy(p.a); cudaEventDestroy(p.b); }
    g_prof.clear();
    return n;
}

int pdf_grid_create(pdf_grid **out, int nx, const double *x_knots, int nsub, const int *nq,
                    const double *q2_knots, const double *values, int nflav,
                    const int *flavour_pids, int nmem)
{
    if (!out || !x_knots || !nq || !q2_knots || !values || !flavour_pids) return PDF_EINVAL;
    if (nx < 2 || nsub < 1 || nflav < 1 || nflav > 64 || nmem < 1) return PDF_EINVAL;
    for (int i = 0; i < nx; ++i) {
        if (!finite_pos_h(x_knots[i])) return PDF_EINVAL;
        if (i && !(x_knots[i] > x_knots[i - 1])) return PDF_EINVAL;
    }
    int tot = 0;
    for (int k = 0; k < nsub; ++k) {
        if (nq[k] < 2) return PDF_EINVAL;
        for (int j = 0; j < nq[k]; ++j) {
            double q = q2_knots[tot + j];
            if (!finite_pos_h(q)) return PDF_EINVAL;
            if (j && !(q > q2_knots[tot + j - 1])) return PDF_EINVAL;
        }
        if (k && std::memcmp(&q2_knots[tot], &q2_knots[tot - 1], sizeof(double)) != 0) return PDF_EINVAL;
        tot += nq[k];
    }
    size_t per_mem = (size_t)nx * tot * nflav;
    for (size_t e = 0; e < per_mem * nmem; ++e) if (!std::isfinite(values[e])) return PDF_EINVAL;

    pdf_grid *g = new (std::nothrow) pdf_grid();
    if (!g) return PDF_ENOMEM;
    cudaGetDevice(&g->device);
    g->xk.assign(x_knots, x_knots + nx);
    g->qk.assign(q2_knots, q2_knots + tot);
    g->nq.assign(nq, nq + nsub);
    g->pids.assign(flavour_pids, flavour_pids + nflav);
    g->qoff.resize(nsub + 1);
    std::vector<int> sub_of(tot), cell_adj(tot);
    g->qoff[0] = 0;
    for (int k = 0; k < nsub; ++k) {
        g->qoff[k + 1] = g->qoff[k] + nq[k];
        for (int j = 0; j < nq[k]; ++j) { sub_of[g->qoff[k] + j] = k; cell_adj[g->qoff[k] + j] = (j == nq[k] - 1) ? 1 : 0; }
    }
    int nfp = (nflav + 1) & ~1;                       // even: 16-byte vector loads of a node row
    size_t vdev = (size_t)nmem * tot * nx * nfp;
    int rc = PDF_OK;
#define TRY(expr) do { rc = (expr); if (rc != PDF_OK) { free_grid(g); return rc; } } while (0)
#define TRYC(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { rc = cuda_fail(e__, #call); free_grid(g); return rc; } } while (0)
    TRY(dev_alloc(&g->d_xk, nx)); TRY(dev_alloc(&g->d_uk, nx));
    TRY(dev_alloc(&g->d_qk, tot)); TRY(dev_alloc(&g->d_sk, tot));
    TRY(dev_alloc(&g->d_sub_of, tot)); TRY(dev_alloc(&g->d_qoff, nsub + 1)); TRY(dev_alloc(&g->d_cell_adj, tot));
    TRY(dev_alloc(&g->d_cx, nx)); TRY(dev_alloc(&g->d_cq, tot));
    TRY(dev_alloc(&g->d_V, vdev)); TRY(dev_alloc(&g->d_err, 1));
    double *d_src = nullptr;
    TRY(dev_alloc(&d_src, per_mem * nmem));
    TRYC(cudaMemcpy(g->d_xk, x_knots, sizeof(double) * nx, cudaMemcpyHostToDevice));
    TRYC(cudaMemcpy(g->d_qk, q2_knots, sizeof(double) * tot, cudaMemcpyHostToDevice));
    TRYC(cudaMemcpy(g->d_sub_of, sub_of.data(), sizeof(int) * tot, cudaMemcpyHostToDevice));
    TRYC(cudaMemcpy(g->d_cell_adj, cell_adj.data(), sizeof(int) * tot, cudaMemcpyHostToDevice));
    TRYC(cudaMemcpy(g->d_qoff, g->qoff.data(), sizeof(int) * (nsub + 1), cudaMemcpyHostToDevice));
    TRYC(cudaMemcpy(d_src, values, sizeof(double) * per_mem * nmem, cudaMemcpyHostToDevice));
    TRYC(cudaMemset(g->d_err, 0, sizeof(unsigned long long)));
    TRYC(cudaMemset(g->d_cq, 0, sizeof(CellTab) * tot));
    {   // a-1: the layout kernels
        LaunchScope a(0, "k_log_knots");
        k_log_knots<<<(nx + 127) / 128, 128>>>(g->d_xk, g->d_uk, nx);
    }
    { LaunchScope a(0, "k_log_knots"); k_log_knots<<<(tot + 127) / 128, 128>>>(g->d_qk, g->d_sk, tot); }
    { LaunchScope a(0, "k_cell_tables"); k_cell_tables<<<(nx + 127) / 128, 128>>>(g->d_uk, g->d_cx, 0, nx); }
    size_t suboff = 0;
    for (int k = 0; k < nsub; ++k) {
        { LaunchScope a(0, "k_cell_tables");
          k_cell_tables<<<(nq[k] + 127) / 128, 128>>>(g->d_sk, g->d_cq, g->qoff[k], nq[k]); }
        size_t cnt = (size_t)nx * nq[k] * nfp * nmem;
        { LaunchScope a(0, "k_relayout");
          k_relayout<<<(unsigned)((cnt + 255) / 256), 256>>>(d_src, g->d_V, nx, nq[k], nflav, nfp, tot,
                                                            g->qoff[k], per_mem, suboff, nmem); }
        suboff += (size_t)nx * nq[k] * nflav;
    }
    cudaError_t e = cudaDeviceSynchronize();
    cudaFree(d_src);
    if (e != cudaSuccess) { rc = cuda_fail(e, "grid layout"); free_grid(g); return rc; }
#undef TRY
#undef TRYC
    GridDev &d = g->d;
    d.nx = nx; d.nsub = nsub; d.nflav = nflav; d.nfp = nfp; d.nmem = nmem; d.nqtot = tot;
    d.xk = g->d_xk; d.qk = g->d_qk; d.uk = g->d_uk; d.sk = g->d_sk;
    d.sub_of = g->d_sub_of; d.qoff = g->d_qoff; d.cell_adj = g->d_cell_adj; d.cx = g->d_cx; d.cq = g->d_cq;
    d.V = g->d_V; d.memstride = (size_t)tot * nx * nfp;
    d.q2plus = 1.01 * q2_knots[0];
    d.na = 0; d.alphas_mode = PDF_ALPHAS_FREEZE; d.extrap = PDF_EXTRAP_CONTINUATION; d.C = nullptr; d.err_count = g->d_err;
    rc = stream_plan_init(g->bplan, g->d, g->xk, g->qk, nsub);
    if (rc != PDF_OK) { free_grid(g); return rc; }
    // pdf_xfxq2_noalloc: the static scratch array's address on this device (resolved once per device; no allocation).
    // A failure leaves the pointer null and only that entry point unusable.
    noalloc_setup(g->device, &g->noalloc_ws);
    *out = g;
    return PDF_OK;
}

int pdf_grid_destroy(pdf_grid *g)
{
    free_grid(g);
    return PDF_OK;
}

int pdf_grid_set_alphas(pdf_grid *g, int n, const double *q2_knots, const double *values)
{
    if (!g || n < 2 || !q2_knots || !values) return PDF_EINVAL;
    // knots increase; a knot may appear twice (a flavour threshold: the end of one sub-line and the start of the next,
    // PAPER.md L1835), every sub-line has at least 2 knots
    for (int j = 0; j < n; ++j) {
        if (!finite_pos_h(q2_knots[j]) || !std::isfinite(values[j])) return PDF_EINVAL;
        if (j && !(q2_knots[j] >= q2_knots[j - 1])) return PDF_EINVAL;
        if (j && q2_knots[j] == q2_knots[j - 1] && (j == 1 || j == n - 1 || q2_knots[j - 1] == q2_knots[j - 2] ||
                                                      q2_knots[j + 1] == q2_knots[j])) return PDF_EINVAL;
    }
    cudaFree(g->d_ak); cudaFree(g->d_alk); cudaFree(g->d_av); cudaFree(g->d_ca); cudaFree(g->d_acell); cudaFree(g->d_alut);
    g->d_ak = g->d_alk = g->d_av = g->d_acell = nullptr; g->d_ca = nullptr; g->d_alut = nullptr; g->d.na = 0;
    int rc;
    if ((rc = dev_alloc(&g->d_ak, n)) || (rc = dev_alloc(&g->d_alk, n)) || (rc = dev_alloc(&g->d_av, n)) ||
        (rc = dev_alloc(&g->d_ca, n)) || (rc = dev_alloc(&g->d_acell, 6 * (size_t)n)) || (rc = dev_alloc(&g->d_alut, kAlphaLutMax))) return rc;
    CK(cudaMemcpy(g->d_ak, q2_knots, sizeof(double) * n, cudaMemcpyHostToDevice));
    CK(cudaMemcpy(g->d_av, values, sizeof(double) * n, cudaMemcpyHostToDevice));
    { LaunchScope a(0, "k_log_knots"); k_log_knots<<<(n + 127) / 128, 128>>>(g->d_ak, g->d_alk, n); }
    // cell constants per sub-line (one-sided slopes at its ends, C-5); the zero-width cell between the two copies of a
    // threshold is never selected: the search takes the LATER copy of a repeated knot (C-3)
    CK(cudaMemset(g->d_ca, 0, sizeof(CellTab) * n));
    for (int first = 0; first < n;) {
        int last = first;
        while (last + 1 < n && q2_knots[last + 1] != q2_knots[last]) ++last;
        const int m = last - first + 1;
        LaunchScope a(0, "k_cell_tables");
        k_cell_tables<<<(m + 127) / 128, 128>>>(g->d_alk, g->d_ca, first, m);
        first = last + 1;
    }
    { LaunchScope a(0, "k_alphas_cells"); k_alphas_cells<<<(n + 127) / 128, 128>>>(g->d_ca, g->d_av, g->d_acell, n); }
    {   // search table on the bit pattern of Q2: entry = the cell at the bucket's lower edge (the walk on the device makes it exact)
        std::vector<double> k(q2_knots, q2_knots + n);
        std::vector<unsigned short> lut;
        make_search_table(k, n - 2, g->d.ashift, g->d.abase, lut);
        g->d.nalut = (int)lut.size();
        CK(cudaMemcpy(g->d_alut, lut.data(), sizeof(unsigned short) * lut.size(), cudaMemcpyHostToDevice));
    }
    CK(cudaDeviceSynchronize());
    g->d.na = n; g->d.ak = g->d_ak; g->d.alk = g->d_alk; g->d.av = g->d_av; g->d.ca = g->d_ca;
    g->d.acell = g->d_acell; g->d.alut = g->d_alut;
    return PDF_OK;
}

int pdf_grid_set_coupling(pdf_grid *g, const double *C)
{
    if (!g || !C) return PDF_EINVAL;
    size_t n = (size_t)g->d.nflav * g->d.nflav;
    for (size_t e = 0; e < n; ++e) if (!std::isfinite(C[e])) return PDF_EINVAL;
    if (!g->d_C) { int rc = dev_alloc(&g->d_C, n); if (rc) return rc; }
    CK(cudaMemcpy(g->d_C, C, sizeof(double) * n, cudaMemcpyHostToDevice));
    g->d.C = g->d_C;
    g->h_C.assign(C, C + n);
    return PDF_OK;
}

int pdf_grid_set_workspace(pdf_grid *g, void *dev_ptr, size_t bytes)
{
    if (!g) return PDF_EINVAL;
    g->ws = dev_ptr; g->ws_bytes = dev_ptr ? bytes : 0;
    return PDF_OK;
}

int pdf_grid_set_option(pdf_grid *g, int option, long long value)
{
    if (!g) return PDF_EINVAL;
    switch (option) {
    case PDF_OPT_PATH:
        if (value < PDF_PATH_AUTO || value > PDF_PATH_BINNED) return PDF_EINVAL;
        g->path = (int)value; return PDF_OK;
    case PDF_OPT_ALPHAS_MODE:
        if (value != PDF_ALPHAS_FREEZE && value != PDF_ALPHAS_LOGGRAD) return PDF_EINVAL;
        g->d.alphas_mode = (int)value; return PDF_OK;
    case PDF_OPT_EXTRAPOLATION:
        if (value < PDF_EXTRAP_CONTINUATION || value > PDF_EXTRAP_ERROR) return PDF_EINVAL;
        g->d.extrap = (int)value; return PDF_OK;
    case PDF_OPT_CHUNK:
        if (value < 0) return PDF_EINVAL;
        g->chunk = value; return PDF_OK;
    default: return PDF_EINVAL;
    }
}

int pdf_grid_limits(const pdf_grid *g, double *xmin, double *xmax, double *q2min, double *q2max)
{
    if (!g) return PDF_EINVAL;
    if (xmin) *xmin = g->xk.front();
    if (xmax) *xmax = g->xk.back();
    if (q2min) *q2min = g->qk.front();
    if (q2max) *q2max = g->qk.back();
    return PDF_OK;
}

}  // extern "C"

#include "pdfgrid_eval.inl"
#include "mc_entry.inl"
#include "pdf_noalloc.inl"
