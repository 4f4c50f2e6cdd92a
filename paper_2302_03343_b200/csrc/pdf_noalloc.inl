// pdf_noalloc.inl -- pdf_xfxq2_noalloc (included at the end of pdfgrid.cu): the binned path's persistent kernel
// (k_pdf_stream, pdf_stream.cuh) for callers that may not allocate -- code under CUDA graph capture, tight serving
// loops, harnesses that forbid cudaMalloc.  The kernel's scratch (ticket / chunk counters, cell bins, class lists)
// lives in ONE file-scope static device array of PDF_NOALLOC_SCRATCH_BYTES (64 MiB) instead of a caller workspace:
//   - every GPU that loads the library holds the array until the process exits;
//   - the array's name is a host-side stand-in in host code, not a device address: its address is resolved with
//     cudaGetSymbolAddress once per device, at set-up (pdf_grid_create, with the grid's device current), and only that
//     pointer is ever handed to a kernel;
//   - all calls on a device share it, and it keeps the last call's contents: the counters that must start at zero are
//     cleared on the stream at the start of every call; two calls that overlap on the GPU (different streams, or two
//     grids on one device) race on it -- the caller orders them;
//   - the call runs the queries as ONE chunk in ONE ring slot (the general path keeps a ring of 8 slots of <= 256Ki
//     queries in flight), so n is limited by what one slot of this grid's geometry takes of the array.
// The entry point calls no cudaMalloc / cudaFree and no allocating library routine: a memset and a launch on `stream`.

namespace {

static __device__ __align__(256) unsigned char g_noalloc_scratch[PDF_NOALLOC_SCRATCH_BYTES];

constexpr int kNoallocMaxDev = 64;
void *g_noalloc_ptr[kNoallocMaxDev];           // the array's device address on every device that was set up
int g_noalloc_state[kNoallocMaxDev];           // 0: not yet resolved, 1: resolved
std::mutex g_noalloc_mu;

// set-up, once per device, with `device` current (pdf_grid_create calls it)
int noalloc_setup(int device, void **ptr)
{
    *ptr = nullptr;
    if (device < 0 || device >= kNoallocMaxDev) return PDF_EINVAL;
    std::lock_guard<std::mutex> l(g_noalloc_mu);
    if (!g_noalloc_state[device]) {
        void *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) return cuda_fail(e, "cudaGetSymbolAddress(g_noalloc_scratch)");
        g_noalloc_ptr[device] = p;
        g_noalloc_state[device] = 1;
    }
    *ptr = g_noalloc_ptr[device];
    return PDF_OK;
}

// one ring slot for one chunk: [ctrl | counts (nbins + 32) | bins nbins * cap | lists kNumLists * chunk]
size_t noalloc_slot_bytes(const StreamPlan &p, long long chunk, StreamDev &d)
{
    stream_caps(p, chunk, d);
    size_t b = sizeof(unsigned long long) * kCtrlWords;
    b += align_up(sizeof(unsigned) * (size_t)(d.nbins + 32), 256);
    b += align_up(sizeof(Payload) * (size_t)d.nbins * d.cap, 256);
    b += align_up(sizeof(Payload) * (size_t)kNumLists * chunk, 256);
    return b;
}

// the largest n (a multiple of the A tile) whose slot fits the array; the slot size does not decrease with n
long long noalloc_max_n(const StreamPlan &p)
{
    if (!p.usable) return 0;
    StreamDev d;
    long long lo = 0, hi = (1LL << 24) / kS3TileA;                 // tiles; 2^24 queries would need > 3 GB
    while (lo < hi) {
        const long long mid = (lo + hi + 1) / 2;
        if (noalloc_slot_bytes(p, mid * kS3TileA, d) <= (size_t)PDF_NOALLOC_SCRATCH_BYTES) lo = mid; else hi = mid - 1;
    }
    return lo * kS3TileA;
}

}  // namespace

extern "C" {

int pdf_xfxq2_noalloc(const pdf_grid *g, const int *pids, int npid, long long n, const double *x, const double *q2,
                      double *out, long long *max_n, void *stream)
{
    if (!g) return PDF_EINVAL;
    const long long limit = noalloc_max_n(g->bplan);
    if (max_n) *max_n = limit;
    if (n < 0) return PDF_EINVAL;
    ColMap cm;
    int rc = build_colmap(g, pids, npid, cm);
    if (rc) return rc;
    if (!g->bplan.usable || limit <= 0) return PDF_ELIMIT;        // the grid does not fit the binned path or the array
    if (n > limit) return PDF_ELIMIT;
    if (n == 0) return PDF_OK;
    if (!x || !q2 || !out) return PDF_EINVAL;
    if (!g->noalloc_ws) { g_last_cuda_error = "the static scratch array was not resolved at pdf_grid_create"; return PDF_ECUDA; }
    if ((rc = on_device(g))) return rc;
    cudaStream_t s = (cudaStream_t)stream;

    StreamArgs A;
    A.ctab = nullptr; A.nchunks_dev = nullptr; A.orig = nullptr;
    A.x2 = nullptr; A.w = nullptr; A.f1 = nullptr; A.coup = g->bplan.d_coup;
    A.G = g->d; A.cm = cm;
    A.chunk = (n + kS3TileA - 1) / kS3TileA * kS3TileA;            // the whole call is one chunk
    if (noalloc_slot_bytes(g->bplan, A.chunk, A.B) > (size_t)PDF_NOALLOC_SCRATCH_BYTES) return PDF_ELIMIT;
    {
        char *c = (char *)g->noalloc_ws;                            // 256-byte aligned by declaration
        A.W.ctrl = (unsigned long long *)c; c += sizeof(unsigned long long) * kCtrlWords;
        A.W.counts = (unsigned *)c; c += align_up(sizeof(unsigned) * (size_t)(A.B.nbins + 32), 256);
        A.W.bins = (Payload *)c; c += align_up(sizeof(Payload) * (size_t)A.B.nbins * A.B.cap, 256);
        A.W.lists = (Payload *)c;
    }
    A.x = x; A.q2 = q2; A.out = out; A.n = n; A.ld = npid;
    A.nchunks = 1;
    A.ta = (int)(A.chunk / kS3TileA);
    A.identity = cm.n == kNF;
    for (int f = 0; f < kNF && A.identity; ++f) A.identity = cm.col[f] == f;
    A.count_err = 1;
    A.q_is_q = 0;
    // the array keeps the last call's contents: the ticket, the slot's counters and the bin / list counts start at zero
    const size_t zero_bytes = (size_t)((char *)A.W.bins - (char *)A.W.ctrl);
    CK(cudaMemsetAsync(A.W.ctrl, 0, zero_bytes, s));
    const size_t smem = stream_smem_bytes(g->d, A.B);
    int per_sm = 0, sms = 0;
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, g->device));
    const auto kern = g->d.extrap != kExtrapContinuation ? k_pdf_stream_opt : A.identity ? k_pdf_stream : k_pdf_stream_cols;   // rows of npid doubles: the stride fits 32 bits
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kS3Threads, smem));
    if (per_sm < 1) return PDF_ECUDA;
    const unsigned long long max_ctas = (unsigned long long)per_sm * sms;         // all CTAs must be co-resident
    const unsigned long long tickets = (unsigned long long)(A.ta + A.B.tb);
    const unsigned long long want = (tickets + kS3Warps - 1) / kS3Warps;
    g_launches.fetch_add(1, std::memory_order_relaxed);
    kern<<<(unsigned)(want < max_ctas ? want : max_ctas), kS3Threads, smem, s>>>(A);
    CK(cudaGetLastError());
    g->last_path = PDF_PATH_BINNED;
    return PDF_OK;
}

}  // extern "C"
