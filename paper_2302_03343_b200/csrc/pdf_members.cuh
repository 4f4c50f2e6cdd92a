// pdf_members.cuh -- a-8, the member axis on the binned path (configs[3]: 100 replica grids, one
// member id per query).
//
// All members share the knots, so cell search, t_x / t_q and the node weights do not depend on
// the member; only the values do.  With ~10^6 (member, cell) pairs no chunk of 3.6e5 queries is
// cell-coherent, so the queries of a slice (<= 2^25) are first partitioned by member:
//   k_member_hist     histogram of the member ids of the slice (shared-memory counters per CTA)
//   k_member_plan     exclusive scan -> first slot of every member; chunk table: every member's run
//                     is cut in equal pieces of <= chunk queries {first, count, member}
//   k_member_scatter  x, q2 -> xs, q2s in member order; orig[slot] = the query the slot came from.  A
//                     CTA ranks its 4096 queries per member in shared memory, reserves its runs with
//                     one global atomic per (CTA, member), sorts the tile in shared memory and writes
//                     the runs out in slot order (~40 consecutive slots per run at 100 members);
//                     queries with a member id outside [0, nmem) get their NaN row here and count as
//                     errors (C-10)
//   k_pdf_stream      the persistent binned kernel over the chunk table: chunk c evaluates against
//                     V + member(c) * memstride; the payload carries orig[slot], so every row goes
//                     straight to its query's place in `out` (no sorted copy, no gather pass)
// The order of the queries inside a member's run is whatever the atomics gave: every row depends on
// its own query only, so the result does not.
#pragma once

namespace pdfg {

constexpr long long kMemSlice = 1 << 25;      // queries partitioned at a time (scratch: 20 B per query of a slice)
constexpr int kMemMax = 4096;                 // members the shared-memory histograms hold
constexpr int kMemTileQ = 8;                  // queries per thread of k_member_scatter
constexpr int kMemScatThreads = 512;          // its CTA: 4096 queries, sorted by member in shared memory before they leave
constexpr unsigned kNoSlot = 0xffffffffu;

struct MemberWs {
    unsigned *hist;       // [nmem]
    unsigned *cursor;     // [nmem] next free slot of every member's run
    int *nchunks;         // [1]
    int *ctab;            // [max_chunks][4]
    unsigned *orig;       // [slice] query (slice-local) of every slot
    double *xs, *q2s;     // [slice]
};

// slices of equal length for a call of n queries
inline long long member_slice(long long n)
{
    const long long ns = (n + kMemSlice - 1) / kMemSlice;
    long long sl = ns ? (n + ns - 1) / ns : 0;
    sl = (sl + 2047) / 2048 * 2048;
    return sl < n ? sl : n;
}

inline long long member_max_chunks(long long slice, long long chunk, int nmem) { return (slice + chunk - 1) / chunk + nmem; }

inline size_t member_scratch_bytes(long long slice, long long chunk, int nmem, int npid)
{
    size_t b = 3 * align_up(sizeof(unsigned) * (size_t)nmem + 16, 256);
    b += align_up(sizeof(int) * 4 * (size_t)member_max_chunks(slice, chunk, nmem), 256);
    b += align_up(sizeof(unsigned) * (size_t)slice, 256);
    b += 2 * align_up(sizeof(double) * (size_t)slice, 256);
    (void)npid;
    return b + 256;
}

inline void member_carve(void *p, long long slice, long long chunk, int nmem, MemberWs &w)
{
    char *c = (char *)align_up((size_t)p, 256);
    const size_t hb = align_up(sizeof(unsigned) * (size_t)nmem + 16, 256);
    w.hist = (unsigned *)c; c += hb;
    w.cursor = (unsigned *)c; c += hb;
    w.nchunks = (int *)c; c += hb;
    w.ctab = (int *)c; c += align_up(sizeof(int) * 4 * (size_t)member_max_chunks(slice, chunk, nmem), 256);
    w.orig = (unsigned *)c; c += align_up(sizeof(unsigned) * (size_t)slice, 256);
    w.xs = (double *)c; c += align_up(sizeof(double) * (size_t)slice, 256);
    w.q2s = (double *)c;
}

__global__ void __launch_bounds__(256)
k_member_hist(const int *__restrict__ member, long long n, int nmem, unsigned *__restrict__ hist)
{
    extern __shared__ unsigned s_h[];
    for (int k = threadIdx.x; k < nmem; k += blockDim.x) s_h[k] = 0u;
    __syncthreads();
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        const int m = __ldcs(member + e);
        if (m >= 0 && m < nmem) atomicAdd(s_h + m, 1u);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < nmem; k += blockDim.x) {
        const unsigned c = s_h[k];
        if (c) atomicAdd(hist + k, c);
    }
}

// one CTA: scan of the histogram and the chunk table (a few hundred entries)
__global__ void __launch_bounds__(256)
k_member_plan(const unsigned *__restrict__ hist, int nmem, int chunk, unsigned *__restrict__ cursor,
              int *__restrict__ ctab, int *__restrict__ nchunks)
{
    extern __shared__ unsigned s_h[];
    for (int k = threadIdx.x; k < nmem; k += blockDim.x) s_h[k] = hist[k];
    __syncthreads();
    if (threadIdx.x) return;
    unsigned start = 0;
    int nc = 0;
    for (int m = 0; m < nmem; ++m) {
        const unsigned cnt = s_h[m];
        cursor[m] = start;
        const unsigned pieces = (cnt + (unsigned)chunk - 1) / (unsigned)chunk;
        unsigned step = pieces ? (cnt + pieces - 1) / pieces : 0u;     // equal pieces, whole A tiles (chunk is a multiple)
        step = (step + kS3TileA - 1) / kS3TileA * kS3TileA;
        for (unsigned o = 0; o < cnt; o += step) {
            const unsigned len = cnt - o < step ? cnt - o : step;
            reinterpret_cast<int4 *>(ctab)[nc++] = make_int4((int)(start + o), (int)len, m, 0);
        }
        start += cnt;
    }
    *nchunks = nc;
}

// shared memory of k_member_scatter: 3 counter arrays, warp totals, then the tile sorted by member
inline size_t member_scatter_smem(int nmem)
{
    return align_up(sizeof(unsigned) * 3 * (size_t)nmem + 256, 16) + (size_t)kMemScatThreads * kMemTileQ * (8 + 8 + 2 + 2);
}

__global__ void __launch_bounds__(kMemScatThreads)
k_member_scatter(const double *__restrict__ x, const double *__restrict__ q2, const int *__restrict__ member,
                 long long n, int nmem, unsigned *__restrict__ cursor, double *__restrict__ xs,
                 double *__restrict__ q2s, unsigned *__restrict__ orig, double *__restrict__ out, long long ld, int npid,
                 unsigned long long *err_count)
{
    constexpr int T = kMemScatThreads, TILE = T * kMemTileQ;
    extern __shared__ __align__(16) unsigned char s_raw[];
    unsigned *s_c = reinterpret_cast<unsigned *>(s_raw);          // [nmem] queries of the tile per member
    unsigned *s_b = s_c + nmem;                                   // [nmem] first global slot of the tile's run
    unsigned *s_l = s_b + nmem;                                   // [nmem] first slot of the run inside the sorted tile
    unsigned *s_w = s_l + nmem;                                   // [T/32 + 1] scan scratch
    double *sx = reinterpret_cast<double *>(s_raw + align_up(sizeof(unsigned) * 3 * (size_t)nmem + 256, 16));
    double *sq = sx + TILE;
    unsigned short *sm = reinterpret_cast<unsigned short *>(sq + TILE);
    unsigned short *so = sm + TILE;                               // the query's place inside the tile
    for (int k = threadIdx.x; k < nmem; k += T) s_c[k] = 0u;
    __syncthreads();
    const long long t0 = (long long)blockIdx.x * TILE;
    unsigned tag[kMemTileQ];                      // member << 16 | rank inside the CTA's tile
    double xv[kMemTileQ], qv[kMemTileQ];
#pragma unroll
    for (int q = 0; q < kMemTileQ; ++q) {
        const long long e = t0 + q * T + threadIdx.x;
        tag[q] = kNoSlot;
        xv[q] = 0.0; qv[q] = 0.0;
        if (e < n) {
            const int m = __ldcs(member + e);
            xv[q] = __ldcs(x + e); qv[q] = __ldcs(q2 + e);
            if (m >= 0 && m < nmem) tag[q] = ((unsigned)m << 16) | atomicAdd(s_c + m, 1u);
        }
    }
    __syncthreads();
    // one global atomic per (CTA, member); exclusive scan of the counts = the runs inside the sorted tile
    for (int k = threadIdx.x; k < nmem; k += T) {
        const unsigned c = s_c[k];
        s_b[k] = c ? atomicAdd(cursor + k, c) : 0u;
    }
    {
        const int per = (nmem + T - 1) / T, b0 = threadIdx.x * per;
        unsigned sum = 0;
        for (int i = 0; i < per; ++i) if (b0 + i < nmem) sum += s_c[b0 + i];
        unsigned inc = sum;
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { unsigned v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
        if (lane == 31) s_w[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            unsigned w = lane < T / 32 ? s_w[lane] : 0u, wi = w;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { unsigned v = __shfl_up_sync(0xffffffffu, wi, d); if (lane >= d) wi += v; }
            if (lane < T / 32) s_w[lane] = wi - w;
            if (lane == 31) s_w[T / 32] = wi;                     // valid queries of the tile
        }
        __syncthreads();
        unsigned run = s_w[warp] + inc - sum;
        for (int i = 0; i < per; ++i) if (b0 + i < nmem) { s_l[b0 + i] = run; run += s_c[b0 + i]; }
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < kMemTileQ; ++q) {
        const long long e = t0 + q * T + threadIdx.x;
        if (e >= n) continue;
        if (tag[q] != kNoSlot) {
            const unsigned m = tag[q] >> 16, rank = tag[q] & 0xffffu;
            const unsigned l = s_l[m] + rank;
            sx[l] = xv[q]; sq[l] = qv[q]; sm[l] = (unsigned short)m; so[l] = (unsigned short)(q * T + threadIdx.x);
        } else {                                                  // no such member: NaN row, counted (C-10)
            double *o = out + e * ld;
            for (int p = 0; p < npid; ++p) o[p] = qnan();
            atomicAdd(err_count, 1ULL);
        }
    }
    __syncthreads();
    // the sorted tile leaves in slot order: consecutive threads write consecutive slots of a run
    const unsigned total = s_w[T / 32];
    for (unsigned j = threadIdx.x; j < total; j += T) {
        const unsigned m = sm[j], g = s_b[m] + (j - s_l[m]);
        xs[g] = sx[j];
        q2s[g] = sq[j];
        orig[g] = (unsigned)t0 + so[j];
    }
}

}  // namespace pdfg
