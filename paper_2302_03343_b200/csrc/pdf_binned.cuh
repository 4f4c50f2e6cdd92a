// pdf_binned.cuh -- the binned, warp-coherent evaluation path (placeholder geometry; kernels follow).
#pragma once
#include "pdf_common.cuh"
#include "pdf_generic.cuh"

namespace pdfg {

struct BinnedPlan {
    int ncx = 0, ncq = 0;     // x cells, global Q2 cells (lower-knot index space)
    int nkeys = 0;
    bool usable = false;
};

inline void binned_plan_init(BinnedPlan &p, int nx, int nsub, const int *qoff, int nflav, int nmem)
{
    p.ncx = nx - 1;
    p.ncq = qoff[nsub];
    p.nkeys = 0;
    p.usable = false;
    (void)nflav; (void)nmem;
}

inline bool binned_qualifies(const BinnedPlan &p, const ColMap &, const int *member, long long) { return p.usable && !member; }
inline bool binned_lumi_qualifies(const BinnedPlan &p, long long) { return p.usable; }
inline size_t binned_workspace_bytes(const BinnedPlan &, long long, long long) { return 0; }
inline int binned_xfxq2(const GridDev &, const BinnedPlan &, const ColMap &, long long, const double *, const double *,
                        double *, long long, void *, size_t, long long, cudaStream_t) { return -1; }
inline int binned_lumi(const GridDev &, const BinnedPlan &, long long, const double *, const double *, const double *,
                       const double *, double *, void *, size_t, long long, cudaStream_t) { return -1; }

}  // namespace pdfg
