"""Run by test_gpu_parity.test_binned_first_calls_in_a_fresh_process: the first binned calls of a
process (cold caches, freshly allocated outputs: the spin-waits of the pipeline are really taken)
must agree with the direct kernels."""
import os
import sys

import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2302_03343_b200 import binding as B, synth  # noqa: E402

n = int(sys.argv[1])
spec = synth.grid_c1()
x, q = synth.queries_c2(spec, n, seed=synth.BASE_SEED + 31)
g = B.PdfGrid.from_spec(spec, workspace_for=n)
xd, qd = x.cuda(), q.cuda()
g.pdf_grid_set_option(B.PDF_OPT_PATH, B.PDF_PATH_DIRECT)
d = g.pdf_xfxq2(spec.pids, xd, qd)
g.pdf_grid_set_option(B.PDF_OPT_PATH, B.PDF_PATH_BINNED)
worst = 0
for rep in range(3 if n <= 4_000_000 else 2):
    b = g.pdf_xfxq2(spec.pids, xd, qd)
    assert torch.equal(torch.isnan(b), torch.isnan(d))
    # on the device: every row; the two kernels sum in different orders, so an element may differ by a few ulp of
    # the stencil's scale (bounded below by the row's largest value) where it cancels, else by ~1e-15 relative
    dz = d.nan_to_num()
    err = (b.nan_to_num() - dz).abs()
    tol = 1e-9 * dz.abs() + 1e-11 * dz.abs().max(dim=1, keepdim=True).values + 1e-300
    bad = int(((err > tol).any(dim=1)).sum())
    del dz, tol
    worst = max(worst, bad)
    del b, err
print("COLD_BAD_ROWS", worst)
sys.exit(1 if worst else 0)
