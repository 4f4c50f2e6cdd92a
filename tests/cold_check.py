"""Run by test_gpu_parity.test_binned_first_calls_in_a_fresh_process: the first binned calls of a
process (cold caches, freshly allocated outputs: the spin-waits of the pipeline are really taken)
must agree with the direct kernels."""
import os
import sys

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2302_03343_b200 import binding as B, synth  # noqa: E402

n = int(sys.argv[1])
spec = synth.grid_c1()
x, q = synth.queries_c2(spec, n, seed=synth.BASE_SEED + 31)
g = B.PdfGrid.from_spec(spec, workspace_for=n)
xd, qd = x.cuda(), q.cuda()
g.pdf_grid_set_option(B.PDF_OPT_PATH, B.PDF_PATH_DIRECT)
d = g.pdf_xfxq2(spec.pids, xd, qd).cpu().numpy()
g.pdf_grid_set_option(B.PDF_OPT_PATH, B.PDF_PATH_BINNED)
worst = 0
for rep in range(3):
    b = g.pdf_xfxq2(spec.pids, xd, qd).cpu().numpy()
    assert np.array_equal(np.isnan(b), np.isnan(d))
    err = np.abs(np.nan_to_num(b) - np.nan_to_num(d)) / (np.abs(np.nan_to_num(d)) + 1e-30)
    bad = int((err.max(axis=1) > 1e-9).sum())
    worst = max(worst, bad)
print("COLD_BAD_ROWS", worst)
sys.exit(1 if worst else 0)
