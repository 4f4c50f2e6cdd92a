import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


def make_oracle_grid(oracle, spec):
    g = oracle.OracleGrid(spec.x_knots.numpy(), [q.numpy() for q in spec.q2_subgrids],
                          spec.values.numpy(), spec.pids, nmem=spec.nmem)
    if spec.alphas_q2 is not None:
        g.set_alphas(spec.alphas_q2.numpy(), spec.alphas_val.numpy())
    if spec.coupling is not None:
        g.set_coupling(spec.coupling.numpy())
    return g
