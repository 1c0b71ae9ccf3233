import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def dense_4x4_smooth():
    """Dense Q (3072 x 3072) on 4^4 with exp(0.3 i H) links at m = -1.6, its eigendecomposition and the exact
    sign function - shared by the sign / low-mode pins (BASELINE.json north_star, fourth oracle check)."""
    import numpy as np

    from lattice_inputs import gauge_field
    from oracle import wilson

    dims = (4, 4, 4, 4)
    U = gauge_field(dims, "smooth", eps=0.3)
    m = -1.6
    Qmat = wilson.dense_Q(U, m)
    lam, W = np.linalg.eigh(0.5 * (Qmat + Qmat.conj().T))
    return dict(dims=dims, U=U, m=m, Qmat=Qmat, lam=lam, W=W)
