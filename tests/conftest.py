import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")
    config.addinivalue_line("markers", "slow: longer-running CPU check")


@pytest.fixture(scope="session")
def golden_dir():
    return os.path.join(ROOT, "tests", "golden")


def read_golden(path):
    """Golden files: '#' comment lines (with the citation), then 'key value' lines."""
    out = {}
    with open(path) as fh:
        for line in fh:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, v = line.split(None, 1)
            out[k] = float(v)
    return out


def body_vector_error(got, want, f_oracle, floor=1e-6):
    """Parity measure for per-body sums of bead forces (F_i, T_i: eq. 18), arrays of shape (N_body, 3).

    north_star: relative L2 <= 1e-8 on forces and torques.  The plain relative L2 error |got - want| / |want| is returned
    whenever the oracle's own norm is at least ``floor`` x the bead-force scale  max_d sum_a |f_a,d|; only when the body sums
    vanish by symmetry (a single sphere, the ion-free lattice: |want| is rounding noise of a sum of O(1) terms) the error is
    measured against that bead-force scale instead.  Returns (error, "rel" | "abs")."""
    import numpy as np
    got, want = np.asarray(got, dtype=np.float64), np.asarray(want, dtype=np.float64)
    fscale = float(np.abs(np.asarray(f_oracle)).sum(0).max())
    nw = float(np.linalg.norm(want))
    d = float(np.linalg.norm(got - want))
    if nw >= floor * fscale:
        return d / nw, "rel"
    return d / max(fscale, 1e-300), "abs"
