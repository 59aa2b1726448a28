"""Host logic of the CUDA library (no GPU): the piecewise-polynomial table of the real-space pair kernel
(csrc/realtab.h) against the oracle's closed form of eq. 20 and its derivative, for the Ewald
parameters of all five configurations.  The table is product code; the oracle shares nothing with it."""
import numpy as np
import pytest

import oracle as orc
import paper_2401_04865_b200 as pce

# (bead radius a, box L, grid) of configs 1-5
CASES = [(0.137952, 10.0, 32), (0.069142, 20.0, 64), (0.034591, 40.0, 128), (0.069142, 16.0, 256), (0.0992, 43.756, 512)]


@pytest.mark.parametrize("a,L,Ng", CASES)
def test_table_matches_closed_form(a, L, Ng):
    pce.build()
    p = pce.suggest_params([L] * 3, [Ng] * 3, a, 1e-10)
    xi, rc = p.xi, p.rc
    rng = np.random.default_rng(3)
    r = np.concatenate([
        np.exp(rng.uniform(np.log(0.26 * a), np.log(rc * 0.999999), size=20000)),   # log-uniform over the whole range
        2 * a * (1 + np.array([-1e-3, -1e-9, 0.0, 1e-9, 1e-3])),                      # around the kink at r = 2a
        np.linspace(0.26 * a, 2 * a, 2001), np.linspace(2 * a, rc * 0.999999, 4001),
    ])
    R, dR = pce.real_kernel_host(a, xi, rc, r)
    assert np.all(np.isfinite(R)) and np.all(np.isfinite(dR))
    Ro = np.array([orc.R(t, a, xi) for t in r])
    dRo = np.array([orc.dR(t, a, xi) for t in r])
    # absolute accuracy on the scale of the contact value R(2a): sums of ~200 such terms must hold 1e-9 relative
    scale, dscale = abs(orc.R(2 * a, a, xi)), abs(orc.dR(2 * a, a, xi))
    assert np.abs(R - Ro).max() < 2e-13 * scale
    assert np.abs(dR - dRo).max() < 2e-12 * dscale
    # and relative accuracy where the kernel is not yet negligible (further out the closed form itself, a
    # cancelling sum of O(1) terms in fp64, is no better than ~1e-17 absolute)
    big = np.abs(Ro) > 1e-4 * scale
    assert (np.abs(R - Ro)[big] / np.abs(Ro)[big]).max() < 1e-11


def test_out_of_range_is_nan_and_bad_arguments():
    pce.build()
    R, dR = pce.real_kernel_host(0.1, 3.0, 1.5, np.array([0.01, 1.6, 0.5]))
    assert np.isnan(R[0]) and np.isnan(R[1]) and np.isfinite(R[2])
    with pytest.raises(pce.PceError):
        pce.real_kernel_host(-0.1, 3.0, 1.5, np.array([0.5]))
