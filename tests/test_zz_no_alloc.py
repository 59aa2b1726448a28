"""pce_radial_profile_static -- the double-layer observables (eqs. 48-49) for callers that cannot allocate
device memory: an analysis hook that runs inside a simulation engine whose own pool holds the GPU's memory, where a cudaMalloc
can fail mid-run or stall the device between the engine's kernels.  The entry point takes the ions, the bead charges and the
output arrays from the caller and keeps its only scratch (the shell counters) in a fixed array of the library image.

What is checked: its output against the existing path (pce_radial_profile on a context) on the same ions and the same centre,
to the tolerances tests/test_gpu_dynamics.py holds that path to against the oracle (counts exact, g 1e-12, rho 1e-12 of its
scale, Q'(r) 1e-11) -- on TWO calls in a row with different shells and different charges, because the counter array is shared
and keeps the previous call's contents: a call that forgot to clear it would fail the second comparison.  The size limit is
checked too (that part needs no GPU).

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the parity
tests of the hot path.  It passes alone in a fresh process and after the other tests (the first call on a device does the
one-time address look-up wherever it happens)."""
import ctypes

import numpy as np
import pytest

import workloads as wl


def test_more_shells_than_the_fixed_array_holds_is_refused_with_a_message():
    """No GPU needed: the size check comes before any CUDA call."""
    import paper_2401_04865_b200 as pce
    pce.build()
    lib = pce.load()
    err = ctypes.create_string_buffer(512)
    d3 = (ctypes.c_double * 3)(10.0, 10.0, 10.0)
    rc = lib.pce_radial_profile_static(None, 0, None, None, None, None, 0, None, d3, d3, 0.1, 1.0, pce.PROFILE_STATIC_MAX_BINS + 1,
                                       None, None, None, None, err, len(err))
    assert rc == -1  # PCE_EINVAL
    msg = err.value.decode()
    assert "PCE_PROFILE_STATIC_MAX_BINS" in msg and str(pce.PROFILE_STATIC_MAX_BINS) in msg
    rc = lib.pce_radial_profile_static(None, 0, None, None, None, None, 0, None, d3, d3, 0.1, 1.0, 0, None, None, None, None, err, len(err))
    assert rc == -1 and b"n_bins" in err.value


@pytest.mark.gpu
def test_static_scratch_profile_equals_the_context_path_on_two_calls_in_a_row():
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = wl.config3(n_salt=3000)
    assert (w.x >= 0).all() and (w.x < w.L).all()  # the context's wrap into the box is then the identity
    ctx = pce.context_for(w, tol=1e-6)
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    # a stated reference point, so that both paths measure distances from the same centre (pce_set_centres)
    centre = np.asarray(w.L) * 0.5 + np.array([0.013, -0.021, 0.008])
    ctx.set_centres(*(torch.tensor([c], dtype=torch.float64, device="cuda") for c in centre))
    nbead = w.N_bead
    rng = np.random.default_rng(5)
    q_first = torch.cat([torch.full((nbead,), float(w.Q_body[0]) / nbead, dtype=torch.float64, device="cuda"), qi])
    # second call: other shells, some ions neutral, the species swapped, other bead charges
    flip = torch.from_numpy(np.where(rng.uniform(size=w.N_ion) < 0.1, 0.0, -1.3)).cuda()
    q_second = torch.cat([torch.from_numpy(rng.normal(size=nbead)).cuda(), qi * flip])
    xi, yi, zi = x[nbead:].contiguous(), y[nbead:].contiguous(), z[nbead:].contiguous()
    for q, r_lo, nb in ((q_first, 1.0, 5000), (q_second, 2.5, 3777), (q_first, 0.0, pce.PROFILE_STATIC_MAX_BINS)):
        want = ctx.radial_profile(0, q, r_lo, nb)
        got = pce.radial_profile_static(xi, yi, zi, q[nbead:].contiguous(), q[:nbead].contiguous(), centre, w.L, w.a, r_lo, nb)
        torch.cuda.synchronize()
        cw = want["counts"].cpu().numpy()                       # (n_bins, 2)
        cg = got["counts"].view(2, nb).T.cpu().numpy()
        assert cw.sum() > 500 and (cg == cw).all()
        assert np.allclose(got["g"].view(2, nb).T.cpu().numpy(), want["g"].cpu().numpy(), rtol=1e-12, atol=0)
        rw = want["rho"].cpu().numpy()
        assert np.abs(got["rho"].cpu().numpy() - rw).max() < 1e-12 * np.abs(rw).max()
        Qw = want["Qcum"].cpu().numpy()
        assert np.abs(got["Qcum"].cpu().numpy() - Qw).max() < 1e-11 * np.abs(Qw).max()
    with pytest.raises(pce.PceError, match="PCE_PROFILE_STATIC_MAX_BINS"):
        pce.radial_profile_static(xi, yi, zi, qi, None, centre, w.L, w.a, 0.0, pce.PROFILE_STATIC_MAX_BINS + 1)
    ctx.close()
