"""GPU parity of the grand capacitance tensor (eq. 15) and of the effective permittivity (eq. 36-37,
PAPER.md:306-311) against the oracle's dense C = Sigma' M^-1 Sigma'^T.  The CUDA path solves M_bb q = Sigma'^T e_k per column
(plain preconditioned CG on the spectral-Ewald operator) and gets eps_eff from three constrained solves of eq. 13; the oracle
evaluates eq. 36 from the blocks of the dense C."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl

pytestmark = pytest.mark.gpu

TOL = 1e-9


@pytest.fixture(scope="module")
def pce():
    import torch
    import paper_2401_04865_b200 as p
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    p.build()
    return p


def _tensor(pce, w, cols=None, **kw):
    ctx = pce.context_for(w, **kw)
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    nb = w.N_body
    cols = np.arange(4 * nb) if cols is None else np.asarray(cols)
    Cg, info = ctx.capacitance_columns(cols)
    eps, einfo = ctx.effective_permittivity()
    ctx.close()
    assert info["converged"] and einfo["converged"], (info, einfo)
    return Cg.cpu().numpy(), eps, cols


def _check(pce, w, cols=None):
    Cg, eps, cols = _tensor(pce, w, cols)
    Co = orc.capacitance(w.x, w.body_offset, w.L, w.a, w.eps_f)
    nb = w.N_body
    # row j of the GPU result is column cols[j] of C; compare block by block on each block's own scale
    ref = Co[:, cols].T
    for name, sl in (("q", slice(0, nb)), ("S", slice(nb, 4 * nb))):
        for cname, csel in (("Psi", cols < nb), ("E", cols >= nb)):
            if not csel.any():
                continue
            blk, rblk = Cg[csel][:, sl], ref[csel][:, sl]
            scale = np.sqrt(np.abs(np.diag(Co)[sl]).max() * np.abs(np.diag(Co)[cols[csel]]).max())  # sqrt(C_ii C_kk): Cauchy-Schwarz scale
            assert np.abs(blk - rblk).max() < TOL * scale, (name, cname, np.abs(blk - rblk).max(), scale)
    eps_o = orc.effective_permittivity(Co, nb, float(np.prod(w.L)), w.eps_f)
    assert np.abs(eps - eps_o).max() < TOL * np.abs(eps_o).max(), (eps, eps_o)
    return Cg, Co, eps


def test_capacitance_single_sphere_config1(pce):
    """config 1: C_qE = C_SPsi = 0 by symmetry, C_SE = (S/E0) I with S the config-1 dipole (+14.8 %)."""
    w = wl.config1()
    Cg, Co, eps = _check(pce, w)
    assert np.abs(Cg - Cg.T).max() < 1e-9 * np.abs(Cg).max()
    assert np.abs(Cg[0, 1:]).max() < 1e-9 * np.sqrt(Cg[0, 0] * Cg[1, 1])
    assert Cg[3, 3] / (4 * np.pi) - 1 == pytest.approx(0.1484, abs=2e-4)
    assert eps[2, 2] == pytest.approx(1 + Cg[3, 3] / 1000.0, rel=1e-9)


def test_capacitance_two_spheres_config2(pce):
    """config 2 (two 642-bead spheres; the ions carry no unknowns and are left out of C): all 8 columns."""
    w = wl.config2(d=2.5)
    Cg, Co, eps = _check(pce, w)
    assert np.abs(Cg - Cg.T).max() < 1e-8 * np.abs(Cg).max()  # symmetric (M is)


def test_capacitance_cubic_lattice_couplings_vanish(pce):
    """2 x 2 x 2 simple-cubic array of identical spheres: body-summed couplings C_qE and C_SPsi vanish and
    eps_eff is isotropic; a subset of columns is enough for the parity check (first body: potential and the three fields)."""
    w = wl.config4(subdiv=2, nside=2, spacing=4.0, n_ion=0, with_ions=False, Ng=64)
    nb = w.N_body
    cols = [0, nb, nb + 1, nb + 2, 3, nb + 3 * 5 + 1]
    Cg, Co, eps = _check(pce, w, cols)
    # uniform field on all bodies: charge response sums to zero body by body
    assert np.abs(eps - eps[0, 0] * np.eye(3)).max() < 1e-9 * eps[0, 0]
    assert eps[0, 0] > 1.0
