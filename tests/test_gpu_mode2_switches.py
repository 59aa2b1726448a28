"""The library's switches through FFT mode 2 -- the own (x, y) passes of fftxy.cu plus the fused z pass, the only arrangement the
512^3 headline configuration runs -- on 128^3 and 256^3 meshes.  A small system on a large mesh keeps the oracle cheap (its cost
depends on the particle count only), so every particle is compared:
  PCE_FLAG_FIELD_IK: k_zfft_scale with a derivative index into the second spectrum, then the inverse passes
                         that discard consumed rows; psi, E <= 1e-9 against the oracle, wave-space momentum <= 1e-13;
  P_matvec = P - 2       (pce.h): the solver matvec's own window, bins and Green's-function tables; psi and q <= 1e-9;
  PCE_FLAG_DETERMINISTIC : two runs bit for bit, and <= 1e-9 against the oracle.
Plus the long fibers of PAPER.md:333 (aspect ratios up to 40), which need these mesh sizes."""
import numpy as np
import pytest

import oracle as orc
import workloads as wl
from conftest import body_vector_error

pytestmark = pytest.mark.gpu


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - b) / max(np.linalg.norm(b), 1e-300))


def _E(out):
    import torch
    return torch.stack(out[1:], dim=1).cpu().numpy()


def _system(ng):
    return wl.tiny_random(seed=70 + ng, n_body=2, n_ion=50, L=6.0, Ng=ng, neutral=False)


@pytest.mark.parametrize("ng", [128, 256])
def test_ik_field_mode_through_the_own_fft_passes(ng):
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = _system(ng)
    q = np.random.default_rng(ng).normal(size=w.N)
    q -= q.mean()
    psi_o, E_o = orc.ewald_eval(w.x, q, w.L, w.a)
    ctx = pce.context_for(w, field_ik=True)
    assert ctx.info()["fft_mode"] == 2
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    for _ in range(2):                                   # twice: the second spectrum and the row discards leave nothing behind
        out = ctx.evaluate(torch.from_numpy(q).cuda())
        psi, E = out[0].cpu().numpy(), _E(out)
        assert rel(psi, psi_o) < 1e-9 and rel(E, E_o) < 1e-9, (rel(psi, psi_o), rel(E, E_o))
        # total force of the wave-space part vanishes to rounding; the real-space part is pairwise antisymmetric
        assert np.abs((q[:, None] * E).sum(axis=0)).max() < 1e-13 * np.abs(q[:, None] * E).sum(axis=0).max()
    # and through the solve: fields of the induced charges
    qs, Phi, info = ctx.solve(Q, qi, w.E0)
    f = ctx.forces(qs, w.E0)
    qo, Phio, _ = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
    oo = orc.forces_torques(w.x, w.body_offset, qo, w.E0, w.L, w.a, Phi_body=Phio)
    assert info["converged"] and rel(qs.cpu().numpy(), qo) < 1e-9 and rel(f["f"].cpu().numpy(), oo["f"]) < 1e-8
    ctx.close()


@pytest.mark.parametrize("ng", [128, 256])
def test_narrower_solver_window_through_the_own_fft_passes(ng):
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = _system(ng)
    ctx = pce.context_for(w, tol=1e-11)                  # P = 22
    P = ctx.params.P
    ctx.close()
    ctx = pce.context_for(w, tol=1e-11, P_matvec=P - 2)
    info = ctx.info()
    assert info["fft_mode"] == 2 and info["P_matvec"] == P - 2
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    qb = np.random.default_rng(ng + 1).normal(size=w.N_bead)
    psi_o = orc.ewald_eval(w.x[:w.N_bead], qb, w.L, w.a, field=False)
    assert rel(ctx.matvec(torch.from_numpy(qb).cuda()).cpu().numpy(), psi_o) < 1e-9
    q, Phi, si = ctx.solve(Q, qi, w.E0)
    f = ctx.forces(q, w.E0)
    qo, Phio, _ = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
    oo = orc.forces_torques(w.x, w.body_offset, qo, w.E0, w.L, w.a, Phi_body=Phio)
    assert si["converged"] and rel(q.cpu().numpy(), qo) < 1e-9
    assert rel(f["psi"].cpu().numpy(), oo["psi"]) < 1e-9 and rel(f["f"].cpu().numpy(), oo["f"]) < 1e-8
    ctx.close()


@pytest.mark.parametrize("ng", [128, 256])
def test_deterministic_gather_through_the_own_fft_passes(ng):
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = _system(ng)
    qv = torch.from_numpy(np.random.default_rng(ng + 2).normal(size=w.N)).cuda()
    runs = []
    for _ in range(2):
        ctx = pce.context_for(w, deterministic=True)
        assert ctx.info()["fft_mode"] == 2
        x, y, z, Q, qi = pce.upload(w)
        ctx.set_system(w.body_offset, x, y, z)
        ev = [t.clone() for t in ctx.evaluate(qv)]
        q, Phi, si = ctx.solve(Q, qi, w.E0)
        f = ctx.forces(q, w.E0)
        runs.append(ev + [q.clone(), f["f"].clone(), f["T"].clone()])
        ctx.close()
    for u, v in zip(*runs):
        assert torch.equal(u, v)
    psi_o, E_o = orc.ewald_eval(w.x, qv.cpu().numpy(), w.L, w.a)
    assert rel(runs[0][0].cpu().numpy(), psi_o) < 1e-9
    assert rel(torch.stack(runs[0][1:4], dim=1).cpu().numpy(), E_o) < 1e-9
    qo, _, _ = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
    assert rel(runs[0][4].cpu().numpy(), qo) < 1e-9


@pytest.mark.parametrize("chi,ng", [(20, 128), (40, 256)])
def test_long_fibers_dipole_and_torque(chi, ng):
    """Aspect ratios 20 and 40 (PAPER.md:333 studies chi = 5 ... 40): induced charges, dipole, bead forces and the aligning torque
    of a four-line fiber along and at 45 degrees to the field, against the oracle's dense solve."""
    import paper_2401_04865_b200 as pce
    pce.build()
    for deg in (0, 45):
        w = wl.fiber_in_field(chi=chi, theta=np.deg2rad(deg), Ng=ng)
        ctx = pce.context_for(w)
        x, y, z, Q, qi = pce.upload(w)
        ctx.set_system(w.body_offset, x, y, z)
        q, Phi, info = ctx.solve(Q, qi, w.E0)
        assert info["converged"]
        out = ctx.forces(q, w.E0)
        qo, Phio, _ = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
        oo = orc.forces_torques(w.x, w.body_offset, qo, w.E0, w.L, w.a, Phi_body=Phio)
        assert rel(q.cpu().numpy(), qo) < 1e-9, (deg, rel(q.cpu().numpy(), qo))
        assert rel(out["S"].cpu().numpy(), oo["S"]) < 1e-9
        assert rel(out["f"].cpu().numpy(), oo["f"]) < 1e-8
        eT, kind = body_vector_error(out["T"].cpu().numpy(), oo["T"], oo["f"])
        assert eT < 1e-8, (deg, eT, kind)
        if deg == 45:
            assert kind == "rel" and out["T"][0, 1].item() < 0
        ctx.close()
