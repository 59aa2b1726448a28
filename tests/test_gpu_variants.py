"""SURVEY.md 8(f) f4 variants on the device: ik-differentiated fields (PCE_FLAG_FIELD_IK) and rod-like "fiber"
bodies of four bead lines, each against the oracle at the north-star bars."""
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


@pytest.mark.parametrize("fused_z", [True, False])
def test_ik_field_mode_matches_the_oracle_and_conserves_momentum(fused_z):
    """E from -i k times the scaled spectrum: parity <= 1e-9 with the oracle (and so with the window-gradient mode), and the
    total electrostatic force sum_a q_a E_a vanishes to rounding -- spread and gather use the same window, the ik multiplier is
    odd in k -- which the window-gradient mode only does to the Ewald tolerance."""
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = wl.config2(d=2.4)
    rng = np.random.default_rng(5)
    q = rng.normal(size=w.N)
    q -= q.mean()
    psi_o, E_o = orc.ewald_eval(w.x, q, w.L, w.a)
    tot = {}
    for ik in (True, False):
        ctx = pce.context_for(w, field_ik=ik, fused_z=fused_z)
        x, y, z, Q, qi = pce.upload(w)
        ctx.set_system(w.body_offset, x, y, z)
        out = ctx.evaluate(torch.from_numpy(q).cuda())
        psi, E = out[0].cpu().numpy(), _E(out)
        assert rel(psi, psi_o) < 1e-9 and rel(E, E_o) < 1e-9, (ik, rel(psi, psi_o), rel(E, E_o))
        tot[ik] = np.abs((q[:, None] * E).sum(axis=0)).max() / np.abs(q[:, None] * E).sum(axis=0).max()
        ctx.close()
    assert tot[True] < 1e-13, tot
    assert tot[True] < 0.05 * tot[False], tot


def test_ik_field_mode_in_a_rectangular_box_and_through_the_solve():
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = wl.tiny_random(seed=21, n_body=2, n_ion=40, L=6.0, Ng=32)
    w.L = np.array([6.0, 7.5, 9.0])
    w.Ng = np.array([32, 40, 48])          # N_z = 48: the 3-D cuFFT path with the separate scaling pass
    ctx = pce.context_for(w, field_ik=True)
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    q, Phi, info = ctx.solve(Q, qi, w.E0)
    out = ctx.forces(q, w.E0)
    qo, Phio, _ = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
    oo = orc.forces_torques(w.x, w.body_offset, qo, w.E0, w.L, w.a, Phi_body=Phio)
    assert rel(q.cpu().numpy(), qo) < 1e-9 and rel(out["f"].cpu().numpy(), oo["f"]) < 1e-8
    assert body_vector_error(out["F"].cpu().numpy(), oo["F"], oo["f"])[0] < 1e-8
    assert body_vector_error(out["T"].cpu().numpy(), oo["T"], oo["f"])[0] < 1e-8
    ctx.close()


@pytest.mark.parametrize("chi", [5, 10])
def test_fiber_dipole_and_torque_versus_angle(chi):
    """Fig. 4 of the paper as a parity case: dipole and torque of a four-line fiber at 0, 30, 45, 90 degrees to the field."""
    import paper_2401_04865_b200 as pce
    pce.build()
    for deg in (0, 30, 45, 90):
        w = wl.fiber_in_field(chi=chi, theta=np.deg2rad(deg), Ng=64 if chi == 5 else 96)
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
        if deg in (30, 45):
            assert kind == "rel" and out["T"][0, 1].item() < 0      # a real torque, towards alignment with E0
        ctx.close()


def test_fiber_with_ions_full_parity():
    import paper_2401_04865_b200 as pce
    pce.build()
    w = wl.fiber_in_field(chi=10, theta=0.6, n_ion=400, Ng=96)
    ctx = pce.context_for(w)
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    q, Phi, info = ctx.solve(Q, qi, w.E0)
    out = ctx.forces(q, w.E0)
    qo, Phio, _ = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
    oo = orc.forces_torques(w.x, w.body_offset, qo, w.E0, w.L, w.a, Phi_body=Phio)
    assert rel(q.cpu().numpy(), qo) < 1e-9 and rel(out["psi"].cpu().numpy(), oo["psi"]) < 1e-9
    assert rel(out["f"].cpu().numpy(), oo["f"]) < 1e-8
    assert body_vector_error(out["F"].cpu().numpy(), oo["F"], oo["f"])[0] < 1e-8
    assert body_vector_error(out["T"].cpu().numpy(), oo["T"], oo["f"])[0] < 1e-8
    ctx.close()


def test_set_centres_moves_the_reference_point_only():
    """pce_set_centres (eq. 12): with X_i shifted by d_i the charges are unchanged, Phi_i grows by d_i.E0 (the
    constant r.E0 loses), S_i = S_i - d_i Q_i and T_i = T_i - d_i x F_i -- textbook change of reference point, with the
    un-shifted run already pinned to the oracle."""
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = wl.tiny_random(seed=33, n_body=3, n_ion=30, L=7.0, Ng=32, neutral=True)
    ctx = pce.context_for(w)
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    q0, Phi0, _ = ctx.solve(Q, qi, w.E0)
    o0 = ctx.forces(q0, w.E0)
    X0, _ = orc.body_centres(w.x, w.body_offset, w.L)
    d = np.random.default_rng(1).normal(size=(w.N_body, 3)) * 0.3
    Xn = torch.from_numpy(np.ascontiguousarray((X0 + d).T)).cuda()
    ctx.set_centres(Xn[0].contiguous(), Xn[1].contiguous(), Xn[2].contiguous())
    q1, Phi1, _ = ctx.solve(Q, qi, w.E0)
    o1 = ctx.forces(q1, w.E0)
    assert rel(q1.cpu().numpy(), q0.cpu().numpy()) < 1e-10
    assert np.allclose(Phi1.cpu().numpy(), Phi0.cpu().numpy() + d @ w.E0, rtol=0, atol=1e-9 * np.abs(Phi0.cpu().numpy()).max())
    F0, T0, S0 = (o0[k].cpu().numpy() for k in ("F", "T", "S"))
    assert np.allclose(o1["F"].cpu().numpy(), F0, atol=1e-9 * np.abs(F0).max())
    assert np.allclose(o1["S"].cpu().numpy(), S0 - d * w.Q_body[:, None], atol=1e-9 * np.abs(S0).max())
    assert np.allclose(o1["T"].cpu().numpy(), T0 - np.cross(d, F0), atol=1e-9 * max(np.abs(T0).max(), np.abs(F0).max()))
    ctx.close()


def test_deterministic_flag_gives_bit_identical_results():
    """PCE_FLAG_DETERMINISTIC (deterministic reductions): two evaluations and two solves of the same inputs
    agree bit for bit, and with the oracle / the default (atomic) gather to the usual bars."""
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = wl.config2(d=2.3)
    rng = np.random.default_rng(8)
    qv = torch.from_numpy(rng.normal(size=w.N)).cuda()
    outs = []
    for det in (True, True, False):
        ctx = pce.context_for(w, deterministic=det)
        x, y, z, Q, qi = pce.upload(w)
        ctx.set_system(w.body_offset, x, y, z)
        ev = [t.clone() for t in ctx.evaluate(qv)]
        mv = ctx.matvec(qv[:w.N_bead].contiguous()).clone()
        q, Phi, info = ctx.solve(Q, qi, w.E0)
        f = ctx.forces(q, w.E0)
        outs.append((ev, mv, q.clone(), f["f"].clone(), f["T"].clone()))
        ctx.close()
    a, b, c = outs
    for u, v in zip(a[0] + [a[1], a[2], a[3], a[4]], b[0] + [b[1], b[2], b[3], b[4]]):
        assert torch.equal(u, v)                                   # bit for bit
    for u, v in zip(a[0] + [a[1], a[2]], c[0] + [c[1], c[2]]):
        assert rel(u.cpu().numpy(), v.cpu().numpy()) < 1e-12       # the atomic gather differs by rounding only
    psi_o, E_o = orc.ewald_eval(w.x, qv.cpu().numpy(), w.L, w.a)
    assert rel(a[0][0].cpu().numpy(), psi_o) < 1e-9
    assert rel(torch.stack(a[0][1:], dim=1).cpu().numpy(), E_o) < 1e-9
    # a mesh off the brick lattice cannot honour the flag: refused at create
    w2 = wl.tiny_random(seed=3, n_body=1, n_ion=10, L=6.0, Ng=36)
    with pytest.raises(pce.PceError):
        pce.context_for(w2, deterministic=True)


def test_own_fft_passes_on_a_mesh_with_fewer_planes_than_rows():
    """FFT mode 2 (own (x, y) passes + fused z pass) on a 128 x 128 x 64 mesh in a flat box: the plane pipeline of fftxy.cu with
    N_z != N_x, against the oracle and against the cuFFT 3-D arrangement."""
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = wl.tiny_random(seed=41, n_body=2, n_ion=60, L=6.0, Ng=32)
    w.L = np.array([12.0, 12.0, 6.0])
    w.Ng = np.array([128, 128, 64])
    rng = np.random.default_rng(2)
    q = rng.normal(size=w.N)
    q -= q.mean()
    psi_o, E_o = orc.ewald_eval(w.x, q, w.L, w.a)
    res = {}
    for fused in (True, False):
        ctx = pce.context_for(w, fused_z=fused)
        assert ctx.info()["fft_mode"] == (2 if fused else 0)
        x, y, z, Q, qi = pce.upload(w)
        ctx.set_system(w.body_offset, x, y, z)
        out = ctx.evaluate(torch.from_numpy(q).cuda())
        res[fused] = (out[0].cpu().numpy(), _E(out))
        assert rel(res[fused][0], psi_o) < 1e-9 and rel(res[fused][1], E_o) < 1e-9
        ctx.close()
    assert rel(res[True][0], res[False][0]) < 1e-12


@pytest.mark.parametrize("ng", [256, 512])
def test_large_mesh_passes_against_the_oracle_on_full_vectors(ng):
    """The 256- and 512-point instances of the own FFT passes and of the fused z pass pinned to the oracle on EVERY particle (the
    oracle's cost depends on the particle count only, so a small system on a large mesh is cheap to check): potentials, fields,
    induced charges, torques."""
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = wl.tiny_random(seed=50 + ng, n_body=2, n_ion=50, L=6.0, Ng=ng, neutral=False)
    # Ewald tolerance 1e-11 (P = 22): the torque of a 12-bead icosahedron is a small difference of r x f terms, so the relative
    # torque error is the relative force error times that cancellation (about 10 here)
    ctx = pce.context_for(w, tol=1e-11)
    assert ctx.info()["fft_mode"] == 2
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    rng = np.random.default_rng(ng)
    qv = rng.normal(size=w.N)
    out = ctx.evaluate(torch.from_numpy(qv).cuda())
    psi_o, E_o = orc.ewald_eval(w.x, qv, w.L, w.a)
    assert rel(out[0].cpu().numpy(), psi_o) < 1e-9 and rel(_E(out), E_o) < 1e-9
    q, Phi, info = ctx.solve(Q, qi, w.E0)
    f = ctx.forces(q, w.E0)
    qo, Phio, _ = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
    oo = orc.forces_torques(w.x, w.body_offset, qo, w.E0, w.L, w.a, Phi_body=Phio)
    assert info["converged"] and rel(q.cpu().numpy(), qo) < 1e-9
    assert rel(f["f"].cpu().numpy(), oo["f"]) < 1e-8
    assert body_vector_error(f["T"].cpu().numpy(), oo["T"], oo["f"])[0] < 1e-8
    ctx.close()


def test_narrower_window_for_the_solver_matvec():
    """pce_params.P_matvec = P - 2: the solver's bead-only matvec spreads and gathers with 18 instead of 20 support points (its own
    bead binning, hit lists and Green's-function tables).  Potentials, and with them the induced charges, stay within the 1e-9
    bar; the final evaluation (fields, forces) still uses P."""
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = wl.config2(d=3.0)
    rng = np.random.default_rng(4)
    qb = rng.normal(size=w.N_bead)
    psi_o = orc.ewald_eval(w.x[:w.N_bead], qb, w.L, w.a, field=False)
    qo, Phio, _ = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
    oo = orc.forces_torques(w.x, w.body_offset, qo, w.E0, w.L, w.a, Phi_body=Phio)
    for fused in (True, False):
        ctx = pce.context_for(w, P_matvec=18, fused_z=fused)
        assert ctx.info()["P_matvec"] == 18 and ctx.params.P == 20
        x, y, z, Q, qi = pce.upload(w)
        ctx.set_system(w.body_offset, x, y, z)
        assert rel(ctx.matvec(torch.from_numpy(qb).cuda()).cpu().numpy(), psi_o) < 1e-9
        q, Phi, info = ctx.solve(Q, qi, w.E0)
        f = ctx.forces(q, w.E0)
        assert info["converged"] and rel(q.cpu().numpy(), qo) < 1e-9
        assert rel(f["psi"].cpu().numpy(), oo["psi"]) < 1e-9 and rel(f["f"].cpu().numpy(), oo["f"]) < 1e-8
        assert rel(f["S"].cpu().numpy(), oo["S"]) < 1e-9
        ctx.close()
    with pytest.raises(pce.PceError):
        pce.context_for(w, P_matvec=22)   # wider than P: refused
