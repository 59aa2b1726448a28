"""Brownian-dynamics step (eqs. 40-46, 62) and double-layer observables (eqs. 48-49) on the device against the oracle
(oracle/dynamics.py): identical noise -- the library's own Philox stream against the oracle's own implementation of the same
generator -- so positions after a step agree to rounding; then config 3 as BASELINE.json states it (100 steps, dt = 1e-4)
driven entirely on the device, with per-frame electrostatics parity on the identical positions."""
import numpy as np
import pytest

import oracle as orc
from oracle import dynamics as ody
import workloads as wl
from conftest import body_vector_error

pytestmark = pytest.mark.gpu


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - b) / max(np.linalg.norm(b), 1e-300))


def _min_image(d, L):
    return d - L * np.round(d / L)


def _pos(x, y, z):
    import torch
    return torch.stack([x, y, z], dim=1).cpu().numpy()


def _ctx(w, **kw):
    import paper_2401_04865_b200 as pce
    pce.build()
    ctx = pce.context_for(w, **kw)
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    return ctx, Q, qi


def test_one_step_matches_the_oracle_with_the_generators_own_noise():
    """Crowded small system (many overlaps on purpose: ions placed at random), bodies moving: positions after one step <= 1e-12
    of the box, with the device's Philox normals against the oracle's."""
    import torch
    rng = np.random.default_rng(77)
    w = wl.config2(d=2.6, n_ion=300)
    x0 = w.x.copy()
    # squeeze some ions into overlap with each other and with the spheres' beads (hard-sphere forces of all three kinds)
    x0[w.N_bead:w.N_bead + 40] = x0[w.N_bead + 40:w.N_bead + 80] + rng.normal(size=(40, 3)) * 0.6 * w.a
    x0[w.N_bead + 100:w.N_bead + 120] = x0[:20] + rng.normal(size=(20, 3)) * 0.8 * w.a
    x0[w.N_bead + 120:w.N_bead + 130] = x0[700:710] + rng.normal(size=(10, 3)) * 0.8 * w.a
    w.x = x0 - w.L * np.floor(x0 / w.L)
    ctx, Q, qi = _ctx(w)
    f = torch.from_numpy(rng.normal(size=(w.N, 3)) * 5.0).cuda()
    dt, gamma, kT, seed, step = 3e-4 * w.a ** 2, 1.3, 0.9, 20240104 + (7 << 33), 12
    for move in (False, True):
        if move:
            ctx.set_positions(*(torch.from_numpy(np.ascontiguousarray(w.x[:, d])).cuda() for d in range(3)))
        xg = _pos(*ctx.bd_step(f, dt, gamma, kT, seed=seed, step=step, move_bodies=move))
        noise = ody.normals(seed, step, w.N_ion)
        xo = ody.bd_step(w.x, w.body_offset, f.cpu().numpy(), w.L, w.a, dt, gamma, kT, noise, move_bodies=move)
        hs = ody.hard_sphere_forces(w.x, w.body_offset, w.L, w.a, gamma, dt)
        assert np.count_nonzero(np.abs(hs).sum(axis=1)) > 100            # the case exercises eq. 46
        assert np.abs(hs[:w.N_bead]).sum() > 0 and np.abs(hs[w.N_bead:]).sum() > 0
        err = np.abs(_min_image(xg - xo, w.L)).max()
        assert err < 1e-12 * w.L[0], (move, err)
        if not move:
            assert (xg[:w.N_bead] == w.x[:w.N_bead]).all()
        else:
            assert np.abs(_min_image(xg[:w.N_bead] - w.x[:w.N_bead], w.L)).max() > 1e-9
            # rigid: bead-bead distances inside a body unchanged
            b0, b1 = w.x[:642], xg[:642]
            d0 = np.linalg.norm(_min_image(b0[:50, None] - b0[None, :50], w.L), axis=2)
            d1 = np.linalg.norm(_min_image(b1[:50, None] - b1[None, :50], w.L), axis=2)
            assert np.abs(d1 - d0).max() < 1e-12
    # caller-supplied noise takes the place of the generator
    ctx.set_positions(*(torch.from_numpy(np.ascontiguousarray(w.x[:, d])).cuda() for d in range(3)))
    nz = rng.normal(size=(w.N_ion, 3))
    xg = _pos(*ctx.bd_step(f, dt, gamma, kT, noise=torch.from_numpy(nz).cuda()))
    xo = ody.bd_step(w.x, w.body_offset, f.cpu().numpy(), w.L, w.a, dt, gamma, kT, nz)
    assert np.abs(_min_image(xg - xo, w.L)).max() < 1e-12 * w.L[0]
    # the context advanced: the operator now acts at the new positions
    q = torch.from_numpy(rng.normal(size=w.N)).cuda()
    psi = ctx.evaluate(q, field=False).cpu().numpy()
    po = orc.ewald_eval(xo, q.cpu().numpy(), w.L, w.a, field=False)
    assert rel(psi, po) < 1e-9
    ctx.close()


def test_hard_sphere_image_path_and_edge_cases():
    """2a-cells collapse to explicit images in a thin box; ions only; a pair in exact contact feels nothing."""
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    rng = np.random.default_rng(3)
    L, Ng, a = np.array([1.0, 4.0, 4.0]), np.array([16, 32, 32]), 0.2   # L_x / 2a = 2.5 < 3 cells
    n = 160
    x = rng.uniform(0, 1, (n, 3)) * L
    p = pce.suggest_params(L, Ng, a, 1e-6)
    ctx = pce.Context(p)
    t = [torch.from_numpy(np.ascontiguousarray(x[:, d])).cuda() for d in range(3)]
    ctx.set_system(np.array([0], dtype=np.int32), *t)
    f = torch.zeros(n, 3, dtype=torch.float64, device="cuda")
    xg = _pos(*ctx.bd_step(f, 1e-3, 1.0, 0.0))
    xo = ody.bd_step(x, [0], np.zeros((n, 3)), L, a, 1e-3, 1.0, 0.0, np.zeros((n, 3)), brute=True)
    assert np.abs(ody.hard_sphere_forces(x, [0], L, a, 1.0, 1e-3, brute=True)).sum() > 0
    assert np.abs(_min_image(xg - xo, L)).max() < 1e-13
    ctx.close()


def test_radial_profile_matches_the_oracle():
    import torch
    w = wl.config3(n_salt=3000)
    ctx, Q, qi = _ctx(w, tol=1e-6)
    q = torch.cat([torch.full((w.N_bead,), float(w.Q_body[0]) / w.N_bead, dtype=torch.float64, device="cuda"), qi])
    r_lo, nb = 1.0, 5000
    out = ctx.radial_profile(0, q, r_lo, nb)
    X, _ = orc.body_centres(w.x, w.body_offset, w.L)
    o = ody.radial_profile(w.x[w.N_bead:], w.q_ion, X[0], w.L, w.a, r_lo, nb, Q=float(w.Q_body[0]))
    assert (out["counts"].cpu().numpy() == o["counts"]).all() and o["counts"].sum() > 1000
    assert np.allclose(out["g"].cpu().numpy(), o["g"], rtol=1e-12, atol=0)
    scale = np.abs(o["rho"]).max()
    assert np.abs(out["rho"].cpu().numpy() - o["rho"]).max() < 1e-12 * scale
    assert np.abs(out["Qcum"].cpu().numpy() - o["Qcum"]).max() < 1e-11 * np.abs(o["Qcum"]).max()
    ctx.close()
