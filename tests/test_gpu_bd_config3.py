"""Config 3 as BASELINE.json states it: charged colloid (2562 beads, Q = -100 e) + 20 100 ions, 100 Brownian-dynamics
steps with dt = 1e-4 and Gaussian noise from the seed.  The whole trajectory runs on the device (pce_solve warm-started,
pce_forces, pce_bd_step with the library's Philox stream; the colloid is held fixed, reading A13); at frames 0, 50 and
99 the CUDA path is compared with the oracle on the IDENTICAL positions (trajectory-level parity is meaningless for chaotic
dynamics), and at those frames the step itself is compared with the oracle's step from the same forces."""
import numpy as np
import pytest

import oracle as orc
from oracle import dynamics as ody
import workloads as wl
from conftest import body_vector_error

pytestmark = pytest.mark.gpu


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - b) / max(np.linalg.norm(b), 1e-300))


def test_config3_100_bd_steps_parity_at_frames():
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    w = wl.config3()
    n_steps, frames = 100, (0, 50, 99)
    dt = 1e-4 * w.a ** 2  # time unit gamma a^2 / kT with a the bead radius (reading B5)
    seed = wl.configs.BASE_SEED + 3
    ctx = pce.context_for(w)
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    pos = torch.stack([x, y, z], dim=1)
    q_prev, its, kept = None, [], {}
    for step in range(n_steps):
        q, Phi, info = ctx.solve(Q, qi, w.E0, q0=q_prev)
        assert info["converged"], (step, info)
        out = ctx.forces(q, w.E0)
        its.append(info["iters"])
        q_prev = q
        xn = torch.stack(ctx.bd_step(out["f"], dt, 1.0, 1.0, seed=seed, step=step), dim=1)
        if step in frames:
            kept[step] = (pos.cpu().numpy(), q.cpu().numpy(), Phi.cpu().numpy(), out["psi"].cpu().numpy(), out["f"].cpu().numpy(),
                          out["F"].cpu().numpy(), out["T"].cpu().numpy(), xn.cpu().numpy())
        pos = xn
    ctx.close()
    L = float(w.L[0])
    pf = pos.cpu().numpy()
    # the colloid stayed where it was, the ions diffused by about sqrt(2 dt n) per coordinate, all positions are wrapped
    assert (pf[:w.N_bead] == w.x[:w.N_bead]).all()
    dx = pf[w.N_bead:] - w.x[w.N_bead:]
    dx -= L * np.round(dx / L)
    assert 0.8 < dx.std() / np.sqrt(2 * dt * n_steps) < 1.3
    assert pf.min() >= 0 and pf.max() < L
    # eq. 46 keeps the hard spheres apart: whatever overlap a step creates is a small fraction of a bead radius
    from scipy.spatial import cKDTree
    d, _ = cKDTree(pf, boxsize=L).query(pf[w.N_bead:], k=2)
    assert d[:, 1].min() > 2 * w.a - 0.2 * w.a
    # warm start from the previous step: fewer iterations than the cold first solve
    assert np.mean(its[1:]) < its[0]
    for step in frames:
        p, qg, Phig, psig, fg, Fg, Tg, xn = kept[step]
        qo, Phio, _ = orc.solve_induced(p, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a, w.eps_f)
        oo = orc.forces_torques(p, w.body_offset, qo, w.E0, w.L, w.a, w.eps_f, Phi_body=Phio)
        r = {"q": rel(qg, qo), "psi": rel(psig, oo["psi"]), "f": rel(fg, oo["f"]),
             "Phi": float(np.abs(Phig - Phio).max() / np.abs(oo["psi"]).max()),
             "F": body_vector_error(Fg, oo["F"], oo["f"])[0], "T": body_vector_error(Tg, oo["T"], oo["f"])[0]}
        assert r["q"] < 1e-9 and r["psi"] < 1e-9 and r["Phi"] < 1e-9, (step, r)
        assert r["f"] < 1e-8 and r["F"] < 1e-8 and r["T"] < 1e-8, (step, r)
        # the step itself, from the same positions and the same (device) forces, with the oracle's own Philox stream
        xo = ody.bd_step(p, w.body_offset, fg, w.L, w.a, dt, 1.0, 1.0, ody.normals(seed, step, w.N_ion))
        e = xn - xo
        e -= L * np.round(e / L)
        assert np.abs(e).max() < 1e-12 * L, (step, np.abs(e).max())
