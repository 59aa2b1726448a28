"""Config 3 as BASELINE.json states it: charged colloid (2562 beads, Q = -100 e) + 20 100 ions, 100 Brownian-dynamics
steps with dt = 1e-4 and Gaussian noise from the seed.  The trajectory is generated once (forces from the CUDA path,
update by the harness workloads/dynamics.py); at frames 0, 50 and 99 the CUDA path is compared with the oracle on the
IDENTICAL positions (trajectory-level parity is meaningless for chaotic dynamics)."""
import copy

import numpy as np
import pytest

import oracle as orc
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
    noise = wl.dynamics.noise_for(wl.configs.BASE_SEED + 3, n_steps, w.N_ion)
    ctx = pce.context_for(w)
    x, y, z, Q, qi = pce.upload(w)
    ctx.set_system(w.body_offset, x, y, z)
    pos = w.x.copy()
    q_prev, its_warm, kept = None, [], {}
    for step in range(n_steps):
        if step:
            xt = torch.from_numpy(np.ascontiguousarray(pos.T)).cuda()
            ctx.set_positions(xt[0].contiguous(), xt[1].contiguous(), xt[2].contiguous())
        q, Phi, info = ctx.solve(Q, qi, w.E0, q0=q_prev)
        assert info["converged"], (step, info)
        out = ctx.forces(q, w.E0)
        its_warm.append(info["iters"])
        q_prev = q
        if step in frames:
            kept[step] = (pos.copy(), q.cpu().numpy(), Phi.cpu().numpy(), out["psi"].cpu().numpy(), out["f"].cpu().numpy(),
                          out["F"].cpu().numpy(), out["T"].cpu().numpy())
        f_ion = out["f"][w.N_bead:].cpu().numpy()
        pos[w.N_bead:] = wl.dynamics.bd_step(pos[w.N_bead:], f_ion, noise[step], dt, float(w.L[0]), w.a, np.full(3, w.L[0] / 2), 1.0)
    ctx.close()
    # the harness kept the hard-sphere constraints, and the ions moved
    d = pos[w.N_bead:] - w.L[0] / 2
    assert np.linalg.norm(d, axis=1).min() >= 1.0 + 2 * w.a - 1e-9
    assert np.abs(pos[w.N_bead:] - w.x[w.N_bead:]).max() > 10 * np.sqrt(2 * dt)
    # warm start from the previous step: fewer iterations than the cold first solve
    assert np.mean(its_warm[1:]) < its_warm[0]
    for step in frames:
        p, qg, Phig, psig, fg, Fg, Tg = kept[step]
        wf = copy.copy(w)
        wf.x = p
        qo, Phio, _ = orc.solve_induced(p, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a, w.eps_f)
        oo = orc.forces_torques(p, w.body_offset, qo, w.E0, w.L, w.a, w.eps_f, Phi_body=Phio)
        r = {"q": rel(qg, qo), "psi": rel(psig, oo["psi"]), "f": rel(fg, oo["f"]),
             "Phi": float(np.abs(Phig - Phio).max() / np.abs(oo["psi"]).max()),
             "F": body_vector_error(Fg, oo["F"], oo["f"])[0], "T": body_vector_error(Tg, oo["T"], oo["f"])[0]}
        assert r["q"] < 1e-9 and r["psi"] < 1e-9 and r["Phi"] < 1e-9, (step, r)
        assert r["f"] < 1e-8 and r["F"] < 1e-8 and r["T"] < 1e-8, (step, r)
