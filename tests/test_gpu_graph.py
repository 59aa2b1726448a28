"""The Krylov iteration as a replayed CUDA graph (krylov.cu): a context on a capturable stream replays one captured iteration;
a context on the legacy default stream cannot be captured and enqueues the same kernels one by one.  The captured iteration
names buffers and sizes that change with the positions (near-field CSR, hit / pair lists, grid dimensions) and, in the
deterministic mode, the partial-sum buffer that the first pce_forces after a solve reallocates -- so the sequence every
Brownian-dynamics step runs, solve -> forces -> new positions -> solve, is held here to the plain-launch path (itself held to
the oracle by tests/test_gpu_parity.py), with the bodies moved from far apart to nearly touching so that the near field doubles
and its arrays are reallocated between the two solves."""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


def _sequence(pce, torch, stream, det):
    far, near = wl.config2(d=8.0, n_ion=300), wl.config2(d=2.2, n_ion=300)
    assert far.N == near.N
    out = {}
    ctx = pce.context_for(far, stream=stream, deterministic=det)
    x, y, z, Q, qi = pce.upload(far)
    ctx.set_system(far.body_offset, x, y, z)
    out["nnz0"] = ctx.info()["nnz_near"]
    q, Phi, info = ctx.solve(Q, qi, far.E0)
    out["q1"], out["info1"] = q.clone(), info
    f = ctx.forces(q, far.E0)
    out["F1"] = f["F"].clone()
    x, y, z, Q, qi = pce.upload(near)
    ctx.set_positions(x, y, z)
    out["nnz1"] = ctx.info()["nnz_near"]
    q, Phi, info = ctx.solve(Q, qi, near.E0)
    out["q2"], out["info2"] = q.clone(), info
    f = ctx.forces(q, near.E0)
    out["F2"], out["T2"] = f["F"].clone(), f["T"].clone()
    q, Phi, info = ctx.solve(Q, qi, near.E0, q0=q)  # warm start straight after forces: converged at once, still consistent
    out["q3"], out["info3"] = q.clone(), info
    torch.cuda.synchronize()
    ctx.close()
    return out


@pytest.mark.parametrize("det", [False, True], ids=["atomics", "deterministic"])
def test_graph_replay_survives_forces_and_moved_bodies(det):
    import torch
    import paper_2401_04865_b200 as pce
    pce.build()
    plain = _sequence(pce, torch, None, det)           # legacy default stream: no capture
    s = torch.cuda.Stream()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        graph = _sequence(pce, torch, s, det)
    assert plain["info1"]["graph_replays"] == 0 and plain["info2"]["graph_replays"] == 0
    assert graph["info1"]["graph_replays"] > 0 and graph["info2"]["graph_replays"] > 0
    assert graph["nnz1"] > 1.5 * graph["nnz0"]         # beyond the 10 % head-room: csr_col / csr_val were reallocated
    for k in ("info1", "info2"):
        assert graph[k]["converged"] and plain[k]["converged"]
        assert abs(graph[k]["iters"] - plain[k]["iters"]) <= (0 if det else 1)
    for k in ("q1", "F1", "q2", "F2", "T2", "q3"):
        g, p = graph[k].cpu().numpy(), plain[k].cpu().numpy()
        if det:
            assert np.array_equal(g, p), k          # same kernels, same order: bit for bit
        elif k[0] == "q":
            assert np.linalg.norm(g - p) <= 1e-10 * np.linalg.norm(p), k
        elif k[0] == "F":                           # T2 is a 1e5-fold cancellation (nearly touching spheres): deterministic leg only
            assert np.linalg.norm(g - p) <= 1e-8 * np.linalg.norm(p), k
