"""Pins of the Brownian-dynamics oracle (oracle/dynamics.py; eqs. 40-49, 62) against what the paper and the
mathematics fix: the generator's published known-answer vectors, the moments of the normal deviates, the defining property of
the potential-free hard-sphere step (overlapping pairs end in contact), brute force for the neighbour search,
rigid-body kinematics in closed form, the Einstein relation of free diffusion, and counting identities of the observables."""
import os

import numpy as np

import oracle as orc
from oracle import dynamics as dy


def test_philox_known_answers(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "philox4x32_10_kat.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for row in rows:
        v = [int(t, 16) for t in row]
        out = dy.philox4x32(np.array(v[0:4], dtype=np.uint32), np.array(v[4:6], dtype=np.uint32))
        assert [int(o) for o in out] == v[6:10]
    # vectorised form = element-wise form
    ctr = np.arange(40, dtype=np.uint32).reshape(10, 4)
    key = np.arange(20, dtype=np.uint32).reshape(10, 2) * np.uint32(2654435761)
    many = dy.philox4x32(ctr, key)
    for i in range(10):
        assert (many[i] == dy.philox4x32(ctr[i], key[i])).all()


def test_normals_have_the_moments_of_a_standard_normal_and_distinct_streams():
    n = 400_000
    z = dy.normals(seed=20240107, step=3, n=n)
    assert z.shape == (n, 3)
    se = 1.0 / np.sqrt(n)
    assert np.all(np.abs(z.mean(axis=0)) < 5 * se)
    assert np.all(np.abs(z.var(axis=0) - 1.0) < 5 * np.sqrt(2.0) * se)
    assert np.all(np.abs((z ** 3).mean(axis=0)) < 5 * np.sqrt(15.0) * se)
    assert np.all(np.abs((z ** 4).mean(axis=0) - 3.0) < 5 * np.sqrt(96.0) * se)
    c = np.corrcoef(z.T)
    assert np.abs(c - np.eye(3)).max() < 5 * se
    # P(|z| < 1) of the normal law (erf(1/sqrt 2) = 0.682689...)
    assert np.all(np.abs((np.abs(z) < 1).mean(axis=0) - 0.6826894921370859) < 5 * 0.4654 * se)
    # another step or another seed gives another, uncorrelated stream; the same (seed, step) the same one
    z2, z3 = dy.normals(20240107, 4, n), dy.normals(20240108, 3, n)
    assert abs(np.corrcoef(z[:, 0], z2[:, 0])[0, 1]) < 5 * se and abs(np.corrcoef(z[:, 0], z3[:, 0])[0, 1]) < 5 * se
    assert (dy.normals(20240107, 3, 100) == z[:100]).all()


def test_overlapping_pair_ends_in_contact_after_one_step():
    """"separating them to contact at the end of the time step" -- eq. 46 with eqs. 42-44."""
    a, dt, gamma, L = 0.3, 1e-3, 2.5, 10.0
    for r0 in (0.2 * a, a, 1.9 * a):
        d = np.array([1.0, 2.0, -2.0]) / 3.0
        x = np.array([[0.05, 5.0, 9.9], [0.05, 5.0, 9.9]]) + np.outer([0.5, -0.5], r0 * d)
        xn = dy.bd_step(x, [0], np.zeros((2, 3)), L, a, dt, gamma, 1.0, np.zeros((2, 3)), brute=True)
        dn = xn[0] - xn[1]
        dn -= L * np.round(dn / L)
        assert abs(np.linalg.norm(dn) - 2 * a) < 1e-13
        assert np.allclose(dn / np.linalg.norm(dn), d, atol=1e-12)     # along the line of centres
        mid = x.mean(axis=0)
        mn = xn[1] + 0.5 * dn
        assert np.allclose((mn - mid) - L * np.round((mn - mid) / L), 0, atol=1e-13)  # the pair's centre does not move
    # at or beyond contact: no force
    x = np.array([[1.0, 1.0, 1.0], [1.0 + 2 * a, 1.0, 1.0]])
    assert (dy.hard_sphere_forces(x, [0], L, a, gamma, dt, brute=True) == 0).all()


def test_hard_sphere_neighbour_search_matches_the_double_loop_and_skips_own_body():
    rng = np.random.default_rng(5)
    L, a = np.array([3.0, 3.5, 4.0]), 0.25
    x = rng.uniform(0, 1, (150, 3)) * L
    off = np.array([0, 30, 50])
    f1 = dy.hard_sphere_forces(x, off, L, a, 1.3, 1e-3)
    f2 = dy.hard_sphere_forces(x, off, L, a, 1.3, 1e-3, brute=True)
    assert np.abs(f2).max() > 0 and np.allclose(f1, f2, rtol=1e-13, atol=1e-13 * np.abs(f2).max())
    assert np.allclose(f1.sum(axis=0), 0, atol=1e-9 * np.abs(f1).max())          # Newton's third law
    # beads of one body never push each other: a body alone feels nothing
    assert (dy.hard_sphere_forces(x[:30], np.array([0, 30]), L, a, 1.3, 1e-3, brute=True) == 0).all()


def test_rigid_body_step_closed_forms():
    """Free-draining rigid motion (eq. 62; reading A16): a ring of n beads of radius R in the plane z = const under a pure
    torque T e_z turns by T dt / (gamma n R^2); under a pure force it translates by F dt / (n gamma); distances are kept."""
    n, R, gamma, dt, L, a = 12, 1.5, 0.7, 0.05, 20.0, 0.05
    ph = 2 * np.pi * np.arange(n) / n
    ring = np.stack([R * np.cos(ph), R * np.sin(ph), np.zeros(n)], axis=1) + np.array([19.5, 10.0, 0.2])  # across the boundary
    xw = ring - L * np.floor(ring / L)
    tz = 3.0
    f = (tz / (n * R)) * np.stack([-np.sin(ph), np.cos(ph), np.zeros(n)], axis=1)   # tangential forces: torque tz, no net force
    xn = dy.bd_step(xw, [0, n], f, L, a, dt, gamma, 1.0, np.zeros((0, 3)), move_bodies=True)
    X0, r0 = orc.body_centres(xw, [0, n], L)
    X1, r1 = orc.body_centres(xn, [0, n], L)
    assert np.allclose(X1, X0, atol=1e-13)
    ang = tz * dt / (gamma * n * R * R)
    c, s = np.cos(ang), np.sin(ang)
    assert np.allclose(r1, r0 @ np.array([[c, -s, 0], [s, c, 0], [0, 0, 1]]).T, atol=1e-13)
    # pure force
    F = np.array([0.3, -0.2, 0.9])
    xn = dy.bd_step(xw, [0, n], np.tile(F / n, (n, 1)), L, a, dt, gamma, 1.0, np.zeros((0, 3)), move_bodies=True)
    X1, r1 = orc.body_centres(xn, [0, n], L)
    assert np.allclose(X1 - X0, F * dt / (n * gamma), atol=1e-13) and np.allclose(r1, r0, atol=1e-13)
    # general force field on a random body: rigid to rounding, and the angular velocity satisfies I Omega = L
    rng = np.random.default_rng(11)
    body = rng.normal(size=(40, 3)) + 7.0
    f = rng.normal(size=(40, 3))
    xn = dy.bd_step(body, [0, 40], f, L, a, dt, gamma, 1.0, np.zeros((0, 3)), move_bodies=True)
    d0 = np.linalg.norm(body[:, None] - body[None], axis=2)
    d1 = np.linalg.norm(xn[:, None] - xn[None], axis=2)
    assert np.abs(d1 - d0).max() < 1e-13
    _, r = orc.body_centres(body, [0, 40], L)
    _, rn = orc.body_centres(xn, [0, 40], L)
    T = np.cross(r, f).sum(axis=0)
    I = gamma * ((r * r).sum() * np.eye(3) - r.T @ r)
    Om = np.linalg.solve(I, T)
    # first order in dt the bead displacement is (U + Omega x r) dt (eq. 62)
    U = f.sum(axis=0) / (40 * gamma)
    lin = (U + np.cross(Om, r)) * dt
    assert np.abs((xn - body) - lin).max() < 2 * (np.linalg.norm(Om) * dt) ** 2 * np.abs(r).max()
    # bodies held fixed (reading A13) when move_bodies is off; a single bead does not rotate
    assert (dy.bd_step(body, [0, 40], f, L, a, dt, gamma, 1.0, np.zeros((0, 3))) == body).all()


def test_free_ions_obey_the_einstein_relation():
    """No forces: <|dx|^2> = 6 (kT / gamma) dt per step (eq. 41 with eq. 43); a constant force adds the drift f dt / gamma."""
    n, dt, gamma, kT, L, a = 200_000, 2e-3, 1.7, 0.8, 1e6, 1e-9
    rng = np.random.default_rng(2)
    x = rng.uniform(0.25, 0.75, (n, 3)) * L
    f = np.tile([0.5, 0.0, -1.0], (n, 1))
    xn = dy.bd_step(x, [0], f, L, a, dt, gamma, kT, dy.normals(9, 0, n))
    dx = xn - x
    drift = f[0] * dt / gamma
    se = np.sqrt(2 * kT * dt / gamma / n)
    assert np.all(np.abs(dx.mean(axis=0) - drift) < 5 * se)
    msd = ((dx - drift) ** 2).sum(axis=1).mean()
    assert abs(msd / (6 * kT * dt / gamma) - 1) < 5 * np.sqrt(2.0 / (3 * n))


def test_radial_profile_counting_identities():
    rng = np.random.default_rng(3)
    L, a, n = 30.0, 0.5, 60_000
    x = rng.uniform(0, L, (n, 3))
    q = np.where(np.arange(n) % 2 == 0, 0.7, -0.7)
    centre = np.array([1.0, 29.0, 15.0])  # near a corner: minimum image matters
    r_lo, nb = 2.0, 220                   # shells out to 2 + 220 * 0.05 = 13 < L/2
    o = dy.radial_profile(x, q, centre, L, a, r_lo, nb, Q=-3.0)
    d = x - centre
    d -= L * np.round(d / L)
    r = np.linalg.norm(d, axis=1)
    # shell counts add up to the number of ions inside the outer radius
    assert o["counts"].sum() == np.count_nonzero((r >= r_lo) & (r < r_lo + nb * 0.1 * a))
    # uniform ions: g -> 1 within counting noise (eq. 49)
    outer = slice(100, None)
    n_exp = (n / 2) / L ** 3 * 4 * np.pi * o["r_mid"][outer] ** 2 * 0.1 * a
    zscore = (o["counts"][outer, 0] - n_exp) / np.sqrt(n_exp)
    assert abs(zscore.mean()) < 5 / np.sqrt(len(n_exp)) and abs(zscore.std() - 1) < 0.25
    assert abs(o["g"][outer].mean() - 1) < 0.02
    # eq. 48: the windowed density integrates to the enclosed charge; every ion at least a window half-width inside
    # [r_lo, r_k] is counted with weight (number of window centres within a of it) * dr / 2a = 1 exactly
    k = 180
    rk = r_lo + (k + 1) * 0.1 * a
    inside = (r >= r_lo + a) & (r < rk - a)
    edge = ((r >= r_lo - a) & (r < r_lo + a)) | ((r >= rk - a) & (r < rk + a))
    assert abs(o["Qcum"][k] - (-3.0) - q[inside].sum()) <= np.abs(q[edge]).sum() + 1e-9
    # a point charge well inside the range contributes exactly its charge to the plateau
    o1 = dy.radial_profile(centre[None] + np.array([[5.0123, 0, 0]]), np.array([1.3]), centre, L, a, r_lo, nb)
    assert abs(o1["Qcum"][-1] - 1.3) < 1e-12 and o1["counts"].sum() == 1
