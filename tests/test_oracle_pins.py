"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-type the oracle's formula or re-call its routine: each checks
it against a quadrature of the defining integral, a textbook routine written
here from scratch, a closed form, an invariant or brute force (SURVEY.md 8(c)
C.3, P1-P12).  CPU only.
"""
import os

import mpmath as mp
import numpy as np
import pytest
from scipy import integrate, special

import oracle as orc
import workloads as wl
from workloads import geometry as geo
from conftest import read_golden


# ---------------------------------------------------------------- P1: eq. 10
@pytest.mark.parametrize("r_over_a", [0.0, 0.3, 1.0, 1.7, 2.0, 2.6, 4.0])
def test_eq10_is_shell_shell_average(r_over_a):
    """eq. 10 (reading G1) = potential of a unit shell of radius a
    averaged over a second shell of radius a at centre distance r."""
    a = 0.37
    r = r_over_a * a

    def pot(mu):  # Newton: shell potential at distance s from its centre
        s = np.sqrt(a * a + r * r - 2 * a * r * mu)
        return 1.0 / (4 * np.pi * max(s, a))

    pts = [r / (2 * a)] if 0 < r < 2 * a else None
    val, _ = integrate.quad(pot, -1, 1, points=pts, epsabs=1e-14, epsrel=1e-13)
    assert orc.M_free(r, a) == pytest.approx(0.5 * val, rel=1e-11)


def test_eq10_limits():
    a = 0.2
    assert orc.M_free(0.0, a) == pytest.approx(1 / (4 * np.pi * a), rel=1e-15)
    assert orc.M_free(2 * a, a) == pytest.approx(1 / (8 * np.pi * a), rel=1e-15)
    assert orc.M_free(5.0, a) == pytest.approx(1 / (4 * np.pi * 5.0), rel=1e-15)  # Coulomb
    h = 1e-7  # C^1 at r = 2a
    dl = (orc.M_free(2 * a, a) - orc.M_free(2 * a - h, a)) / h
    dr = (orc.M_free(2 * a + h, a) - orc.M_free(2 * a, a)) / h
    assert dl == pytest.approx(dr, rel=1e-5)


# ---------------------------------------------------------------- P2: eq. 20 / 21
def _R_fourier(r, a, xi):
    """Radial inverse Fourier transform of (1-h) j0^2/k^2 (eq. 19 line 2)."""
    mp.mp.dps = 30
    r, a, xi = mp.mpf(r), mp.mpf(a), mp.mpf(xi)

    def piece(u, c):
        if u == 0:
            return mp.mpf(0)
        f = lambda k: c * mp.sin(k * u) * (1 - mp.exp(-k * k / (4 * xi * xi))) / (k ** 3 * a * a)
        return mp.quadosc(f, [0, mp.inf], omega=abs(u))

    # sin(kr) sin^2(ka) = sin(kr)/2 - sin(k(r+2a))/4 - sin(k(r-2a))/4
    tot = piece(r, mp.mpf(1) / 2) + piece(r + 2 * a, -mp.mpf(1) / 4) + piece(r - 2 * a, -mp.mpf(1) / 4)
    return float(tot / (2 * mp.pi ** 2 * r))


@pytest.mark.parametrize("r,a,xi", [(1.2, 1.0, 0.7), (0.4, 0.5, 1.3), (2.0, 1.0, 0.7), (3.1, 0.7, 0.9)])
def test_eq20_is_fourier_integral(r, a, xi):
    assert orc.R(r, a, xi) == pytest.approx(_R_fourier(r, a, xi), rel=1e-12, abs=1e-16)


def _W_quad(r, a, xi):
    """Wave-space kernel in real space: 1/(2 pi^2 r) int sin(kr)/k h(k) j0(ka)^2 dk
    (eq. 19 line 1 for one pair in free space) -- exponentially convergent."""
    f = lambda k: np.sin(k * r) / k * np.exp(-k * k / (4 * xi * xi)) * np.sinc(k * a / np.pi) ** 2
    kmax = 2 * xi * 6.5
    val, _ = integrate.quad(f, 0, kmax, epsabs=1e-15, epsrel=1e-13, limit=400)
    return val / (2 * np.pi ** 2 * r)


@pytest.mark.parametrize("a,xi", [(1.0, 0.7), (0.2, 1.0), (0.0346, 1.04), (0.5, 3.0)])
def test_eq20_plus_wave_kernel_is_eq10(a, xi):
    """R(r) + W(r) = M_free(r) for all r (eq. 19 = eq. 9), incl. r < 2a and across 2a."""
    for r in np.array([0.05, 0.5, 1.0, 1.9, 2.0, 2.1, 3.0, 6.0, 12.0]) * a:
        lhs = orc.R(r, a, xi) + _W_quad(r, a, xi)
        assert lhs == pytest.approx(orc.M_free(r, a), rel=2e-11, abs=1e-14), (r, a, xi)


@pytest.mark.parametrize("a,xi", [(1.0, 0.7), (0.2, 1.0), (0.0346, 1.04)])
def test_eq21_self_term(a, xi):
    """R(0) = M_free(0) - W(0), W(0) = 1/(2 pi^2) int h j0^2 dk; and R(r->0) -> R(0)."""
    f = lambda k: np.exp(-k * k / (4 * xi * xi)) * np.sinc(k * a / np.pi) ** 2
    val, _ = integrate.quad(f, 0, 2 * xi * 6.5, epsabs=1e-15, epsrel=1e-13, limit=400)
    assert orc.R0(a, xi) == pytest.approx(1 / (4 * np.pi * a) - val / (2 * np.pi ** 2), rel=1e-12)
    assert orc.R(1e-4 * a, a, xi) == pytest.approx(orc.R0(a, xi) - 1e-4 * a / (16 * np.pi * a * a), rel=1e-7)  # + O(r^2)
    assert orc.R(1e-9 * a, a, xi) == pytest.approx(orc.R0(a, xi), rel=1e-8)


def test_eq22_point_limit_and_xi_limits():
    """a -> 0 gives erfc(xi r)/(4 pi r) (eq. 22); xi -> inf gives 0;
    xi -> 0 gives eq. 10."""
    r, xi = 0.8, 1.1
    assert orc.R(r, 1e-4, xi) == pytest.approx(special.erfc(xi * r) / (4 * np.pi * r), rel=1e-7)
    # xi -> inf: (1-h) -> k^2/4xi^2, so R -> (shell-shell overlap density)/(4 xi^2)
    # = 1/(32 pi a^2 xi^2 r) inside 2a, and exponentially small outside
    assert orc.R(0.3, 0.5, 60.0) == pytest.approx(1 / (32 * np.pi * 0.25 * 3600 * 0.3), rel=1e-3)
    assert abs(orc.R(1.3, 0.5, 60.0)) < 1e-12
    # xi -> 0: W -> 1/(2 pi^2) int exp(-k^2/4xi^2) dk = xi/(2 pi^1.5), so R -> eq. 10 - xi/(2 pi^1.5)
    for rr in (0.3, 2.3):
        assert orc.R(rr, 0.5, 1e-3) == pytest.approx(orc.M_free(rr, 0.5) - 1e-3 / (2 * np.pi ** 1.5), abs=1e-9)


@pytest.mark.parametrize("a,xi", [(1.0, 0.7), (0.0346, 1.04)])
def test_dR_matches_finite_difference(a, xi):
    for r in np.array([0.3, 1.0, 1.9, 2.1, 3.0, 8.0, 20.0]) * a:
        h = 1e-4 * a
        # Richardson-extrapolated central difference
        d1 = (orc.R(r + h, a, xi) - orc.R(r - h, a, xi)) / (2 * h)
        d2 = (orc.R(r + 2 * h, a, xi) - orc.R(r - 2 * h, a, xi)) / (4 * h)
        fd = (4 * d1 - d2) / 3
        assert orc.dR(r, a, xi) == pytest.approx(fd, rel=1e-8, abs=1e-12), r
    # a -> 0: derivative of eq. 22
    r = 0.9
    ex = -special.erfc(xi * r) / (4 * np.pi * r * r) - 2 * xi / np.sqrt(np.pi) * np.exp(-(xi * r) ** 2) / (4 * np.pi * r)
    assert orc.dR(r, 1e-4, xi) == pytest.approx(ex, rel=1e-6)


# ---------------------------------------------------------------- textbook point-charge Ewald (written here)
def _point_ewald_matrix(x, L, xi, s=6.0):
    """Textbook Ewald for unit point charges in a cubic box with the k = 0 term
    removed: sum_n erfc(xi r)/(4 pi r) + (1/V) sum_k exp(-k^2/4xi^2)/k^2 cos(k.r)
    - 1/(4 xi^2 V); diagonal: images n != 0, minus the self term xi/(2 pi^1.5)."""
    N = len(x)
    V = L ** 3
    rc, kmax = s / xi, 2 * s * xi
    m = int(np.ceil(rc / L))
    shifts = np.array([[i, j, k] for i in range(-m, m + 1) for j in range(-m, m + 1) for k in range(-m, m + 1)]) * L
    km = int(np.floor(kmax * L / (2 * np.pi)))
    kk = np.array([[i, j, k] for i in range(-km, km + 1) for j in range(-km, km + 1) for k in range(-km, km + 1)
                   if (i, j, k) != (0, 0, 0)]) * 2 * np.pi / L
    k2 = (kk * kk).sum(1)
    kk, k2 = kk[k2 <= kmax ** 2], k2[k2 <= kmax ** 2]
    gk = np.exp(-k2 / (4 * xi * xi)) / k2
    M = np.zeros((N, N))
    for i in range(N):
        for j in range(N):
            d = x[i] - x[j]
            d -= L * np.round(d / L)
            rr = np.linalg.norm(d + shifts, axis=1)
            rr = rr[(rr > 0) & (rr < rc)]
            real = (special.erfc(xi * rr) / (4 * np.pi * rr)).sum()
            wave = (gk * np.cos(kk @ d)).sum() / V
            M[i, j] = real + wave - 1 / (4 * xi * xi * V)
            if i == j:
                M[i, j] -= xi / (2 * np.pi ** 1.5)
    return M


def test_shell_vs_point_ewald_offset():
    """P5: if every pair and every image is >= 2a apart, M - M_point =
    a^2/(3V) off the diagonal and 1/(4 pi a) + a^2/(3V) on it."""
    rng = np.random.default_rng(3)
    L, a = 5.0, 0.2
    x = wl.geometry.place_ions(rng, 7, L, 2 * a + 0.05, lambda p: np.ones(len(p), bool))
    M = orc.pair_matrix(x, L, a)
    Mp = _point_ewald_matrix(x, L, xi=1.7)
    D = M - Mp
    V = L ** 3
    off = D[~np.eye(7, dtype=bool)]
    assert np.allclose(off, a * a / (3 * V), rtol=0, atol=2e-13)
    assert np.allclose(np.diag(D), 1 / (4 * np.pi * a) + a * a / (3 * V), rtol=0, atol=2e-13)


def test_madelung_nacl(golden_dir):
    """P6: 8-ion rock-salt cell, d = 1, a = 0.4."""
    alpha = read_golden(os.path.join(golden_dir, "madelung_nacl.txt"))["alpha"]
    pts = np.array([[i, j, k] for i in range(2) for j in range(2) for k in range(2)], dtype=float)
    q = np.array([(-1.0) ** int(p.sum()) for p in pts])
    a = 0.4
    psi = orc.ewald_eval(pts, q, 2.0, a, field=False)
    U = 0.5 * q @ psi - (q * q).sum() / (8 * np.pi * a)
    assert -U * 4 * np.pi / 4 == pytest.approx(alpha, rel=1e-12)
    # and through the dense pair function (different xi, different code path)
    M = orc.pair_matrix(pts, 2.0, a)
    U2 = 0.5 * q @ M @ q - (q * q).sum() / (8 * np.pi * a)
    assert -U2 * 4 * np.pi / 4 == pytest.approx(alpha, rel=1e-12)


def test_bruteforce_image_sum():
    """P7: eq. 10 summed over whole image cells (no Ewald machinery) for a
    neutral, inversion-symmetric set with one overlapping pair; potential
    differences converge to the oracle's as the image shell count grows."""
    L, a = 4.0, 0.3
    c = np.full(3, L / 2)
    base = np.array([[0.7, 0.2, -0.4], [0.85, 0.45, -0.3], [-0.3, 1.1, 0.9]])  # first two overlap (r < 2a)
    x = np.concatenate([c + base, c - base])
    q = np.array([1.0, -0.6, -0.4, 1.0, -0.6, -0.4])
    assert np.linalg.norm(base[0] - base[1]) < 2 * a
    psi = orc.ewald_eval(x, q, L, a, field=False)
    ref = psi - psi[0]

    def brute(Rmax):
        n = np.arange(-Rmax, Rmax + 1)
        sh = np.array(np.meshgrid(n, n, n, indexing="ij")).reshape(3, -1).T * L
        out = np.zeros(len(x))
        for i in range(len(x)):
            for j in range(len(x)):
                rr = np.linalg.norm(x[i] - x[j] + sh, axis=1)
                out[i] += q[j] * np.where(rr >= 2 * a, 1 / (4 * np.pi * np.maximum(rr, 1e-300)),
                                          (4 * a - rr) / (16 * np.pi * a * a)).sum()
        return out - out[0]

    e8 = np.linalg.norm(brute(8) - ref) / np.linalg.norm(ref)
    e16 = np.linalg.norm(brute(16) - ref) / np.linalg.norm(ref)
    assert e8 < 2e-4 and e16 < 3e-5 and e16 < e8 / 3


# ---------------------------------------------------------------- P3 / P4: operator invariants
def test_xi_independence_and_symmetry():
    w = wl.tiny_random(seed=11, n_body=2, n_ion=8, L=5.0, a=0.18, overlap_pair=True, neutral=False)
    q = np.random.default_rng(5).normal(size=w.N)  # NOT neutral: exercises the k=0 constant (reading A1)
    xi0 = orc.default_xi(w.L)
    p1, E1 = orc.ewald_eval(w.x, q, w.L, w.a, xi=xi0)
    p2, E2 = orc.ewald_eval(w.x, q, w.L, w.a, xi=1.5 * xi0)
    p3, E3 = orc.ewald_eval(w.x, q, w.L, w.a, xi=0.45 * xi0)  # r_c > L: image loop
    for p, E in ((p2, E2), (p3, E3)):
        assert np.linalg.norm(p - p1) / np.linalg.norm(p1) < 1e-13
        assert np.linalg.norm(E - E1) / np.linalg.norm(E1) < 1e-13
    M = orc.pair_matrix(w.x, w.L, w.a)
    assert np.abs(M - M.T).max() == 0.0
    assert np.linalg.norm(M @ q - p1) / np.linalg.norm(p1) < 1e-13
    np.linalg.cholesky(M)  # positive definite
    y = np.random.default_rng(6).normal(size=w.N)
    py = orc.ewald_eval(w.x, y, w.L, w.a, field=False)
    assert q @ py == pytest.approx(y @ p1, rel=1e-12)


def test_field_is_minus_gradient_of_potential():
    """E_alpha = -grad_alpha sum_beta M_ab q_b with q fixed (the beta = alpha term has no gradient)."""
    w = wl.tiny_random(seed=4, n_body=1, n_ion=5, L=4.0, a=0.15, overlap_pair=True)
    q = np.random.default_rng(2).normal(size=w.N)
    _, E = orc.ewald_eval(w.x, q, w.L, w.a)
    h = 1e-5
    for al in (0, w.N - 1, w.N - 4):
        for d in range(3):
            xp, xm = w.x.copy(), w.x.copy()
            xp[al, d] += h
            xm[al, d] -= h
            fd = -(orc.ewald_eval(xp, q, w.L, w.a, targets=[al], field=False)[0]
                   - orc.ewald_eval(xm, q, w.L, w.a, targets=[al], field=False)[0]) / (2 * h)
            assert E[al, d] == pytest.approx(fd, rel=1e-7, abs=1e-9)


# ---------------------------------------------------------------- P8: solve invariants
def test_solve_invariants_dense_vs_cg():
    w = wl.tiny_random(seed=21, n_body=3, n_ion=10, L=6.0, a=0.2)
    q, Phi, info = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a, method="dense")
    off = w.body_offset
    for i in range(w.N_body):
        assert q[off[i]:off[i + 1]].sum() == pytest.approx(w.Q_body[i], abs=1e-13)
    psi = orc.ewald_eval(w.x, q, w.L, w.a, field=False)
    r = orc.rel_positions(w.x, off, w.L)
    resid = psi[:w.N_bead] - r @ w.E0
    for i in range(w.N_body):
        seg = resid[off[i]:off[i + 1]]
        assert np.ptp(seg) < 1e-12 * max(1.0, np.abs(psi).max())  # equipotential, eq. 12
        assert seg.mean() == pytest.approx(Phi[i], abs=1e-12)
    assert info["kkt_residual"] < 1e-13
    q2, Phi2, info2 = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a, method="cg")
    assert np.linalg.norm(q2 - q) / np.linalg.norm(q) < 1e-11
    assert np.linalg.norm(Phi2 - Phi) / np.linalg.norm(Phi) < 1e-11


# ---------------------------------------------------------------- P9: conducting sphere
def test_conducting_sphere_dipole(golden_dir):
    g = read_golden(os.path.join(golden_dir, "paper_sphere_dipole.txt"))
    errs = {}
    for sub in (1, 2, 3):
        w = wl.config1(subdiv=sub, L=10.0)
        q, Phi, _ = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
        r = orc.rel_positions(w.x, w.body_offset, w.L)
        S = (r * q[:, None]).sum(0)
        assert abs(S[0]) < 1e-12 and abs(S[1]) < 1e-12
        errs[w.N] = S[2] / g["coef"] - 1.0
    # always larger than the exact dipole, decreasing ~ N^-1/2
    assert errs[42] > errs[162] > errs[642] > 0
    slope = np.log(errs[642] / errs[42]) / np.log(642 / 42)
    assert -0.65 < slope < -0.45
    at1000 = errs[642] * (642 / 1000.0) ** 0.5
    assert 0.03 < at1000 < 0.08  # "about ~5% for N ~ 1000"
    assert abs(at1000 - g["err_at_1000"]) < 0.03


# ---------------------------------------------------------------- P10 / P11: forces and torques
def _W_resolved(x, w):
    q, Phi, _ = orc.solve_induced(x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
    return orc.forces_torques(x, w.body_offset, q, w.E0, w.L, w.a, Phi_body=Phi)


def test_forces_torques_are_minus_gradient_of_W():
    """eq. 17/18 vs central differences of the re-solved constrained energy W
    (reading A8) under rigid translation / rotation of a body and ion moves."""
    w = wl.tiny_random(seed=33, n_body=2, n_ion=5, L=6.0, a=0.2)
    out = _W_resolved(w.x, w)
    off = w.body_offset
    h = 1e-5
    X = out["X"]
    # translation of body 0
    for d in range(3):
        xp, xm = w.x.copy(), w.x.copy()
        xp[off[0]:off[1], d] += h
        xm[off[0]:off[1], d] -= h
        fd = -(_W_resolved(xp, w)["W"] - _W_resolved(xm, w)["W"]) / (2 * h)
        assert out["F"][0, d] == pytest.approx(fd, rel=2e-7, abs=1e-9)
    # rotation of body 1 about its centre, axis z and x
    for axis in (np.array([0, 0, 1.0]), np.array([1.0, 0, 0])):
        def rot(th):
            K = np.array([[0, -axis[2], axis[1]], [axis[2], 0, -axis[0]], [-axis[1], axis[0], 0]])
            Rm = np.eye(3) + np.sin(th) * K + (1 - np.cos(th)) * K @ K
            xx = w.x.copy()
            rb = out["r"][off[1]:off[2]]
            xx[off[1]:off[2]] = X[1] + rb @ Rm.T
            return xx
        fd = -(_W_resolved(rot(h), w)["W"] - _W_resolved(rot(-h), w)["W"]) / (2 * h)
        assert out["T"][1] @ axis == pytest.approx(fd, rel=2e-7, abs=1e-9)
    # an ion
    al = w.N - 2
    for d in range(3):
        xp, xm = w.x.copy(), w.x.copy()
        xp[al, d] += h
        xm[al, d] -= h
        fd = -(_W_resolved(xp, w)["W"] - _W_resolved(xm, w)["W"]) / (2 * h)
        assert out["f"][al, d] == pytest.approx(fd, rel=2e-7, abs=1e-9)


def test_net_force_and_isolated_torque():
    w = wl.tiny_random(seed=12, n_body=2, n_ion=7, L=6.0, a=0.2, neutral=True)
    out = _W_resolved(w.x, w)
    tot_q = w.Q_body.sum() + w.q_ion.sum()
    assert np.abs(out["f"].sum(0) - tot_q * w.E0).max() < 1e-13
    # energies: W = U_eq16 + 1/2 sum_i Q_i Psi_0,i  (reading A8), Psi_0 = -X.E0
    Psi0 = np.concatenate([-out["X"] @ w.E0, -(w.x[w.N_bead:] @ w.E0)])
    Qall = np.concatenate([w.Q_body, w.q_ion])
    assert out["W"] == pytest.approx(out["U_eq16"] + 0.5 * Qall @ Psi0, rel=1e-11, abs=1e-12)
    # single elongated body in a large box: torque ~ S x E0
    pts = geo.fibonacci_spheroid(40, 0.25, 1.0)
    a = geo.bead_radius(pts)
    Rm = geo.random_rotation(np.random.default_rng(1))
    L = 30.0
    x = pts @ Rm.T + L / 2
    E0 = np.array([0.3, 0.1, 1.0])
    qs, Phi, _ = orc.solve_induced(x, [0, 40], [0.0], [], E0, L, a)
    o = orc.forces_torques(x, [0, 40], qs, E0, L, a, Phi_body=Phi)
    SxE = np.cross(o["S"][0], E0)
    assert np.linalg.norm(o["T"][0] - SxE) / np.linalg.norm(SxE) < 2e-2
    assert np.linalg.norm(o["F"][0]) < 1e-12


# ---------------------------------------------------------------- P12: lattice symmetry
def test_cubic_lattice_symmetry():
    """Ion-free simple-cubic array: identical dipoles, no forces, no torques,
    equal body potentials (C_qE = C_SPsi = 0)."""
    w = wl.config4(subdiv=1, nside=2, spacing=3.0, n_ion=0, with_ions=False, Ng=32)
    q, Phi, _ = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
    o = orc.forces_torques(w.x, w.body_offset, q, w.E0, w.L, w.a, Phi_body=Phi)
    assert np.abs(o["S"] - o["S"][0]).max() < 1e-12
    assert np.abs(o["F"]).max() < 1e-12 and np.abs(o["T"]).max() < 1e-12
    assert np.ptp(Phi) < 1e-12
    # same dipole as one sphere alone in the primitive cell
    w1 = wl.config1(subdiv=1, L=3.0)
    w1.E0[:] = w.E0
    q1, Phi1, _ = orc.solve_induced(w1.x, w1.body_offset, w1.Q_body, w1.q_ion, w1.E0, w1.L, w1.a)
    S1 = (orc.rel_positions(w1.x, w1.body_offset, w1.L) * q1[:, None]).sum(0)
    assert np.abs(o["S"][0] - S1).max() < 1e-11


# ---------------------------------------------------------------- reading A7: a body across the periodic boundary
def test_body_centres_for_a_body_across_the_periodic_boundary():
    """X_i is the mean of the body's beads unwrapped about its first bead ("centre of mass", reading A7).
    Translating the whole periodic system by any vector must translate X_i (mod L) and leave r_ij, the induced charges,
    forces and torques unchanged -- also when the translation leaves the body straddling a face, an edge or a corner of
    the box, where a naive mean of wrapped coordinates is wrong by ~L/2."""
    w = wl.tiny_random(seed=31, n_body=2, n_ion=6, L=6.0, a=0.2)
    off, L = w.body_offset, w.L
    X0, r0 = orc.body_centres(w.x, off, L)
    q0, Phi0, _ = orc.solve_induced(w.x, off, w.Q_body, w.q_ion, w.E0, L, w.a)
    o0 = orc.forces_torques(w.x, off, q0, w.E0, L, w.a, Phi_body=Phi0)
    c = np.asarray(w.meta["centres"])[0]
    for shift in (np.array([0.03, 0.0, 0.0]) - [c[0], 0, 0],          # body 0 centred on the face x = 0
                  np.array([6.0 - 0.01, 0.02, 0.0]) - [c[0], c[1], 0],  # on the edge x = L, y = 0
                  np.array([0.01, 5.99, 0.02]) - c):                    # on a corner
        xs = w.x + shift
        xs -= L * np.floor(xs / L)
        b0 = xs[off[0]:off[1]]
        assert np.ptp(b0, axis=0).max() > 0.5 * L[0]  # the wrapped beads really sit on both sides of the box
        X, r = orc.body_centres(xs, off, L)
        assert np.abs(r - r0).max() < 1e-12
        dX = X - (X0 + shift)
        assert np.abs(dX - L * np.round(dX / L)).max() < 1e-12
        naive = b0.mean(axis=0)  # what a mean of wrapped coordinates would give: off by a fraction of L
        dn = naive - X[0]
        assert np.abs(dn - L * np.round(dn / L)).max() > 0.1
        q, Phi, _ = orc.solve_induced(xs, off, w.Q_body, w.q_ion, w.E0, L, w.a)
        o = orc.forces_torques(xs, off, q, w.E0, L, w.a, Phi_body=Phi)
        assert np.abs(q - q0).max() < 1e-11 * np.abs(q0).max()
        for k in ("F", "T", "S"):
            assert np.abs(o[k] - o0[k]).max() < 1e-10 * max(np.abs(o0["f"]).sum(0).max(), 1.0), k
        assert np.abs(Phi - Phi0).max() < 1e-11 * max(np.abs(Phi0).max(), 1.0)


def test_dR_small_r_branch():
    """dR/dr for r -> 0 (the oracle's r < 1e-6 a branch and its neighbourhood): R = M_free - W with W smooth and even in r,
    so dR/dr -> dM_free/dr = -1/(16 pi a^2) (eq. 10, reading G1), continuously through the branch point."""
    for a, xi in ((1.0, 0.7), (0.2, 1.3), (0.0346, 1.04)):
        lim = -1.0 / (16 * np.pi * a * a)
        for r in (1e-9 * a, 0.5e-6 * a, 0.99e-6 * a, 1.01e-6 * a, 2e-6 * a, 1e-5 * a):
            assert orc.dR(r, a, xi) == pytest.approx(lim, rel=2e-4), (a, xi, r)


# ---------------------------------------------------------------- grand capacitance tensor (eq. 15) and eps_eff (eq. 36-37)
def test_capacitance_tensor_symmetry_and_cubic_cell_couplings():
    """C = Sigma' M^-1 Sigma'^T is symmetric positive definite; for one sphere in a cubic periodic cell the couplings
    C_qE and C_SPsi vanish by symmetry and C_SE = (S / E0) I with S the dipole of the constrained solve of
    eq. 13 (an independent route: dense KKT system instead of M^-1)."""
    w = wl.config1(subdiv=1, L=6.0)
    C = orc.capacitance(w.x, w.body_offset, w.L, w.a)
    assert C.shape == (4, 4)
    assert np.abs(C - C.T).max() < 1e-12 * np.abs(C).max()
    assert np.linalg.eigvalsh(0.5 * (C + C.T)).min() > 0
    assert np.abs(C[0, 1:]).max() < 1e-11 and np.abs(C[1:, 0]).max() < 1e-11
    q, Phi, _ = orc.solve_induced(w.x, w.body_offset, [0.0], [], [0, 0, 1.0], w.L, w.a)
    S = (orc.rel_positions(w.x, w.body_offset, w.L) * q[:, None]).sum(0)
    assert np.abs(C[1:, 1:] - S[2] * np.eye(3)).max() < 1e-10 * S[2]
    eps = orc.effective_permittivity(C, 1, float(np.prod(w.L)))
    assert np.abs(eps - (1 + S[2] / np.prod(w.L)) * np.eye(3)).max() < 1e-12


def test_capacitance_of_a_sphere_in_a_periodic_cell_textbook_value():
    """C_qPsi of one conducting sphere of radius R in a cubic cell with neutralising background (k = 0 removed,
    PAPER.md:80): Psi/Q = 1/(4 pi R) - zeta/(4 pi L) + R^2/(6 V) + ..., zeta = 2.837297 the textbook Madelung constant
    of a simple-cubic lattice of point charges in a uniform background.  The bead model makes R an effective radius
    a little above 1: checked to 3 %."""
    w = wl.config1(subdiv=3, L=10.0)
    C = orc.capacitance(w.x, w.body_offset, w.L, w.a)
    L = 10.0
    inv_exact = 1 / (4 * np.pi) - 2.837297 / (4 * np.pi * L) + 1.0 / (6 * L ** 3)
    assert 1 / C[0, 0] == pytest.approx(inv_exact, rel=0.03)
    assert 1 / C[0, 0] < inv_exact  # a_eff > R: slightly larger capacitance


def test_effective_permittivity_matches_the_constrained_solves_and_dilute_limit():
    """eq. 36 from the blocks of C (Schur complement C_SE - C_SPsi C_qPsi^-1 C_qE) must equal the mean dipole of the
    constrained solves of eq. 13 with Q = 0 and unit fields, for bodies with no symmetry; and for a dilute cubic array it
    approaches the Clausius-Mossotti value 1 + 3 phi_eff / (1 - phi_eff)."""
    w = wl.tiny_random(seed=41, n_body=3, n_ion=0, L=7.0, a=0.2)
    nb, V = w.N_body, float(np.prod(w.L))
    C = orc.capacitance(w.x, w.body_offset, w.L, w.a)
    eps = orc.effective_permittivity(C, nb, V)
    ref = np.eye(3)
    for d in range(3):
        E0 = np.eye(3)[d]
        q, Phi, _ = orc.solve_induced(w.x, w.body_offset, np.zeros(nb), [], E0, w.L, w.a)
        o = orc.forces_torques(w.x, w.body_offset, q, E0, w.L, w.a, Phi_body=Phi)
        ref[:, d] += o["S"].sum(0) / V
    assert np.abs(eps - ref).max() < 1e-10
    assert np.abs(eps - eps.T).max() < 1e-10
    # dilute simple-cubic array of spheres (one per cell)
    w1 = wl.config1(subdiv=2, L=8.0)
    C1 = orc.capacitance(w1.x, w1.body_offset, w1.L, w1.a)
    e1 = orc.effective_permittivity(C1, 1, 8.0 ** 3)
    phi_eff = (e1[2, 2] - 1) / (e1[2, 2] + 2)  # invert Clausius-Mossotti: phi = (eps - 1)/(eps + 2)
    phi_geo = 4 * np.pi / 3 / 8.0 ** 3
    assert 1.0 < phi_eff / phi_geo < 1.25  # effective radius a few per cent above the geometric one


def test_fiber_torque_follows_the_angle_law_of_an_axisymmetric_polarizable_body():
    """PAPER.md:348 (Fig. 4): for a slender body with polarizability alpha_par along its axis and alpha_perp across it the dipole
    is S = alpha_perp E0 + (alpha_par - alpha_perp)(n.E0) n, hence S.E0 = alpha_perp + (alpha_par - alpha_perp) cos^2 theta and
    |T| = |S x E0| = (alpha_par - alpha_perp) sin(2 theta) / 2: no torque at 0 and 90 degrees, maximum at 45, sense towards
    alignment.  Linear response of eq. 13 fixes these laws exactly for an isolated body; the periodic images of a large box
    perturb them at the 1e-2 level."""
    import workloads as wl
    res = {}
    for deg in (0, 30, 45, 60, 90):
        w = wl.fiber_in_field(chi=5, theta=np.deg2rad(deg), L=30.0)
        q, Phi, _ = orc.solve_induced(w.x, w.body_offset, w.Q_body, w.q_ion, w.E0, w.L, w.a)
        o = orc.forces_torques(w.x, w.body_offset, q, w.E0, w.L, w.a, Phi_body=Phi)
        res[deg] = (o["S"][0], o["T"][0], o["F"][0])
    a_par, a_perp = res[0][0][2], res[90][0][2]
    assert a_par > 3 * a_perp > 0                                  # a slender conductor polarizes along its axis
    tscale = 0.5 * (a_par - a_perp)
    for deg in (0, 90):
        assert np.abs(res[deg][1]).max() < 1e-9 * tscale            # symmetric positions: no torque
    for deg in (30, 45, 60):
        S, T, F = res[deg]
        th = np.deg2rad(deg)
        assert abs(S[2] - (a_perp + (a_par - a_perp) * np.cos(th) ** 2)) < 2e-2 * a_par
        assert abs(T[0]) < 1e-9 * tscale and abs(T[2]) < 1e-9 * tscale
        assert T[1] < 0                                             # the axis (sin th, 0, cos th) turns towards E0 = e_z
        assert abs(-T[1] - tscale * np.sin(2 * th)) < 3e-2 * tscale
        assert np.allclose(T, np.cross(S, w.E0), atol=3e-2 * tscale)  # isolated body: T = S x E0
        assert np.abs(F).max() < 1e-9 * tscale                      # no net force in a uniform field on a neutral body
    assert -res[45][1][1] > -res[30][1][1] and -res[45][1][1] > -res[60][1][1]
