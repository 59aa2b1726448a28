"""CPU oracle of the Brownian-dynamics step and of the double-layer observables (eqs. 40-49, eq. 62).

TEST INFRASTRUCTURE ONLY (see pce_oracle.c).  Plain numpy, written out in the paper's order; shares nothing with the CUDA
path.  The counter-based generator (Philox-4x32-10, Salmon et al. 2011, a published algorithm) is implemented here on its
own; the CUDA path has its own implementation of the same generator, so both draw identical noise from (seed, step, index).

Readings:
  A15  the hard-sphere interaction is eq. 46 taken literally as a pair potential evaluated at x(t): two particles
       of different bodies at distance r < 2a repel with |f| = gamma (2a - r) / (2 dt) along their line of centres, so that in
       the absence of anything else one step of eqs. 42-44 puts them back in contact.  Beads of one rigid body
       do not interact.
  A16  rigid bodies (eq. 62): free-draining -- every bead carries the Stokes drag gamma of eq. 43 and there are no
       hydrodynamic interactions -- so eq. 61 reduces to U = F / (N_i gamma) and Omega = I_gamma^-1 L with
       I_gamma = gamma sum_j (|r_j|^2 I - r_j r_j^T).  The beads move with u = U + Omega x r held constant over the step, i.e.
       r_j is turned by the rotation exp([Omega dt]_x) (Rodrigues' formula), which keeps the body rigid to rounding.  Bodies
       receive no Brownian displacement (colloids >> ions); with move_bodies = False they are held fixed (reading A13).
  A17  Q'(r), eq. 48: radial charge density by a sliding window of width 2a on a grid of step 0.1 a,
       integrated by the rectangle rule from the colloid surface.
"""
from __future__ import annotations

import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = np.uint64(0x9E3779B9)
_W1 = np.uint64(0xBB67AE85)
_MASK = np.uint64(0xFFFFFFFF)


def philox4x32(counter, key, rounds=10):
    """Philox-4x32 (Salmon, Moraes, Dror, Shaw, SC'11): counter (..., 4) uint32, key (..., 2) uint32 -> (..., 4) uint32.
    One round: (hi0, lo0) = M0 * c0, (hi1, lo1) = M1 * c2; c <- (hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0); the key is bumped by
    the Weyl constants between rounds."""
    c = np.asarray(counter, dtype=np.uint64)
    k = np.asarray(key, dtype=np.uint64)
    c0, c1, c2, c3 = (c[..., i].copy() for i in range(4))
    k0, k1 = k[..., 0].copy(), k[..., 1].copy()
    for r in range(rounds):
        if r:
            k0 = (k0 + _W0) & _MASK
            k1 = (k1 + _W1) & _MASK
        p0 = _M0 * c0
        p1 = _M1 * c2
        hi0, lo0 = p0 >> np.uint64(32), p0 & _MASK
        hi1, lo1 = p1 >> np.uint64(32), p1 & _MASK
        c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
    return np.stack([c0, c1, c2, c3], axis=-1).astype(np.uint32)


def normals(seed: int, step: int, n: int):
    """Three standard normal deviates per particle index i = 0..n-1 for time step `step`: counter (i, step, 0, 0), key
    (seed low word, seed high word); uniforms u_k = (r_k + 1/2) 2^-32 in (0, 1); Box-Muller:
    (sqrt(-2 ln u0) cos 2 pi u1, sqrt(-2 ln u0) sin 2 pi u1, sqrt(-2 ln u2) cos 2 pi u3).  Returns (n, 3)."""
    ctr = np.zeros((n, 4), dtype=np.uint32)
    ctr[:, 0] = np.arange(n, dtype=np.uint32)
    ctr[:, 1] = np.uint32(step & 0xFFFFFFFF)
    key = np.array([seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF], dtype=np.uint32)
    r = philox4x32(ctr, np.broadcast_to(key, (n, 2))).astype(np.float64)
    u = (r + 0.5) * 2.0 ** -32
    r0, r2 = np.sqrt(-2.0 * np.log(u[:, 0])), np.sqrt(-2.0 * np.log(u[:, 2]))
    return np.stack([r0 * np.cos(2 * np.pi * u[:, 1]), r0 * np.sin(2 * np.pi * u[:, 1]), r2 * np.cos(2 * np.pi * u[:, 3])], axis=1)


def _body_of(body_offset, N):
    off = np.asarray(body_offset, dtype=np.int64)
    bid = np.arange(N, dtype=np.int64) - int(off[-1]) + (len(off) - 1)  # ions: one-bead bodies after the conductors
    bid[: off[-1]] = np.repeat(np.arange(len(off) - 1), np.diff(off))
    return bid


def hard_sphere_forces(x, body_offset, L, a, gamma, dt, brute=False):
    """f_hs of eq. 46 on every particle: sum over particles of other bodies within 2a (minimum image) of
    gamma (2a - r) / (2 dt) times the unit vector pointing away from the neighbour (reading A15).  brute=True: the plain
    double loop (the pin of the neighbour-search route)."""
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    L = np.broadcast_to(np.asarray(L, dtype=np.float64), (3,))
    bid = _body_of(body_offset, N)
    f = np.zeros((N, 3))
    if brute:
        pairs = [(i, j) for i in range(N) for j in range(i + 1, N)]
        pairs = np.array(pairs, dtype=np.int64).reshape(-1, 2)
    else:
        from scipy.spatial import cKDTree
        xw = x - L * np.floor(x / L)
        xw[xw >= L] = 0.0
        pairs = cKDTree(xw, boxsize=L).query_pairs(2 * a * (1 + 1e-12), output_type="ndarray").astype(np.int64)
    if len(pairs) == 0:
        return f
    i, j = pairs[:, 0], pairs[:, 1]
    d = x[i] - x[j]
    d -= L * np.round(d / L)
    r = np.linalg.norm(d, axis=1)
    ok = (r < 2 * a) & (r > 0) & (bid[i] != bid[j])
    i, j, d, r = i[ok], j[ok], d[ok], r[ok]
    fij = (gamma * (2 * a - r) / (2 * dt) / r)[:, None] * d
    np.add.at(f, i, fij)
    np.add.at(f, j, -fij)
    return f


def rotation(w):
    """exp([w]_x): rotation by |w| about w (Rodrigues)."""
    th = float(np.linalg.norm(w))
    K = np.array([[0, -w[2], w[1]], [w[2], 0, -w[0]], [-w[1], w[0], 0]], dtype=np.float64)
    if th < 1e-8:
        return np.eye(3) + K + 0.5 * K @ K
    return np.eye(3) + (np.sin(th) / th) * K + ((1 - np.cos(th)) / th ** 2) * K @ K


def bd_step(x, body_offset, f, L, a, dt, gamma, kT, noise, move_bodies=False, brute=False):
    """One Euler-Maruyama step of the overdamped Langevin equation (eqs. 40-44):
       ions:    x(t + dt) = x(t) + (f + f_hs) dt / gamma + sqrt(2 kT dt / gamma) N(0, 1)         (eqs. 41-44, 46)
       bodies:  F = sum_j (f + f_hs)_ij,  L = sum_j r_ij x (f + f_hs)_ij  (eq. 18 / eq. 60),
                U = F / (N_i gamma), Omega = I_gamma^-1 L, X += U dt, r_ij <- exp([Omega dt]_x) r_ij  (eq. 62, reading A16)
    x (N, 3): beads (bodies contiguous) then ions; f (N, 3): electrostatic bead / ion forces (eq. 17); noise (N_ion, 3).
    Returns the new positions wrapped into [0, L)."""
    from .oracle import body_centres
    x = np.asarray(x, dtype=np.float64)
    off = np.asarray(body_offset, dtype=np.int64)
    nb, nbead = len(off) - 1, int(off[-1])
    L = np.broadcast_to(np.asarray(L, dtype=np.float64), (3,))
    ft = np.asarray(f, dtype=np.float64) + hard_sphere_forces(x, off, L, a, gamma, dt, brute=brute)
    xn = x.copy()
    xn[nbead:] = x[nbead:] + ft[nbead:] * (dt / gamma) + np.sqrt(2.0 * kT * dt / gamma) * np.asarray(noise, dtype=np.float64)
    if move_bodies and nb:
        X, r = body_centres(x, off, L)
        for i in range(nb):
            sl = slice(off[i], off[i + 1])
            ri, fi = r[sl], ft[sl]
            F, T = fi.sum(axis=0), np.cross(ri, fi).sum(axis=0)
            U = F / ((off[i + 1] - off[i]) * gamma)
            I = gamma * ((ri * ri).sum() * np.eye(3) - ri.T @ ri)
            # a single bead or collinear beads have no (full) rotational resistance: no rotation
            if off[i + 1] - off[i] > 1 and np.linalg.det(I) > 1e-10 * (np.trace(I) / 3.0) ** 3:
                Om = np.linalg.solve(I, T)
            else:
                Om = np.zeros(3)
            xn[sl] = X[i] + U * dt + ri @ rotation(Om * dt).T
    xn -= L * np.floor(xn / L)
    xn[xn >= L] = 0.0
    return xn


def radial_profile(x_ion, q_ion, centre, L, a, r_lo, n_bins, Q=0.0):
    """Double-layer observables about a colloid centre.
    Shells k = 0..n_bins-1: [r_lo + k dr, r_lo + (k + 1) dr) with dr = 0.1 a.
      counts (n_bins, 2): cations / anions per shell ("shell summation");
      g (n_bins, 2): eq. 49 for colloid-(+) and colloid-(-) pairs: count / (n_species * shell volume), n_species = N_species / V;
      rho (n_bins,): radial charge density by the sliding window of width 2a centred on the shell midpoint (reading A17);
      Qcum (n_bins,): eq. 48, Q + sum_{j <= k} rho_j dr.
    """
    x_ion = np.asarray(x_ion, dtype=np.float64)
    q_ion = np.asarray(q_ion, dtype=np.float64)
    L = np.broadcast_to(np.asarray(L, dtype=np.float64), (3,))
    d = x_ion - np.asarray(centre, dtype=np.float64)
    d -= L * np.round(d / L)
    r = np.linalg.norm(d, axis=1)
    dr = 0.1 * a
    counts = np.zeros((n_bins, 2))
    rho = np.zeros(n_bins)
    for k in range(n_bins):
        lo, hi = r_lo + k * dr, r_lo + (k + 1) * dr
        sel = (r >= lo) & (r < hi)
        counts[k, 0] = np.count_nonzero(sel & (q_ion > 0))
        counts[k, 1] = np.count_nonzero(sel & (q_ion < 0))
        mid = 0.5 * (lo + hi)
        rho[k] = q_ion[np.abs(r - mid) < a].sum() / (2 * a)
    V = float(np.prod(L))
    shell = 4.0 * np.pi / 3.0 * ((r_lo + dr * np.arange(1, n_bins + 1)) ** 3 - (r_lo + dr * np.arange(n_bins)) ** 3)
    nsp = np.array([np.count_nonzero(q_ion > 0), np.count_nonzero(q_ion < 0)], dtype=np.float64) / V
    g = counts / np.maximum(nsp[None, :] * shell[:, None], 1e-300)
    return {"counts": counts, "g": g, "rho": rho, "Qcum": Q + np.cumsum(rho) * dr, "r_mid": r_lo + dr * (np.arange(n_bins) + 0.5)}
