"""Thin Brownian-dynamics harness for config 3: ions move by Euler-Maruyama steps of the overdamped
Langevin equation (eqs. 42-44) with the potential-free hard-sphere displacement of eq. 46; the colloid is held fixed
(SURVEY.md reading A13).  Test/bench infrastructure only: none of the electrostatics is computed here -- forces come in
as an argument (from the CUDA path), positions go out, and the oracle is then evaluated on those identical positions."""
from __future__ import annotations

import numpy as np
from scipy.spatial import cKDTree


def noise_for(seed: int, n_steps: int, n_ion: int) -> np.ndarray:
    """Standard normal increments of the whole run, drawn once from the seed: shape (n_steps, n_ion, 3)."""
    return np.random.default_rng(seed).normal(size=(n_steps, n_ion, 3))


def bd_step(x_ion, f_ion, noise, dt, L, a, centre, r_colloid, gamma=1.0, kT=1.0, sweeps=4):
    """x += (f/gamma) dt + sqrt(2 kT dt/gamma) N(0,1)  (eqs. 42-44), then the hard-sphere displacements of the
    potential-free algorithm (eq. 46: overlapping pairs are moved apart to contact, half the overlap each; ions are moved
    radially out of the colloid's excluded shell r_colloid + 2a), then the periodic wrap."""
    x = x_ion + (f_ion / gamma) * dt + np.sqrt(2.0 * kT * dt / gamma) * noise
    x -= L * np.floor(x / L)
    for _ in range(sweeps):
        moved = False
        d = x - centre
        d -= L * np.round(d / L)
        r = np.linalg.norm(d, axis=1)
        inside = r < r_colloid + 2 * a
        if inside.any():
            x[inside] += d[inside] * ((r_colloid + 2 * a - r[inside]) / r[inside])[:, None]
            moved = True
        x -= L * np.floor(x / L)
        x[x >= L] -= L
        pairs = cKDTree(x, boxsize=L).query_pairs(2 * a, output_type="ndarray")
        if len(pairs):
            dij = x[pairs[:, 0]] - x[pairs[:, 1]]
            dij -= L * np.round(dij / L)
            rij = np.linalg.norm(dij, axis=1)
            ok = rij > 0
            shift = 0.5 * (2 * a - rij[ok])[:, None] * dij[ok] / rij[ok][:, None]
            np.add.at(x, pairs[ok, 0], shift)
            np.add.at(x, pairs[ok, 1], -shift)
            moved = True
        x -= L * np.floor(x / L)
        x[x >= L] -= L
        if not moved:
            break
    return x
