"""The five BASELINE.json workloads (plus small stand-ins), seeded and synthetic.

Holds no arithmetic of the method: positions, charges, bodies, box, grid size
and the applied field only.  Ewald parameters are chosen by the library
(pce_suggest_params) on the GPU side and by the oracle on its own side.

Every generator returns a ``Workload``; recipe and readings (B1-B7) are in
DESIGN.md "Input recipe".  Length unit = sphere radius (configs 1-4) or
spheroid short semi-axis (config 5).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
from scipy.spatial import cKDTree

from . import geometry as geo

BASE_SEED = 20240104


@dataclass
class Workload:
    name: str
    x: np.ndarray            # (N, 3) float64, beads (bodies contiguous) then ions, wrapped into [0, L)
    body_offset: np.ndarray  # (N_body + 1,) int32
    Q_body: np.ndarray       # (N_body,) net body charges
    q_ion: np.ndarray        # (N - N_bead,)
    E0: np.ndarray           # (3,)
    L: np.ndarray            # (3,)
    Ng: np.ndarray           # (3,) int
    a: float                 # bead (= ion) radius, the shell "regularization width"
    eps_f: float = 1.0
    meta: dict = field(default_factory=dict)

    @property
    def N(self):
        return self.x.shape[0]

    @property
    def N_bead(self):
        return int(self.body_offset[-1])

    @property
    def N_body(self):
        return len(self.body_offset) - 1

    @property
    def N_ion(self):
        return self.N - self.N_bead


def _wrap(x, L):
    x = x - L * np.floor(x / L)
    x[x >= L] = 0.0  # guard the x == L rounding case
    return x


def _mk(name, beads, off, Q, ions, qion, E0, L, Ng, a, **meta):
    L = np.full(3, float(L)) if np.isscalar(L) else np.asarray(L, dtype=np.float64)
    Ng = np.full(3, int(Ng), dtype=np.int32) if np.isscalar(Ng) else np.asarray(Ng, dtype=np.int32)
    x = np.concatenate([beads, ions]) if len(ions) else beads.copy()
    return Workload(name, _wrap(x, L), np.asarray(off, dtype=np.int32), np.asarray(Q, dtype=np.float64),
                    np.asarray(qion, dtype=np.float64), np.asarray(E0, dtype=np.float64), L, Ng, float(a),
                    1.0, dict(meta))


def _outside_spheres(centres, radius, L):
    centres = np.atleast_2d(centres)

    def keep(p):
        ok = np.ones(p.shape[0], dtype=bool)
        for c in centres:
            d = p - c
            d -= L * np.round(d / L)
            ok &= (d * d).sum(axis=1) >= radius * radius
        return ok
    return keep


def config1(subdiv=2, L=10.0, Ng=32):
    """Single conducting sphere in E0 = (0,0,1)."""
    m = geo.icosphere(subdiv)
    a = geo.bead_radius(m)
    beads = m + L / 2
    return _mk("cfg1_single_sphere", beads, [0, len(m)], [0.0], np.zeros((0, 3)), [], [0, 0, 1.0], L, Ng, a,
               sphere_radius=1.0, subdiv=subdiv)


def config2(d=3.0, seed=BASE_SEED + 2, subdiv=3, n_ion=1000, L=20.0, Ng=64):
    """Two conducting spheres at centre separation d along E0 plus monovalent
    ions (readings B4)."""
    rng = np.random.default_rng(seed)
    m = geo.icosphere(subdiv)
    a = geo.bead_radius(m)
    Rot = geo.random_rotation(rng)
    c1 = np.array([L / 2, L / 2, L / 2 - d / 2])
    c2 = np.array([L / 2, L / 2, L / 2 + d / 2])
    beads = np.concatenate([m + c1, m @ Rot.T + c2])
    ions = geo.place_ions(rng, n_ion, L, 2 * a, _outside_spheres([c1, c2], 1.1, L))
    qion = np.concatenate([np.ones(n_ion // 2), -np.ones(n_ion - n_ion // 2)])
    n = len(m)
    return _mk(f"cfg2_two_spheres_d{d:g}", beads, [0, n, 2 * n], [0.0, 0.0], ions, qion, [0, 0, 1.0], L, Ng, a,
               separation=d, centres=np.stack([c1, c2]))


def config3(seed=BASE_SEED + 3, subdiv=4, n_counter=100, n_salt=10000, L=40.0, Ng=128, coupling=0.5):
    """Charged colloid (Q = -100 e) with explicit double layer
    (readings B5).  e = sqrt(8 pi coupling a), eq. 47."""
    rng = np.random.default_rng(seed)
    m = geo.icosphere(subdiv)
    a = geo.bead_radius(m)
    c = np.full(3, L / 2)
    e = float(np.sqrt(8 * np.pi * coupling * a))
    n_ion = n_counter + 2 * n_salt
    ions = geo.place_ions(rng, n_ion, L, 2 * a, _outside_spheres([c], 1.0 + 2 * a, L))
    qion = e * np.concatenate([np.ones(n_counter + n_salt), -np.ones(n_salt)])
    return _mk("cfg3_charged_colloid", m + c, [0, len(m)], [-n_counter * e], ions, qion, [0, 0, 0.0], L, Ng, a,
               e=e, centre=c)


def config4(seed=BASE_SEED + 4, subdiv=3, nside=4, spacing=4.0, n_ion=100000, Ng=256, with_ions=True):
    """Simple-cubic lattice of nside^3 conducting spheres plus +-1 ions
    (readings B6).  Same mesh orientation on every sphere."""
    rng = np.random.default_rng(seed)
    m = geo.icosphere(subdiv)
    a = geo.bead_radius(m)
    L = nside * spacing
    g = (np.arange(nside) + 0.5) * spacing
    centres = np.array([[cx, cy, cz] for cx in g for cy in g for cz in g])
    beads = np.concatenate([m + c for c in centres])
    off = np.arange(len(centres) + 1) * len(m)
    if with_ions and n_ion:
        tree = cKDTree(centres, boxsize=L)

        def keep(p):
            d, _ = tree.query(p, k=1)
            return d >= 1.0 + 2 * a
        ions = geo.place_ions(rng, n_ion, L, 2 * a, keep)
        qion = np.concatenate([np.ones(n_ion // 2), -np.ones(n_ion - n_ion // 2)])
    else:
        ions, qion = np.zeros((0, 3)), []
    return _mk("cfg4_sc_lattice", beads, off, np.zeros(len(centres)), ions, qion, [0, 0, 0.5], L, Ng, a,
               centres=centres)


def fcc_array(m=2, subdiv=3, phi=0.2, Ng=None, h_over_a=2.3):
    """FCC array of 4 m^3 ideally polarizable spheres (m conventional cells per dimension) in a uniform field, no ions: the
    shape of the paper's only timing workload (Fig. 3d; reading B9: the paper counts N_b = 8 ... 512 bodies, an FCC
    array in a periodic cube holds 4 m^3).  Sphere radius 1, volume fraction phi; mesh spacing at most h_over_a bead radii with N_g the next
    power of two."""
    mesh = geo.icosphere(subdiv)
    a = geo.bead_radius(mesh)
    cell = (4.0 * (4.0 / 3.0) * np.pi / phi) ** (1.0 / 3.0)   # 4 spheres per conventional cell
    L = m * cell
    basis = np.array([[0, 0, 0], [0, 0.5, 0.5], [0.5, 0, 0.5], [0.5, 0.5, 0]]) + 0.25
    centres = np.array([(np.array([i, j, k]) + b) * cell for i in range(m) for j in range(m) for k in range(m) for b in basis])
    beads = np.concatenate([mesh + c for c in centres])
    off = np.arange(len(centres) + 1) * len(mesh)
    if Ng is None:
        Ng = int(2 ** np.ceil(np.log2(L / (h_over_a * a))))
    return _mk(f"fcc_{len(centres)}x{len(mesh)}", beads, off, np.zeros(len(centres)), np.zeros((0, 3)), [], [0, 0, 1.0], L, Ng, a,
               centres=centres, phi=phi)


def config5(seed=BASE_SEED + 5, n_body=500, n_bead=1000, n_ion=1000000, phi=0.1, Ng=512, aspect=4.0):
    """n_body rigid prolate spheroids (1,1,aspect) at volume fraction phi with
    uniformly random orientations plus +-1 ions, E0 = (0.3,0,0)
    (PAPER.md:329-350 for the anisotropic-body/torque shape; readings B7)."""
    rng = np.random.default_rng(seed)
    b, c = 1.0, float(aspect)
    tmpl = geo.fibonacci_spheroid(n_bead, b, c)
    a = geo.bead_radius(tmpl)
    L = float((n_body * (4.0 / 3.0) * np.pi * b * b * c / phi) ** (1.0 / 3.0))
    centres, rots, trees = [], [], []
    beads = []
    rbound = c + a
    tries = 0
    while len(centres) < n_body:
        tries += 1
        if tries > 200000:
            raise RuntimeError("spheroid placement did not converge")
        X = rng.uniform(0, 1, size=3) * L
        Rm = geo.random_rotation(rng)
        pts = tmpl @ Rm.T
        ok = True
        for Xj, tj in zip(centres, trees):
            d = X - Xj
            d -= L * np.round(d / L)
            if d @ d >= (2 * rbound) ** 2:
                continue
            dist, _ = tj.query(pts + d, k=1, distance_upper_bound=2 * a)
            if np.isfinite(dist).any():
                ok = False
                break
        if ok:
            centres.append(X); rots.append(Rm); trees.append(cKDTree(pts)); beads.append(pts + X)
    centres = np.array(centres)
    beads = np.concatenate(beads)
    off = np.arange(n_body + 1) * n_bead
    ctree = cKDTree(centres, boxsize=L)
    btree = cKDTree(beads - L * np.floor(beads / L), boxsize=L)
    bx, cz = b + 2 * a, c + 2 * a

    def keep(p):
        ok = np.ones(p.shape[0], dtype=bool)
        ptree = cKDTree(p, boxsize=L)
        near = ctree.query_ball_tree(ptree, cz)
        for j, idx in enumerate(near):
            if not idx:
                continue
            idx = np.asarray(idx)
            d = p[idx] - centres[j]
            d -= L * np.round(d / L)
            u = d @ rots[j]  # body frame: u = R^T d
            inside = (u[:, 0] ** 2 + u[:, 1] ** 2) / bx ** 2 + u[:, 2] ** 2 / cz ** 2 < 1.0
            ok[idx[inside]] = False
        # the enlarged spheroid is not the parallel surface: also keep 2a from every bead centre
        dist, _ = btree.query(p, k=1, distance_upper_bound=2 * a)
        ok &= ~np.isfinite(dist)
        return ok

    if n_ion:
        ions = geo.place_ions(rng, n_ion, L, 2 * a, keep)
        qion = np.concatenate([np.ones(n_ion // 2), -np.ones(n_ion - n_ion // 2)])
    else:
        ions, qion = np.zeros((0, 3)), []
    return _mk(f"cfg5_spheroids_{n_body}x{n_bead}_{n_ion}ions", beads, off, np.zeros(n_body), ions, qion,
               [0.3, 0, 0], L, Ng, a, centres=centres, rotations=np.array(rots), phi=phi)


def config5_replica(seed=BASE_SEED + 6):
    """Density-matched scaled-down replica of config 5: 8 spheroids + 16 000
    ions, same h (grid 128^3)."""
    return config5(seed=seed, n_body=8, n_bead=1000, n_ion=16000, Ng=128)


def tiny_random(seed=7, n_body=2, n_bead_side=1, n_ion=6, L=6.0, Ng=32, a=0.2, neutral=True,
                overlap_pair=False):
    """Small irregular set for brute-force style checks: n_body icosahedra
    (12 beads, sphere radius 1.07 a/0.5257: neighbouring beads 2.14a apart, i.e.
    NOT at the r = 2a kink of the kernel, so finite differences stay valid) plus ions."""
    rng = np.random.default_rng(seed)
    m = geo.icosphere(0)
    R = 1.07 * a / geo.bead_radius(m)
    beads, off = [], [0]
    centres = []
    while len(centres) < n_body:
        c = rng.uniform(0, L, size=3)
        if all(np.linalg.norm((c - o) - L * np.round((c - o) / L)) > 2 * (R + a) for o in centres):
            centres.append(c)
            beads.append(R * m @ geo.random_rotation(rng).T + c)
            off.append(off[-1] + len(m))
    beads = np.concatenate(beads) if beads else np.zeros((0, 3))
    keep = _outside_spheres(np.array(centres), R + 2 * a, L) if centres else (lambda p: np.ones(len(p), bool))
    ions = geo.place_ions(rng, n_ion, L, 2 * a, keep) if n_ion else np.zeros((0, 3))
    if overlap_pair and n_ion >= 2:
        ions[1] = ions[0] + np.array([0.9 * a, 0.3 * a, -0.2 * a])
    qion = rng.uniform(0.5, 1.5, size=n_ion) * np.where(np.arange(n_ion) % 2 == 0, 1.0, -1.0)
    Q = rng.uniform(-1, 1, size=n_body)
    if neutral and n_ion:
        qion[-1] -= qion.sum() + Q.sum()
    return _mk("tiny_random", beads, off, Q, ions, qion, rng.normal(size=3), L, Ng, a, centres=np.array(centres))


def fiber_in_field(chi=5, theta=0.25 * np.pi, L=None, Ng=64, a=0.25, n_ion=0, seed=BASE_SEED + 7):
    """One rigid fiber of aspect ratio chi (four bead lines) at the box centre, its long axis in the (x, z) plane at
    angle theta to the applied field E0 = (0, 0, 1) (Fig. 4), optionally with ions around it."""
    rng = np.random.default_rng(seed)
    m = geo.fiber(chi, a)
    half = 2.0 * a * chi
    if L is None:
        L = 4.0 * half + 8.0 * a
    c, s = np.cos(theta), np.sin(theta)
    Rot = np.array([[c, 0.0, s], [0.0, 1.0, 0.0], [-s, 0.0, c]])  # about y: the axis e_z goes to (sin theta, 0, cos theta)
    centre = np.full(3, L / 2)
    beads = m @ Rot.T + centre
    if n_ion:
        from scipy.spatial import cKDTree
        tree = cKDTree(beads)

        def keep(p):
            d, _ = tree.query(p, k=1, distance_upper_bound=2.5 * a)
            return ~np.isfinite(d)
        ions = geo.place_ions(rng, n_ion, L, 2 * a, keep)
        qion = np.concatenate([np.ones(n_ion // 2), -np.ones(n_ion - n_ion // 2)])
    else:
        ions, qion = np.zeros((0, 3)), []
    return _mk(f"fiber_chi{chi}", beads, [0, len(m)], np.zeros(1), ions, qion, [0, 0, 1.0], L, Ng, a, theta=theta, chi=chi)


ALL = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}
