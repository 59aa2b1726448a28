"""Seeded geometry generators shared by the oracle tests, the GPU tests and bench.py.

This module holds NO arithmetic of the method (no kernels, no Ewald
parameters, no solver): only point sets.  numpy + scipy.spatial only.
"""
from __future__ import annotations

import numpy as np
from scipy.spatial import cKDTree

GOLDEN_ANGLE = np.pi * (3.0 - np.sqrt(5.0))


def icosphere(subdiv: int) -> np.ndarray:
    """Bead centres on the unit sphere: the 12 icosahedron vertices, then
    ``subdiv`` rounds of edge bisection with radial projection.
    Returns (10*4**subdiv + 2, 3)."""
    t = (1.0 + np.sqrt(5.0)) / 2.0
    v = np.array(
        [[-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0],
         [0, -1, t], [0, 1, t], [0, -1, -t], [0, 1, -t],
         [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1]], dtype=np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array(
        [[0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
         [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
         [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
         [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1]], dtype=np.int64)
    verts = [tuple(p) for p in v]
    for _ in range(subdiv):
        cache = {}
        newf = []

        def mid(i, j):
            key = (min(i, j), max(i, j))
            if key not in cache:
                p = (np.array(verts[i]) + np.array(verts[j])) / 2.0
                p /= np.linalg.norm(p)
                verts.append(tuple(p))
                cache[key] = len(verts) - 1
            return cache[key]

        for a, b, c in f:
            ab, bc, ca = mid(a, b), mid(b, c), mid(c, a)
            newf += [[a, ab, ca], [b, bc, ab], [c, ca, bc], [ab, bc, ca]]
        f = np.array(newf, dtype=np.int64)
    return np.array(verts, dtype=np.float64)


def min_spacing(pts: np.ndarray) -> float:
    """Smallest nearest-neighbour distance of a point set."""
    d, _ = cKDTree(pts).query(pts, k=2)
    return float(d[:, 1].min())


def bead_radius(pts: np.ndarray) -> float:
    """Beads 'as large as possible without overlapping':
    a = half the smallest bead-bead spacing."""
    return 0.5 * min_spacing(pts)


def fibonacci_spheroid(n: int, b: float = 1.0, c: float = 4.0) -> np.ndarray:
    """n points on the prolate spheroid (b, b, c), equal area per point along
    the axis and golden-angle azimuths (DESIGN.md input recipe, config 5)."""
    zz = np.linspace(-c, c, 400001)
    rho = b * np.sqrt(np.clip(1.0 - (zz / c) ** 2, 0.0, None))
    # dA = 2 pi rho sqrt(1 + rho'^2) dz with rho rho' = -b^2 z / c^2
    integrand = 2.0 * np.pi * np.sqrt(rho ** 2 + (b * b * zz / (c * c)) ** 2)
    area = np.concatenate([[0.0], np.cumsum(0.5 * (integrand[1:] + integrand[:-1]) * np.diff(zz))])
    frac = (np.arange(n) + 0.5) / n
    z = np.interp(frac * area[-1], area, zz)
    r = b * np.sqrt(np.clip(1.0 - (z / c) ** 2, 0.0, None))
    phi = GOLDEN_ANGLE * np.arange(n)
    return np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=1)


def random_rotation(rng: np.random.Generator) -> np.ndarray:
    """Uniform rotation on SO(3) from a seeded unit quaternion."""
    q = rng.normal(size=4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def place_ions(rng, n, L, min_sep, keep_mask_fn, oversample=1.3, max_rounds=50):
    """n points uniform in the periodic box [0,L)^3, pairwise >= min_sep apart,
    all satisfying keep_mask_fn(points) (vectorised exclusion of the bodies)."""
    L = np.broadcast_to(np.asarray(L, dtype=np.float64), (3,))
    acc = np.zeros((0, 3))
    for _ in range(max_rounds):
        need = n - acc.shape[0]
        if need <= 0:
            break
        cand = rng.uniform(0.0, 1.0, size=(int(need * oversample) + 16, 3)) * L
        cand = cand[keep_mask_fn(cand)]
        if cand.shape[0] == 0:
            continue
        if min_sep > 0:
            # drop candidates too close to accepted points
            if acc.shape[0]:
                d, _ = cKDTree(acc, boxsize=L).query(cand, k=1, distance_upper_bound=min_sep)
                cand = cand[~np.isfinite(d)]
            # drop the later member of every close pair among the candidates
            if cand.shape[0] > 1:
                pairs = cKDTree(cand, boxsize=L).query_pairs(min_sep, output_type="ndarray")
                bad = np.zeros(cand.shape[0], dtype=bool)
                if pairs.size:
                    bad[pairs[:, 1]] = True
                cand = cand[~bad]
        acc = np.concatenate([acc, cand[:need]])
    if acc.shape[0] < n:
        raise RuntimeError("ion placement did not converge")
    return acc[:n]


def fiber(chi: int, a: float = 1.0) -> np.ndarray:
    """The paper's "fiber": four parallel lines of touching beads of radius a, the lines through the corners of a
    square of side 2a (neighbouring lines touch), 2 chi beads per line at spacing 2a along z -- length 4 a chi over width 4a,
    i.e. ratio of the longest to the shortest axis chi (reading B8).  Centred at the origin; (8 chi, 3)."""
    n = 2 * int(chi)
    z = (np.arange(n) - 0.5 * (n - 1)) * 2.0 * a
    pts = [np.stack([np.full(n, sx * a), np.full(n, sy * a), z], axis=1) for sx in (-1.0, 1.0) for sy in (-1.0, 1.0)]
    return np.concatenate(pts)
