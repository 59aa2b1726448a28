"""Generator self-checks: counts, neutrality, exclusions, and
the paper's printed sphere-to-bead radius ratios (pins geometry reading B1)."""
import os

import numpy as np
import pytest
from scipy.spatial import cKDTree

import workloads as wl
from workloads import geometry as geo
from conftest import read_golden


def test_icosphere_counts_and_paper_ratios(golden_dir):
    g = read_golden(os.path.join(golden_dir, "paper_bead_to_sphere_ratio.txt"))
    for sub, n in enumerate([12, 42, 162, 642, 2562]):
        m = geo.icosphere(sub)
        assert m.shape == (n, 3)
        assert np.allclose(np.linalg.norm(m, axis=1), 1.0, atol=1e-14)
    assert 1 / geo.bead_radius(geo.icosphere(3)) == pytest.approx(g["N642"], abs=0.05)
    assert 1 / geo.bead_radius(geo.icosphere(4)) == pytest.approx(g["N2562"], abs=0.1)
    assert 1 / geo.bead_radius(geo.icosphere(5)) == pytest.approx(g["N10242"], abs=0.1)


def _check(w, min_center_dist=None):
    assert w.x.shape == (w.N, 3) and (w.x >= 0).all() and (w.x < w.L).all()
    assert w.body_offset[0] == 0 and w.body_offset[-1] == w.N_bead
    assert abs(w.Q_body.sum() + w.q_ion.sum()) < 1e-9  # neutral box
    if w.N_ion:
        ions = w.x[w.N_bead:]
        d, _ = cKDTree(ions, boxsize=w.L).query(ions, k=2)
        assert d[:, 1].min() >= 2 * w.a * (1 - 1e-12)
        db, _ = cKDTree(w.x[:w.N_bead], boxsize=w.L).query(ions, k=1)
        assert db.min() >= 2 * w.a * (1 - 1e-12)  # no ion overlaps a bead


def test_configs_1_to_4_self_checks():
    w1 = wl.config1()
    assert (w1.N, w1.N_body) == (162, 1) and w1.a == pytest.approx(0.137952, abs=1e-6)
    _check(w1)
    w2 = wl.config2(d=2.2)
    assert (w2.N_bead, w2.N_ion) == (1284, 1000)
    _check(w2)
    w3 = wl.config3()
    assert (w3.N_bead, w3.N_ion) == (2562, 20100)
    assert w3.Q_body[0] == pytest.approx(-100 * w3.meta["e"])
    _check(w3)
    w4 = wl.config4(n_ion=2000)
    assert w4.N_bead == 41088 and w4.N_body == 64
    _check(w4)
    # seeded: same call, same bits
    assert np.array_equal(wl.config2(d=2.2).x, w2.x)


def test_config5_replica_self_checks():
    w = wl.config5_replica()
    assert (w.N_body, w.N_bead, w.N_ion) == (8, 8000, 16000)
    _check(w)
    # no bead pair of different bodies closer than 2a
    xb = w.x[:w.N_bead]
    pairs = cKDTree(xb, boxsize=w.L).query_pairs(2 * w.a * (1 - 1e-9), output_type="ndarray")
    assert (pairs[:, 0] // 1000 == pairs[:, 1] // 1000).all()
    # equal-area template: nearest-neighbour spacing is narrow
    t = geo.fibonacci_spheroid(1000)
    d, _ = cKDTree(t).query(t, k=2)
    assert d[:, 1].max() / d[:, 1].min() < 1.6


def test_fiber_generator():
    """Four touching bead lines: 8 chi beads, nearest neighbours exactly 2a apart, length / width = chi."""
    import numpy as np
    from scipy.spatial import cKDTree
    import workloads as wl
    from workloads import geometry as geo
    for chi in (5, 10):
        m = geo.fiber(chi, a=0.3)
        assert m.shape == (8 * chi, 3) and np.allclose(m.mean(axis=0), 0)
        d, _ = cKDTree(m).query(m, k=2)
        assert np.allclose(d[:, 1], 0.6)
        ext = m.max(axis=0) - m.min(axis=0) + 0.6
        assert np.isclose(ext[2] / ext[0], chi) and np.isclose(ext[0], ext[1])
    w = wl.fiber_in_field(chi=5, theta=np.pi / 3)
    X = w.x[:w.N_bead].mean(axis=0)
    axis = w.x[w.N_bead // 4 - 1] - w.x[0]  # first line, first to last bead
    axis /= np.linalg.norm(axis)
    assert np.allclose(X, w.L / 2) and np.isclose(axis @ w.E0, np.cos(np.pi / 3))
    wi = wl.fiber_in_field(chi=5, n_ion=50)
    assert wi.N_ion == 50 and abs(wi.q_ion.sum()) < 1e-12
    dmin, _ = cKDTree(wi.x[:wi.N_bead]).query(wi.x[wi.N_bead:], k=1)
    assert dmin.min() >= 2.5 * wi.a


def test_fcc_array_generator():
    """FCC arrays of the paper's timing workload: 4 m^3 spheres, 12 nearest neighbours at a / sqrt 2 of the
    conventional cell, the requested volume fraction, no overlaps."""
    import numpy as np
    from scipy.spatial import cKDTree
    import workloads as wl
    w = wl.fcc_array(2, subdiv=2, phi=0.3)
    assert w.N_body == 32 and w.N_bead == 32 * 162 and w.N_ion == 0
    c = w.meta["centres"]
    L = float(w.L[0])
    assert np.isclose(w.N_body * 4.0 / 3.0 * np.pi / L ** 3, 0.3)
    pairs = cKDTree(c, boxsize=L).query_pairs((L / 2) / np.sqrt(2) * 1.001, output_type="ndarray")
    assert len(pairs) == 32 * 12 // 2                      # every site has 12 nearest neighbours
    d = c[pairs[:, 0]] - c[pairs[:, 1]]
    d -= L * np.round(d / L)
    assert np.allclose(np.linalg.norm(d, axis=1), (L / 2) / np.sqrt(2)) and (L / 2) / np.sqrt(2) > 2 + 2 * w.a
    assert w.Ng[0] & (w.Ng[0] - 1) == 0 and L / w.Ng[0] <= 2.3 * w.a
