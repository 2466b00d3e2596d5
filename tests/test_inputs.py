"""Pins for the seeded input generators (paper_2003_01833_b200/inputs.py): no GPU needed."""
import json
import os

import numpy as np

from paper_2003_01833_b200 import inputs as I

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))


def test_fejer_weights_sum_and_exactness():
    # the (p+1)-point Fejer rule is exact for degree-p polynomials.
    for n in (2, 3, 4, 5, 6, 9):
        x, w = I.fejer1(n)
        assert abs(w.sum() - 2.0) < 1e-14
        assert np.all(w > 0)
        for deg in range(n):                      # degree <= p = n-1
            exact = 0.0 if deg % 2 else 2.0 / (deg + 1)
            assert abs((w * x ** deg).sum() - exact) < 1e-14, (n, deg)
    # ... and the first even degree above p is NOT exact (so the rule is the p-th order one)
    x, w = I.fejer1(4)
    assert abs((w * x ** 4).sum() - 0.4) > 1e-2
    # PAPER.md:158 Eq. (15): points lie strictly inside the cell, never on a vertex
    assert np.all(np.abs(x) < 1.0)
    np.testing.assert_allclose(np.sort(x), np.cos((2 * np.arange(4)[::-1] + 1) * np.pi / 8), atol=1e-15)


def test_paper_mesh_sizes_obey_points_per_cell_rule():
    # N_m = (p+1)^3 N_c -- the paper's own tables obey it
    for key in ("mesh_sizes_p4", "mesh_sizes_p3"):
        for nm in GOLD[key]["values"]:
            assert nm % GOLD[key]["points_per_cell"] == 0


def test_uniform_mesh_config0():
    c = I.config0()
    assert c.N == 32768 and c.meta["cells"] == 512
    assert abs(c.w.sum() - 16.0 ** 3) < 1e-9           # weights sum to the domain volume
    assert c.N == 64 * c.meta["cells"]
    # quadrature integrates a cubic exactly over the domain
    val = (c.w * (1.0 + c.x ** 3 + c.y ** 2 * c.z + c.x * c.y * c.z)).sum()
    assert abs(val - 4096.0) < 1e-8
    # points never coincide with the nucleus
    assert np.sqrt(c.x ** 2 + c.y ** 2 + c.z ** 2).min() > 0.1
    # int psi^2 ~ 1 (coarse mesh: 0.991)
    assert abs((c.w * c.meta["psi"] ** 2).sum() - 1.0) < 2e-2


def test_adaptive_rule_counts_and_volume():
    cells = I.adaptive_cells(20.0, [(0.0, 0.0, 0.0)])
    assert cells[0].shape[0] == 6056                   # 387,584 points
    assert abs((cells[3] ** 3).sum() - 40.0 ** 3) < 1e-6   # cells tile the domain
    # rule holds for every kept cell, and fails for every parent
    d = np.sqrt(cells[0] ** 2 + cells[1] ** 2 + cells[2] ** 2)
    assert np.all(cells[3] <= 0.35 * np.maximum(d, 0.05))
    x, y, z, w = I.mesh_from_cells(cells, 4)
    assert x.shape[0] == 387584
    assert abs(w.sum() - 64000.0) < 1e-6
    assert len(np.unique(np.stack([x, y, z]), axis=1).T) == x.shape[0]   # all points distinct


def test_config1_fields_are_finite_and_seeded():
    a, b = I.config1(), I.config1()
    assert a.n_orb == 2 and a.f.shape == (2, a.N)
    assert np.all(np.isfinite(a.f))
    np.testing.assert_array_equal(a.f, b.f)
    np.testing.assert_allclose(a.k, np.sqrt(2 * np.array([3.86, 0.21])))


def test_random_cloud_is_deterministic():
    a, b = I.random_cloud(1000, 3, seed=7), I.random_cloud(1000, 3, seed=7)
    np.testing.assert_array_equal(a.x, b.x)
    np.testing.assert_array_equal(a.f, b.f)
    assert a.coords().shape == (3, 1000)
