"""Seeded input generators (workloads/): the synthetic states must have the structure DESIGN.md section 5 states."""
import numpy as np

import workloads as W


def _min_gap(x, R, box, periodic):
    from scipy.spatial import cKDTree
    xs = x.copy()
    bs = None
    if any(periodic):
        bs = np.array([box[a] if periodic[a] else 1e30 for a in range(3)])
        xs = xs - xs.min(0) * np.array(periodic)
        xs = np.mod(xs, bs)
    d, j = cKDTree(xs, boxsize=bs).query(xs, k=2)
    return (d[:, 1] - (R + R[j[:, 1]])).min()


def test_paper_bed_spheres_do_not_overlap_and_reach_the_fraction():
    for phi, expect in ((0.15, 2866), (0.30, 5731), (0.45, 8596)):
        lbm, cpl, pd, x, v, w, R = W.paper_bed(phi)
        assert abs(len(R) / expect - 1.0) < 0.03
        assert _min_gap(x, R, (500.0, 200.0, 800.0), (True, True, False)) > 0.0
        assert x[:, 2].min() - R[0] > -0.5 and x[:, 2].max() + R[0] < 799.5
        assert cpl["n_sub"] == 10 and lbm["collision"] == 1
    assert len(W.paper_bed(0.0)[6]) == 0
    # the packed variant bench.py times: columns of touching spheres, nothing overlaps by more than 0.5 % of a diameter
    for phi, expect in ((0.15, 2866), (0.45, 8596)):
        lbm, cpl, pd, x, v, w, R = W.paper_bed(phi, contacts=True)
        assert abs(len(R) / expect - 1.0) < 0.03
        gap = _min_gap(x, R, (500.0, 200.0, 800.0), (True, True, False))
        assert -0.1 < gap < 0.0
        assert x[:, 2].min() - R[0] > -0.6 and x[:, 2].max() + R[0] < 799.5


def test_config_generators_are_seeded_and_shaped():
    pd, x, v, w, R = W.cfg1_gas()
    assert len(R) == 2048 and np.array_equal(x, W.cfg1_gas()[1])
    # (spacing 1.02 d with +-0.05 d jitter: configs[0] starts with some overlapping neighbours, as specified)
    lbm, cpl, pd, x, v, w, R, u = W.cfg4_shear(seed=4, n=64, n_part=300, R=4.0)
    assert _min_gap(x, R, (64.0, 64.0, 64.0), (True, True, False)) > 0.0          # RSA: no overlap, periodic x y
    pd, x, v, w, R = W.cfg5_pour(n_side=20, n_part=8000)
    assert R.min() >= 0.8e-3 and R.max() <= 1.2e-3 and _min_gap(x, R, None, (False,) * 3) > 0.0
