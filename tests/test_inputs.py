"""The seeded input generator (gf_inputs): recipe checks.  It is data tooling shared by both sides, so it is tested on
its own: determinism, counter-based addressing, SU(3)-ness, and the statistics the recipe implies."""
import numpy as np

import gf_inputs as gi
from _util import dag, gauge_transform, to_c


def test_deterministic_and_addressable():
    dims = (4, 6, 4, 2)
    A = gi.make_links(dims, 0.4, 5)
    B = gi.make_links(dims, 0.4, 5)
    assert np.array_equal(A, B)
    sites = np.array([0, 3, 17, 95, 191])
    assert np.array_equal(gi.make_links(dims, 0.4, 5, sites=sites), A[sites])
    assert not np.array_equal(gi.make_links(dims, 0.4, 6), A)
    assert np.array_equal(gi.make_links(dims, 0.4, 5, dtype=np.float32), A.astype(np.float32))


def test_links_are_su3():
    dims = (4, 4, 4, 4)
    Uc = to_c(gi.make_links(dims, 0.6, 2))
    assert np.abs(Uc @ dag(Uc) - np.eye(3)).max() < 4e-15
    assert np.abs(np.linalg.det(Uc) - 1).max() < 4e-15
    G = gi.make_gauge(dims, 2)
    assert np.abs(G @ dag(G) - np.eye(3)).max() < 4e-15 and np.abs(np.linalg.det(G) - 1).max() < 4e-15


def test_recipe_statistics():
    # undoing the hidden gauge rotation leaves exp(i r H): <Re Tr>/3 = 1 - (8/3) r^2 + O(r^4)   (E Tr H^2 = 16)
    dims = (8, 8, 8, 8)
    r = 0.1
    Uc = to_c(gi.make_links(dims, r, 9))
    E = gauge_transform(Uc, dag(gi.make_gauge(dims, 9)), dims)
    m = np.trace(E, axis1=-2, axis2=-1).real.mean() / 3
    assert abs(m - (1 - 8 / 3 * r * r)) < 5e-4
    # Haar: <Tr G> = 0, <|Tr G|^2> = 1
    t = np.trace(gi.make_gauge(dims, 9), axis1=-2, axis2=-1)
    assert abs(t.mean()) < 0.05 and abs((np.abs(t) ** 2).mean() - 1) < 0.08
    # the raw field is a random gauge copy: <Re Tr U> ~ 0
    assert abs(np.trace(Uc, axis1=-2, axis2=-1).real.mean()) < 0.05


def test_configs_table_matches_baseline_json():
    import json, os
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    base = json.load(open(os.path.join(root, "BASELINE.json")))
    assert len(base["configs"]) == len(gi.CONFIGS) == 5
    vols = [4096, 131072, 1048576, 10616832, 33554432]
    for c, v in zip(gi.CONFIGS, vols):
        assert gi.volume(c["dims"]) == v
