"""Pins for the oracle's navigator on the deep synthetic detector hierarchy ("a deeper CMS-like
synthetic hierarchy"; the paper's CMS model, is not available).  Expectations come from outside the
navigator: the brute-force locate (hierarchical point transforms + Inside only), the geometry's own construction, and the
analytic exit distance of the world box that every chain of steps must add up to."""
import numpy as np

import oracle
from paper_1209_5235_b200 import workloads as W

TOL = 1e-9


def unit(rng, n):
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def node_origins(geom, nodes):
    out = []
    for i in nodes:
        x = np.zeros(3)
        while i > 0:
            tr = geom.transforms[geom.placements[i, 3]]
            x = tr[:9].reshape(3, 3) @ x + tr[9:]
            i = geom.placements[i, 0]
        out.append(x)
    return np.array(out)


def depth_of(geom):
    par = geom.placements[:, 0]
    d = np.zeros(geom.n_places, int)
    for i in range(1, geom.n_places):
        d[i] = d[par[i]] + 1
    return d


def test_hierarchy_shape():
    geom = W.cms_like_geometry()
    d = depth_of(geom)
    assert d.max() == 6                                               # world, ECAL, ring, sector, crystal, cone, ball
    st = geom.solid_type[geom.placements[:, 1]]
    assert all((st == t).sum() >= 3 for t in (0, 1, 2, 3))
    assert (geom.placements[1:, 0] < np.arange(1, geom.n_places)).all()
    assert (geom.placements[:, 0] == 0).sum() >= 8                    # the world is voxelised


def test_locate_equals_brute_force_everywhere_and_in_the_deep_branch():
    geom = W.cms_like_geometry()
    og = oracle.OracleGeometry(geom)
    rng = np.random.default_rng(23)
    n = 60000
    h = W.world_half_extent(geom)
    pos = rng.uniform(-1, 1, size=(n, 3)) * h * 0.999
    st = geom.solid_type[geom.placements[:, 1]]
    cones = np.nonzero((st == 3) & (geom.placements[:, 0] > 0))[0]
    cg = node_origins(geom, cones)
    pos[: n // 2] = cg[rng.integers(0, len(cg), n // 2)] + rng.normal(size=(n // 2, 3)) * 50.0
    d = unit(rng, n)
    vol = og.locate(pos, d, use_grid=False)
    assert np.array_equal(vol, og.locate(pos, d, use_grid=True))
    bf = og.locate_bruteforce(pos)
    assert (vol == bf).mean() > 0.9999
    dep = depth_of(geom)[np.maximum(vol, 0)]
    assert all((dep == k).sum() > 30 for k in range(7)) and (dep == 6).sum() > 300    # every level of the tree is hit
    # the ball at the bottom of the first crystal: its centre is inside it, by construction
    balls = np.nonzero((st == 2) & (depth_of(geom) == 6))[0]
    assert np.array_equal(og.locate(node_origins(geom, balls), None), balls)


def test_chained_steps_add_up_to_the_world_exit():
    geom = W.cms_like_geometry()
    og = oracle.OracleGeometry(geom)
    rng = np.random.default_rng(29)
    m = 1500
    h = W.world_half_extent(geom)
    st = geom.solid_type[geom.placements[:, 1]]
    cones = np.nonzero((st == 3) & (geom.placements[:, 0] > 0))[0]
    cg = node_origins(geom, cones)
    x = rng.uniform(-1, 1, size=(m, 3)) * h * 0.98
    x[: m // 2] = cg[rng.integers(0, len(cg), m // 2)] + rng.normal(size=(m // 2, 3)) * 30.0
    w = unit(rng, m)
    v = og.locate(x, w, use_grid=False)
    texit = np.min(np.where(w != 0, (np.sign(w) * h - x) / np.where(w != 0, w, 1), np.inf), axis=1)
    total = np.zeros(m); alive = v >= 0; nsteps = np.zeros(m, int); zero = 0
    x = x.copy()
    for _ in range(400):
        if not alive.any():
            break
        idx = np.nonzero(alive)[0]
        step, nxt = og.compute_step(x[idx], w[idx], v[idx], None, 64, use_grid=True)
        s2, n2 = og.compute_step(x[idx], w[idx], v[idx], None, 64, use_grid=False)
        assert np.array_equal(step, s2) and np.array_equal(nxt, n2)          # the voxel index changes nothing
        assert np.all(np.isfinite(step)) and np.all(step >= 0)
        zero += int((step <= TOL / 2).sum())
        x[idx] += w[idx] * step[:, None]; total[idx] += step; v[idx] = nxt; nsteps[idx] += 1
        alive[idx] = nxt >= 0
    assert not alive.any()
    assert zero <= 3                                                         # (tangential touches excepted)
    assert np.allclose(total, texit, rtol=1e-12, atol=1e-8)
    assert nsteps.max() >= 12 and nsteps.mean() > 4
