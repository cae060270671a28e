"""Pins for the oracle's cone solid (PAPER.md L160 names cones): closed forms on the axis and in
the symmetry plane, dense ray marching of the point set {|z| <= hz, r <= r0 + m z} written out here, the convex round
trip, and the normal's defining property through Inside() only."""
import math

import numpy as np
import pytest

import oracle

TOL = 1e-9
CONE = 3
CASES = [[10.0, 30.0, 40.0], [30.0, 10.0, 25.0], [0.0, 20.0, 15.0], [25.0, 25.0, 30.0], [40.0, 0.0, 10.0]]


def unit(rng, n):
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def member(par, p):
    r1, r2, hz = par
    u = (r1 + r2) / 2 + (r2 - r1) / (2 * hz) * p[..., 2]
    return (np.abs(p[..., 2]) <= hz) & (np.hypot(p[..., 0], p[..., 1]) <= u)


def march(par, p, v, tmax, n=40001):
    ts = np.linspace(0.0, tmax, n)
    m = member(par, p[None, :] + ts[:, None] * v[None, :])
    ch = np.nonzero(m[1:] != m[:-1])[0]
    if len(ch) == 0:
        return math.inf
    lo, hi, m0 = ts[ch[0]], ts[ch[0] + 1], m[ch[0]]
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        if member(par, (p + mid * v)[None, :])[0] == m0:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


def test_cone_closed_forms():
    par = [10.0, 30.0, 40.0]                                 # r0 = 20, slope 0.25
    z = np.linspace(-39, 39, 40)
    p = np.stack([np.zeros_like(z), np.zeros_like(z), z], axis=1)
    ez = np.tile([0.0, 0.0, 1.0], (len(z), 1)); ex = np.tile([1.0, 0.0, 0.0], (len(z), 1))
    assert np.allclose(oracle.solid_eval(CONE, par, TOL, "dist_out", p, ez), 40 - z, rtol=1e-14)
    assert np.allclose(oracle.solid_eval(CONE, par, TOL, "dist_out", p, -ez), 40 + z, rtol=1e-14)
    assert np.allclose(oracle.solid_eval(CONE, par, TOL, "dist_out", p, ex), 20 + 0.25 * z, rtol=1e-13)       # horizontal: u(z)
    # from outside, horizontally towards the axis at height z: enters at x = u(z)
    q = p + ex * 100.0
    assert np.allclose(oracle.solid_eval(CONE, par, TOL, "dist_in", q, -ex), 100 - (20 + 0.25 * z), rtol=1e-13)
    assert np.all(np.isinf(oracle.solid_eval(CONE, par, TOL, "dist_in", q, ex)))
    # along a generator direction from the axis: hits the cone where r(t) = u(z(t)) -- solve by hand: t s = 20 + 0.25 (z0 + t c)
    th = math.radians(50); s_, c_ = math.sin(th), math.cos(th)
    d = np.tile([s_, 0.0, c_], (len(z), 1))
    t_cone = (20 + 0.25 * z) / (s_ - 0.25 * c_)
    t_plane = (40 - z) / c_
    assert np.allclose(oracle.solid_eval(CONE, par, TOL, "dist_out", p, d), np.minimum(t_cone, t_plane), rtol=1e-13)
    # inside classification on the slanted surface
    pts = np.array([[20 + 0.25 * 12.0, 0, 12.0], [0, 20 + 0.25 * -30.0, -30.0]])
    assert oracle.solid_eval(CONE, par, TOL, "inside", pts).tolist() == [1, 1]


@pytest.mark.parametrize("par", CASES)
def test_cone_ray_marching_round_trip_and_normals(par):
    rng = np.random.default_rng(int(par[0] * 7 + par[1]))
    r1, r2, hz = par
    rmax = max(r1, r2)
    cand = rng.uniform(-1, 1, size=(6000, 3)) * np.array([rmax, rmax, hz]) * 1.6
    cls = oracle.solid_eval(CONE, par, TOL, "inside", cand)
    assert np.array_equal(cls == 0, member(par, cand) & (cls != 1)) or np.all((cls == 0) == member(par, cand))
    pin = cand[cls == 0][:250]; pout = cand[cls == 2][:250]
    v = unit(rng, 250)
    dout = oracle.solid_eval(CONE, par, TOL, "dist_out", pin, v[:len(pin)])
    din = oracle.solid_eval(CONE, par, TOL, "dist_in", pout, v[:len(pout)])
    span = 4 * (rmax + hz)
    for i in range(len(pin)):
        assert abs(dout[i] - march(par, pin[i], v[i], span)) < 2e-6
    n_hit = 0
    for i in range(len(pout)):
        m = march(par, pout[i], v[i], span)
        if math.isinf(m):
            continue                                        # a miss (or a graze below the marching resolution)
        # the marcher reports the first change of membership, i.e. the entry
        assert abs(din[i] - m) < 2e-6, (par, pout[i], v[i], din[i], m)
        n_hit += 1
    assert n_hit > 20
    # clear misses are +inf: rays pointing away from the bounding cylinder
    away = pout / np.linalg.norm(pout, axis=1, keepdims=True)
    far = np.linalg.norm(pout[:, :2], axis=1) > rmax + 1
    assert np.all(np.isinf(oracle.solid_eval(CONE, par, TOL, "dist_in", pout[far], away[far])))
    # round trip (convex): leave by t, go s further, come back
    s = rng.uniform(0.1, 20.0, len(pin))
    back = pin + v[:len(pin)] * (dout + s)[:, None]
    assert np.allclose(oracle.solid_eval(CONE, par, TOL, "dist_in", back, -v[:len(pin)]), s, rtol=1e-8, atol=1e-7)
    # normals at the exit points: unit, along the ray, +n out / -n in / tangent stays (Inside() only)
    q = pin + v[:len(pin)] * dout[:, None]
    nrm = oracle.solid_eval(CONE, par, TOL, "normal", q)
    assert np.allclose(np.linalg.norm(nrm, axis=1), 1.0, atol=1e-14)
    assert np.all(np.einsum("ij,ij->i", nrm, v[:len(pin)]) > -1e-12)
    eps = 1e-6
    assert np.all(oracle.solid_eval(CONE, par, TOL, "inside", q + eps * nrm) == 2)
    assert (oracle.solid_eval(CONE, par, TOL, "inside", q - eps * nrm) == 0).mean() > 0.99
    tang = np.cross(nrm, unit(rng, len(q))); tang /= np.linalg.norm(tang, axis=1, keepdims=True)
    assert (oracle.solid_eval(CONE, par, TOL, "inside", q + 1e-5 * tang) == 1).mean() > 0.99


def test_navigation_through_all_four_solid_types():
    """Boxes, tubes, cones and balls, randomly rotated, some with a ball inside: the oracle's locate equals
    the brute-force locate (hierarchical transforms, no navigator), the voxel-accelerated locate changes nothing, and the
    chained steps of a ray add up to the analytic exit distance of the world box without zero-length steps."""
    from paper_1209_5235_b200 import workloads as W
    geom = W.mixed_solids_geometry()
    og = oracle.OracleGeometry(geom)
    rng = np.random.default_rng(17)
    n = 30000
    h = W.world_half_extent(geom)
    pos = rng.uniform(-1, 1, size=(n, 3)) * h * 0.98
    d = unit(rng, n)
    vol = og.locate(pos, d, use_grid=False)
    assert np.array_equal(vol, og.locate(pos, d, use_grid=True))
    bf = og.locate_bruteforce(pos)
    assert (vol == bf).mean() > 0.9999                      # (points within the tolerance of a surface may differ)
    stype = geom.solid_type[geom.placements[np.maximum(vol, 0), 1]]
    assert all((stype[vol > 0] == t).sum() > 20 for t in (0, 1, 2, 3))     # the solids fill ~1 % of the cube
    # chained steps along 400 rays
    m = 400
    x = pos[:m].copy(); w = d[:m]; v = vol[:m].copy()
    total = np.zeros(m); alive = v >= 0; nsteps = np.zeros(m, int)
    texit = np.min(np.where(w != 0, (np.sign(w) * h - x) / np.where(w != 0, w, 1), np.inf), axis=1)
    for _ in range(200):
        if not alive.any():
            break
        idx = np.nonzero(alive)[0]
        step, nxt = og.compute_step(x[idx], w[idx], v[idx], None, 64, use_grid=False)
        assert np.all(np.isfinite(step)) and np.all(step >= 0)
        assert (step <= TOL / 2).sum() <= 2                 # no zero-length steps (tangential touches excepted)
        x[idx] += w[idx] * step[:, None]; total[idx] += step; v[idx] = nxt; nsteps[idx] += 1
        alive[idx] = nxt >= 0
    assert not alive.any()
    assert np.allclose(total, texit, rtol=1e-12, atol=1e-9)
    assert nsteps.max() > 4
