"""Pins for the oracle's isotropic safety distance (reading 17): a lower bound, valid in
every direction, of the distance to the nearest boundary of the current volume or of one of its daughters.  The
paper only poses the boundary problem; what the mathematics fixes is pinned here:
  * points built at a chosen distance d off ONE face (inwards or outwards, every surface kind of every solid): safety = d;
  * the lower-bound property against the directional distances (DistanceToIn / DistanceToOut, pinned on their own by
    ray marching in test_oracle_solids.py / test_oracle_cone.py) over many directions;
  * tightness for box / tube / orb from inside: the direction towards the nearest surface attains it;
  * in a geometry: never larger than any ComputeStep from the same point, daughters only (no grand-daughters), known
    distances to a daughter's face and to the mother's wall, rotated daughters, vol = -1."""
import math

import numpy as np
import pytest

import oracle
from paper_1209_5235_b200 import workloads as W
from paper_1209_5235_b200.workloads import _Builder

TOL = 1e-9
BOX, TUBE, ORB, CONE = 0, 1, 2, 3


def unit(rng, n):
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def saf(stype, params, which, p, precision=64):
    return oracle.solid_eval(stype, params, TOL, which, np.atleast_2d(p), precision=precision)


# ---- points built at distance d off one face -----------------------------------------------------------------
def test_box_offsets_from_one_face():
    h = np.array([30.0, 40.0, 50.0])
    rng = np.random.default_rng(1)
    for axis in range(3):
        for sign in (-1.0, 1.0):
            for d in (0.125, 1.0, 7.5):
                p = rng.uniform(-0.5, 0.5, 3) * h                    # |p_i| <= h_i / 2: the other faces are >= 15 away
                p[axis] = sign * (h[axis] - d)
                assert saf(BOX, h, "safety_out", p)[0] == d and saf(BOX, h, "safety_in", p)[0] == 0.0
                p[axis] = sign * (h[axis] + d)
                assert saf(BOX, h, "safety_in", p)[0] == d and saf(BOX, h, "safety_out", p)[0] == 0.0
    # corner region: the bound is the largest single-face distance (a lower bound of the Euclidean distance sqrt(3^2 + 4^2) = 5)
    assert saf(BOX, h, "safety_in", h + np.array([3.0, 4.0, -1.0]))[0] == 4.0
    # centre: the smallest half-length
    assert saf(BOX, h, "safety_out", np.zeros(3))[0] == 30.0


def test_orb_offsets():
    rng = np.random.default_rng(2)
    u = unit(rng, 50)
    for d in (0.5, 3.0, 60.0):
        assert np.allclose(saf(ORB, (100.0,), "safety_out", u * (100.0 - d)), d, rtol=0, atol=1e-12)
        assert np.allclose(saf(ORB, (100.0,), "safety_in", u * (100.0 + d)), d, rtol=0, atol=1e-12)
    assert saf(ORB, (100.0,), "safety_out", np.zeros(3))[0] == 100.0


def test_tube_offsets_every_surface():
    rmin, rmax, hz, sphi, dphi = 20.0, 60.0, 80.0, 0.3, 1.2
    par = (rmin, rmax, hz, sphi, dphi)
    mid = sphi + dphi / 2

    def cyl(r, phi, z):
        return np.array([r * math.cos(phi), r * math.sin(phi), z])
    for d in (0.25, 2.0):
        # inside, d off each surface (the others are further away)
        assert saf(TUBE, par, "safety_out", cyl(rmax - d, mid, 10.0))[0] == pytest.approx(d, abs=1e-12)
        assert saf(TUBE, par, "safety_out", cyl(rmin + d, mid, -10.0))[0] == pytest.approx(d, abs=1e-12)
        assert saf(TUBE, par, "safety_out", cyl(40.0, mid, hz - d))[0] == pytest.approx(d, abs=1e-12)
        assert saf(TUBE, par, "safety_out", cyl(40.0, mid, -(hz - d)))[0] == pytest.approx(d, abs=1e-12)
        # d off a phi plane: a point at radius r and angle a from the plane is r sin(a) away from it
        a = math.asin(d / 40.0)
        assert saf(TUBE, par, "safety_out", cyl(40.0, sphi + a, 0.0))[0] == pytest.approx(d, abs=1e-12)
        assert saf(TUBE, par, "safety_out", cyl(40.0, sphi + dphi - a, 0.0))[0] == pytest.approx(d, abs=1e-12)
        # outside, d beyond each surface
        assert saf(TUBE, par, "safety_in", cyl(rmax + d, mid, 10.0))[0] == pytest.approx(d, abs=1e-12)
        assert saf(TUBE, par, "safety_in", cyl(rmin - d, mid, 10.0))[0] == pytest.approx(d, abs=1e-12)
        assert saf(TUBE, par, "safety_in", cyl(40.0, mid, hz + d))[0] == pytest.approx(d, abs=1e-12)
        assert saf(TUBE, par, "safety_in", cyl(40.0, sphi - a, 0.0))[0] == pytest.approx(d, abs=1e-12)
        assert saf(TUBE, par, "safety_in", cyl(40.0, sphi + dphi + a, 0.0))[0] == pytest.approx(d, abs=1e-12)
    # full tube without a hole: the axis is rmax (or hz) away
    assert saf(TUBE, (0.0, 60.0, 80.0, 0.0, 2 * math.pi), "safety_out", np.zeros(3))[0] == 60.0


@pytest.mark.parametrize("r1,r2,hz", [(20.0, 60.0, 50.0), (60.0, 20.0, 50.0), (40.0, 40.0, 30.0)])
def test_cone_offsets_along_the_surface_normal(r1, r2, hz):
    """A surface point of the frustum moved by d along the outward unit normal of the lateral surface
    (cos(phi), sin(phi), -m) / sqrt(1 + m^2), m = dr/dz, is d away from it."""
    par = (r1, r2, hz)
    m = (r2 - r1) / (2 * hz)
    cs = 1 / math.sqrt(1 + m * m)
    for phi in (0.1, 2.0, 4.5):
        for z in (-0.4 * hz, 0.0, 0.3 * hz):
            u = (r1 + r2) / 2 + m * z
            q = np.array([u * math.cos(phi), u * math.sin(phi), z])
            nrm = cs * np.array([math.cos(phi), math.sin(phi), -m])
            for d in (0.5, 3.0):
                assert saf(CONE, par, "safety_in", q + d * nrm)[0] == pytest.approx(d, abs=1e-11)
                assert saf(CONE, par, "safety_out", q - d * nrm)[0] == pytest.approx(d, abs=1e-11)
    assert saf(CONE, par, "safety_out", np.array([0.0, 0.0, hz - 1.5]))[0] == pytest.approx(1.5, abs=1e-12)
    assert saf(CONE, par, "safety_in", np.array([1.0, 0.0, -hz - 2.5]))[0] == pytest.approx(2.5, abs=1e-12)


# ---- lower bound against the directional distances, tightness from inside -----------------------------------------
SOLIDS = [
    (BOX, (30.0, 40.0, 50.0), 80.0, True),
    (TUBE, (0.0, 60.0, 80.0, 0.0, 2 * math.pi), 110.0, True),
    (TUBE, (20.0, 60.0, 80.0, 0.0, 2 * math.pi), 110.0, True),
    (TUBE, (20.0, 60.0, 80.0, 0.3, 1.2), 110.0, True),
    (TUBE, (0.0, 60.0, 30.0, -1.0, math.pi), 90.0, True),
    (ORB, (70.0,), 100.0, True),
    (CONE, (20.0, 60.0, 50.0), 90.0, False),
    (CONE, (0.0, 50.0, 40.0), 80.0, False),          # apex on the lower end plane
]


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("stype,par,span,exact", SOLIDS)
def test_safety_is_a_lower_bound_in_every_direction_and_attained_from_inside(stype, par, span, exact, precision):
    rng = np.random.default_rng(7 + stype)
    npts, ndir = 500, 300
    pts = rng.uniform(-span, span, size=(npts, 3))
    if precision == 32:
        pts = pts.astype(np.float32).astype(np.float64)
    inside = oracle.solid_eval(stype, par, TOL, "inside", pts, precision=precision)
    s_in = saf(stype, par, "safety_in", pts, precision).astype(np.float64)
    s_out = saf(stype, par, "safety_out", pts, precision).astype(np.float64)
    assert np.all(s_in >= 0) and np.all(s_out >= 0)
    assert np.all(s_out[inside == 2] == 0) and np.all(s_in[inside == 0] == 0)      # 0 = in, 2 = out
    assert (inside == 0).sum() > 5 and (inside == 2).sum() > 20
    slack = 1e-9 if precision == 64 else 2e-4
    dirs = unit(rng, ndir)
    for i in range(npts):
        p = pts[i]
        # directions towards the nearest point of each kind of surface: axes, radial (xy), radial (3-d), phi-plane normals
        special = [np.eye(3), -np.eye(3)]
        rxy = math.hypot(p[0], p[1])
        if rxy > 0:
            e = np.array([[p[0] / rxy, p[1] / rxy, 0.0]]); special += [e, -e]
        if np.linalg.norm(p) > 0:
            e = (p / np.linalg.norm(p))[None, :]; special += [e, -e]
        if stype == TUBE and par[4] < 2 * math.pi:
            for a, sg in ((par[3], 1.0), (par[3] + par[4], -1.0)):
                special.append(np.array([[sg * math.sin(a), -sg * math.cos(a), 0.0]]))
        v = np.vstack([dirs] + special)
        P = np.repeat(p[None, :], len(v), axis=0)
        if inside[i] == 0:
            t = oracle.solid_eval(stype, par, TOL, "dist_out", P, v, precision=precision).astype(np.float64)
            assert t.min() >= s_out[i] * (1 - slack) - slack
            if exact:                                                  # box, tube, orb: some direction attains the bound
                assert t.min() <= s_out[i] * (1 + slack) + slack
            else:                                                      # cone: within 2 % here (frusta, no apex nearby) or the apex case
                assert t.min() <= s_out[i] * 1.6 + slack
        elif inside[i] == 2:
            t = oracle.solid_eval(stype, par, TOL, "dist_in", P, v, precision=precision).astype(np.float64)
            assert np.all(t >= s_in[i] * (1 - slack) - slack)          # +inf where the ray misses


# ---- in a geometry ---------------------------------------------------------------------------------------------
def test_safety_in_config1_known_distances():
    g = W.slab_geometry(1)
    og = oracle.OracleGeometry(g)
    T = np.asarray(g.transforms, float).reshape(-1, 12)[:, 9:]
    places = np.asarray(g.placements).reshape(-1, 4)
    water = [i for i in range(2, 6)]
    c = T[places[water[0], 3]]
    pts = np.array([
        [0.0, 0.0, -300.0],                 # world: 250 from the lead box (z face), 200 from the world wall
        [0.0, 0.0, -120.0],                 # world: 70 from the lead box
        [480.0, 0.0, 0.0],                  # world: 20 from the world wall
        [c[0], c[1], c[2] + 13.0],          # lead, 3 above the first water box (water boxes are >= 1 apart, faces of the lead >= 1 away)
        [c[0], c[1], c[2] + 9.0],           # water box 0: 1 from its own top face
    ])
    vol = og.locate(pts, None, 64)
    assert list(vol) == [0, 0, 0, 1, water[0]]
    s = og.compute_safety(pts, vol, 64)
    assert s[0] == 200.0 and s[1] == 70.0 and s[2] == 20.0 and s[4] == pytest.approx(1.0, abs=1e-12)
    assert s[3] <= 3.0 + 1e-12 and s[3] > 0
    # outside the world (vol = -1) there is nothing to be safe from: 0
    assert og.compute_safety(pts[:1], np.array([-1], np.int32), 64)[0] == 0.0
    s32 = og.compute_safety(pts.astype(np.float32), vol, 32)
    assert np.allclose(s32, s, rtol=1e-5, atol=1e-4)


@pytest.mark.parametrize("name", ["config1", "mixed", "cmslike", "detector"])
def test_no_computed_step_is_shorter_than_the_safety(name):
    g = {"config1": lambda: W.slab_geometry(1), "mixed": lambda: W.mixed_solids_geometry(3, seed=9),
         "cmslike": W.cms_like_geometry,
         "detector": lambda: W.detector_geometry(seed=4, n_phi=8, n_z=4, barrels=((200, 400),))}[name]()
    og = oracle.OracleGeometry(g)
    pos, _ = W.nav_queries(g, 400, seed=3, dtype=np.float64)
    vol = og.locate(pos, None, 64)
    keep = vol >= 0
    pos, vol = pos[keep], vol[keep]
    s = og.compute_safety(pos, vol, 64)
    assert np.all(s >= 0) and np.isfinite(s).all() and (s > 0).mean() > 0.9
    rng = np.random.default_rng(5)
    tight = np.full(len(pos), np.inf)
    for _ in range(60):
        w = unit(rng, len(pos))
        v2 = og.locate(pos, w, 64)                                  # with a direction: the volume the step starts in
        same = v2 == vol
        step, _ = og.compute_step(pos, w, vol, None, 64)
        assert np.all(step[same] >= s[same] - 1e-9)
        tight = np.minimum(tight, np.where(same, step, np.inf))
    # the bound is not vacuous: over 60 random directions the shortest step found is within 4x of it for most points
    assert np.median(tight / np.maximum(s, 1e-12)) < 4.0


def test_rotated_daughter_safety():
    b = _Builder("rot")
    world = b.place(-1, b.box(500.0, 500.0, 500.0), "vacuum")
    b.place(world, b.box(10.0, 20.0, 30.0), "lead", R=W.rot_z(math.pi / 2), T=(100.0, 0.0, 0.0))     # local x -> global y
    g = b.finish()
    og = oracle.OracleGeometry(g)
    # rotated by 90 degrees about z the box spans x in [80, 120], y in [-10, 10]
    pts = np.array([[70.0, 0.0, 0.0], [100.0, 15.0, 0.0], [100.0, 0.0, 37.0]])
    s = og.compute_safety(pts, np.zeros(3, np.int32), 64)
    assert np.allclose(s, [10.0, 5.0, 7.0], rtol=0, atol=1e-12)
    inside = og.compute_safety(np.array([[100.0, 0.0, 0.0]]), np.array([1], np.int32), 64)
    assert inside[0] == pytest.approx(10.0, abs=1e-12)
