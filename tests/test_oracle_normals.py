"""Pins for the oracle's surface normals ("what is the normal of the boundary surface at that point?";
DESIGN.md "surface normal").  Independent of the normal code itself: closed forms per face, and the defining property
checked through the Inside classification and brute-force locate only -- a short move along +n leaves the solid, along -n
enters it, along any tangent stays on the surface."""
import math

import numpy as np
import pytest

import oracle
from paper_1209_5235_b200 import workloads as W

TOL = 1e-9
BOX, TUBE, ORB = 0, 1, 2


def unit(rng, n):
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def test_box_tube_orb_normals_closed_forms():
    h = [10.0, 20.0, 30.0]
    p = np.array([[10, 3, -4], [-10, 3, -4], [1, 20, 2], [1, -20, 2], [1, 2, 30], [1, 2, -30.0]])
    n = oracle.solid_eval(BOX, h, TOL, "normal", p)
    assert np.array_equal(n, np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1.0]]))
    rng = np.random.default_rng(1)
    ang = rng.uniform(0, 2 * math.pi, 200)
    z = rng.uniform(-40, 40, 200)
    outer = np.stack([80 * np.cos(ang), 80 * np.sin(ang), z], axis=1)
    inner = np.stack([50 * np.cos(ang), 50 * np.sin(ang), z], axis=1)
    tube = [50.0, 80.0, 45.0, 0.0, 7.0]
    rad = np.stack([np.cos(ang), np.sin(ang), np.zeros_like(ang)], axis=1)
    assert np.allclose(oracle.solid_eval(TUBE, tube, TOL, "normal", outer), rad, atol=1e-15)
    assert np.allclose(oracle.solid_eval(TUBE, tube, TOL, "normal", inner), -rad, atol=1e-15)
    caps = np.stack([65 * np.cos(ang), 65 * np.sin(ang), np.where(z > 0, 45.0, -45.0)], axis=1)
    want = np.zeros((200, 3)); want[:, 2] = np.where(z > 0, 1.0, -1.0)
    assert np.array_equal(oracle.solid_eval(TUBE, tube, TOL, "normal", caps), want)
    # sector planes of a 60 degree wedge starting at 30 degrees
    s0, d0 = math.radians(30), math.radians(60)
    sec = [50.0, 80.0, 45.0, s0, d0]
    ps = np.array([[65 * math.cos(s0), 65 * math.sin(s0), 3.0], [65 * math.cos(s0 + d0), 65 * math.sin(s0 + d0), -7.0]])
    ns = oracle.solid_eval(TUBE, sec, TOL, "normal", ps)
    assert np.allclose(ns[0], [math.sin(s0), -math.cos(s0), 0], atol=1e-15)
    assert np.allclose(ns[1], [-math.sin(s0 + d0), math.cos(s0 + d0), 0], atol=1e-15)
    q = unit(rng, 300) * 25.0
    assert np.allclose(oracle.solid_eval(ORB, [25.0], TOL, "normal", q), q / 25.0, atol=1e-15)


@pytest.mark.parametrize("stype,params,scale", [(BOX, [7.0, 11.0, 5.0], 12.0), (TUBE, [20.0, 45.0, 30.0, 0.0, 7.0], 50.0),
                                                 (TUBE, [15.0, 40.0, 25.0, 0.4, 1.1], 45.0), (ORB, [33.0], 40.0)])
def test_normal_is_the_direction_out_of_the_solid(stype, params, scale):
    """Surface points found by shooting rays from inside (DistanceToOut); then, with Inside() only: +n leaves, -n enters,
    tangents stay on the surface."""
    rng = np.random.default_rng(7)
    n = 4000
    p = rng.uniform(-1, 1, size=(n, 3)) * scale
    inside = oracle.solid_eval(stype, params, TOL, "inside", p) == 0
    p = p[inside][:600]
    v = unit(rng, len(p))
    t = oracle.solid_eval(stype, params, TOL, "dist_out", p, v)
    q = p + v * t[:, None]
    assert np.all(oracle.solid_eval(stype, params, TOL, "inside", q) == 1)           # on the surface
    nrm = oracle.solid_eval(stype, params, TOL, "normal", q)
    assert np.allclose(np.linalg.norm(nrm, axis=1), 1.0, atol=1e-14)
    assert np.all(np.einsum("ij,ij->i", nrm, v) > -1e-12)                           # leaving: n.v >= 0
    eps = 1e-6
    assert np.all(oracle.solid_eval(stype, params, TOL, "inside", q + eps * nrm) == 2)
    # -n enters, except next to an edge where another face is closer than eps
    back = oracle.solid_eval(stype, params, TOL, "inside", q - eps * nrm)
    assert (back == 0).mean() > 0.999
    tang = np.cross(nrm, unit(rng, len(q))); tang /= np.linalg.norm(tang, axis=1, keepdims=True)
    small = 1e-5                                                                    # second-order departure << tolerance
    stay = oracle.solid_eval(stype, params, TOL, "inside", q + small * tang)
    assert (stay == 1).mean() > 0.995                                               # (edges: the tangent may leave the face)


def test_compute_step_normal_entry_and_exit():
    """Tiny slab (config 1, unrotated boxes): rays from the world towards the lead box enter through the face whose
    outward normal opposes them; rays from inside the lead box leave through the face they point at."""
    geom = W.slab_geometry(1)
    og = oracle.OracleGeometry(geom)
    rng = np.random.default_rng(3)
    n = 3000
    pos = np.zeros((n, 3)); pos[:, 2] = -300.0; pos[:, :2] = rng.uniform(-40, 40, size=(n, 2))
    d = np.tile([0.0, 0.0, 1.0], (n, 1))
    vol = og.locate(pos, d)
    step, nxt, nrm = og.compute_step_normal(pos, d, vol)
    assert np.all(vol == 0) and np.allclose(step, 250.0) and np.all(nxt == 1)
    assert np.array_equal(nrm, np.tile([0.0, 0.0, -1.0], (n, 1)))                   # entry: the daughter's outward normal
    s0, n0 = og.compute_step(pos, d, vol)
    assert np.array_equal(step, s0) and np.array_equal(nxt, n0)                     # same step as the plain call
    # beyond max_step: no boundary, zero normal
    step, nxt, nrm = og.compute_step_normal(pos, d, vol, max_step=np.full(n, 100.0))
    assert np.all(np.isinf(step)) and np.all(nrm == 0)
    # leaving the world: its own outward normal
    pos2 = rng.uniform(-400, 400, size=(n, 3)); pos2[:, 0] = 450.0
    d2 = unit(rng, n); d2[:, 0] = np.abs(d2[:, 0]) + 2.0; d2 /= np.linalg.norm(d2, axis=1, keepdims=True)
    v2 = og.locate(pos2, d2)
    step, nxt, nrm = og.compute_step_normal(pos2, d2, v2)
    hit_x = np.isclose(pos2[:, 0] + step * d2[:, 0], 500.0)
    assert hit_x.mean() > 0.9 and np.array_equal(nrm[hit_x], np.tile([1.0, 0.0, 0.0], (hit_x.sum(), 1))) and np.all(nxt[hit_x] == -1)


def test_compute_step_normal_on_rotated_solids_via_brute_force_locate():
    """Lattice of randomly rotated boxes / tubes: the normal is a unit vector, opposes the ray on entry, points along it on
    exit, and the two sides of the boundary (x_n +- 1e-6 n) are located -- by the brute-force locate, which knows nothing of
    normals -- in different volumes, the -n side being the volume whose surface it is."""
    geom = W.lattice_geometry(4, seed=7)
    og = oracle.OracleGeometry(geom)
    rng = np.random.default_rng(11)
    n = 6000
    pos = rng.uniform(-1, 1, size=(n, 3)) * W.world_half_extent(geom) * 0.95
    d = unit(rng, n)
    vol = og.locate(pos, d, use_grid=False)
    step, nxt, nrm = og.compute_step_normal(pos, d, vol, use_grid=False)
    ok = np.isfinite(step) & (vol >= 0)
    xn = pos[ok] + d[ok] * step[ok][:, None]
    nn = nrm[ok]
    assert np.allclose(np.linalg.norm(nn, axis=1), 1.0, atol=1e-12)
    parent = geom.placements[:, 0]
    entering = (nxt[ok] > 0) & (parent[np.maximum(nxt[ok], 0)] == vol[ok])           # the step ends on a daughter's surface
    leaving = ~entering                                                              # ... or on the volume's own
    assert entering.sum() > 200
    ndotw = np.einsum("ij,ij->i", nn, d[ok])
    assert np.all(ndotw[entering] < 1e-9) and np.all(ndotw[leaving] > -1e-9)
    eps = 1e-6
    inner = og.locate_bruteforce(xn - eps * nn); outer = og.locate_bruteforce(xn + eps * nn)
    owner = np.where(entering, nxt[ok], vol[ok])                                     # the solid whose surface was hit
    sel = entering | (leaving & (vol[ok] > 0))                                       # (the world's own surface: outside is -1)
    assert (inner[sel] == owner[sel]).mean() > 0.995                                 # (edges and grazes excepted)
    assert (outer[sel] != owner[sel]).mean() > 0.995
    # second leg: carry on from the entry points through the solids just entered -> exit normals
    p2, d2, v2 = xn[entering], d[ok][entering], nxt[ok][entering]
    step2, nxt2, nrm2 = og.compute_step_normal(p2, d2, v2, use_grid=False)
    own = ~((nxt2 > 0) & (parent[np.maximum(nxt2, 0)] == v2))                         # ends on the solid's own surface, not on a nested daughter
    fin = np.isfinite(step2) & (step2 > 1e-6) & own
    assert fin.sum() > 200
    x2 = p2[fin] + d2[fin] * step2[fin][:, None]
    assert np.allclose(np.linalg.norm(nrm2[fin], axis=1), 1.0, atol=1e-12)
    assert np.all(np.einsum("ij,ij->i", nrm2[fin], d2[fin]) > -1e-9)                  # leaving: along the ray
    inner2 = og.locate_bruteforce(x2 - eps * nrm2[fin]); outer2 = og.locate_bruteforce(x2 + eps * nrm2[fin])
    assert (inner2 == v2[fin]).mean() > 0.995 and (outer2 != v2[fin]).mean() > 0.995
