"""Pins for the oracle's solids: analytic cases, dense ray marching of the solid's
point-membership function written out independently here, and the convex round trip.
BASELINE.json north_star: "analytic distances to box and tube surfaces"."""
import math

import numpy as np
import pytest

import oracle

TOL = 1e-9
BOX, TUBE = 0, 1


# ---- independent point membership (exact set definitions, numpy) -------------------------------
def member_box(h, p):
    return np.all(np.abs(p) <= np.asarray(h), axis=-1)


def member_tube(rmin, rmax, hz, sphi, dphi, p):
    r = np.hypot(p[..., 0], p[..., 1])
    ok = (np.abs(p[..., 2]) <= hz) & (r <= rmax) & (r >= rmin)
    if dphi < 2 * math.pi:
        ang = np.mod(np.arctan2(p[..., 1], p[..., 0]) - sphi, 2 * math.pi)
        ok &= ang <= dphi
    return ok


def march(member, p, v, tmax, n=20001):
    """first parameter t in (0, tmax] at which membership along p + t v changes, refined by bisection;
    returns (t, min_gap) or (inf, ...) -- brute force, no solid formulas."""
    ts = np.linspace(0.0, tmax, n)
    m = member(p[None, :] + ts[:, None] * v[None, :])
    ch = np.nonzero(m[1:] != m[:-1])[0]
    if len(ch) == 0:
        return math.inf
    lo, hi = ts[ch[0]], ts[ch[0] + 1]
    m0 = m[ch[0]]
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        if member((p + mid * v)[None, :])[0] == m0:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


def unit(rng, n):
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


# ---- analytic cases ------------------------------------------------------------------------------
def test_box_axis_rays_exact():
    h = (3.0, 4.0, 5.0)
    p = np.array([[1.0, -2.0, 0.5]] * 6)
    v = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], float)
    out = oracle.solid_eval(BOX, h, TOL, "dist_out", p, v)
    assert np.array_equal(out, [2.0, 4.0, 6.0, 2.0, 4.5, 5.5])
    po = np.array([[-10.0, 1, 1], [10.0, 1, 1], [1, -14.0, 1], [1, 1, 25.0], [-10.0, 5.0, 1], [-10, 1, 1]])
    vo = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, 0, -1], [1, 0, 0], [-1, 0, 0]], float)
    got = oracle.solid_eval(BOX, h, TOL, "dist_in", po, vo)
    assert np.array_equal(got, [7.0, 7.0, 10.0, 20.0, math.inf, math.inf])


def test_box_diagonal_ray():
    # from (-10,-10,-10) along (1,1,1)/sqrt3 into the cube of half 2: enters at (-2,-2,-2)
    s3 = math.sqrt(3.0)
    d = oracle.solid_eval(BOX, (2, 2, 2), TOL, "dist_in", [[-10.0, -10, -10]], [[1 / s3, 1 / s3, 1 / s3]])
    assert abs(d[0] - 8 * s3) < 1e-12
    d = oracle.solid_eval(BOX, (2, 2, 2), TOL, "dist_out", [[0.0, 0, 0]], [[1 / s3, 1 / s3, 1 / s3]])
    assert abs(d[0] - 2 * s3) < 1e-12


def test_box_surface_semantics():
    h = (1.0, 1.0, 1.0)
    # on the +x face: moving out -> DistanceToOut 0, moving in -> positive; from outside on the face moving in -> 0
    assert oracle.solid_eval(BOX, h, TOL, "dist_out", [[1.0, 0, 0]], [[1.0, 0, 0]])[0] == 0.0
    assert oracle.solid_eval(BOX, h, TOL, "dist_out", [[1.0, 0, 0]], [[-1.0, 0, 0]])[0] == 2.0
    assert oracle.solid_eval(BOX, h, TOL, "dist_in", [[1.0, 0, 0]], [[-1.0, 0, 0]])[0] == 0.0
    assert oracle.solid_eval(BOX, h, TOL, "dist_in", [[1.0, 0, 0]], [[1.0, 0, 0]])[0] == math.inf
    assert oracle.solid_eval(BOX, h, TOL, "dist_in", [[1.0, 0, 0]], [[0.0, 1.0, 0]])[0] == math.inf   # sliding along the face
    ins = oracle.solid_eval(BOX, h, TOL, "inside", [[0, 0, 0], [1.0, 0, 0], [1.0 + 1e-6, 0, 0], [1 - 1e-6, 0.5, 0]])
    assert list(ins) == [0, 1, 2, 0]


def test_tube_radial_and_chord():
    rmin, rmax, hz = 2.0, 5.0, 10.0
    p = np.array([[3.5, 0, 1.0]] * 2)
    v = np.array([[1.0, 0, 0], [-1.0, 0, 0]])
    out = oracle.solid_eval(TUBE, (rmin, rmax, hz, 0, 2 * math.pi), TOL, "dist_out", p, v)
    assert np.allclose(out, [1.5, 1.5], rtol=0, atol=1e-14)
    # chord of the outer circle at impact parameter b: enter at -sqrt(R^2-b^2), length 2 sqrt(R^2-b^2)
    for b in (0.0, 1.0, 3.0, 4.9):
        half = math.sqrt(rmax * rmax - b * b)
        din = oracle.solid_eval(TUBE, (0.0, rmax, hz, 0, 2 * math.pi), TOL, "dist_in", [[-20.0, b, 0.0]], [[1.0, 0, 0]])[0]
        assert abs(din - (20.0 - half)) < 1e-12
        dout = oracle.solid_eval(TUBE, (0.0, rmax, hz, 0, 2 * math.pi), TOL, "dist_out", [[-half + 1e-3, b, 0.0]], [[1.0, 0, 0]])[0]
        assert abs(dout - (2 * half - 1e-3)) < 1e-11
    # from inside the hole: entry at rmin; from outside through the hole: exit of the first wall at the hole
    assert abs(oracle.solid_eval(TUBE, (rmin, rmax, hz, 0, 2 * math.pi), TOL, "dist_in", [[0.5, 0, 0]], [[1.0, 0, 0]])[0] - 1.5) < 1e-14
    assert abs(oracle.solid_eval(TUBE, (rmin, rmax, hz, 0, 2 * math.pi), TOL, "dist_out", [[-4.0, 0, 0]], [[1.0, 0, 0]])[0] - 2.0) < 1e-14
    # z plane entry and exit
    assert oracle.solid_eval(TUBE, (rmin, rmax, hz, 0, 2 * math.pi), TOL, "dist_in", [[3.0, 0, -15.0]], [[0, 0, 1.0]])[0] == 5.0
    assert oracle.solid_eval(TUBE, (rmin, rmax, hz, 0, 2 * math.pi), TOL, "dist_out", [[3.0, 0, -5.0]], [[0, 0, 1.0]])[0] == 15.0
    # ray along z inside the hole never enters
    assert oracle.solid_eval(TUBE, (rmin, rmax, hz, 0, 2 * math.pi), TOL, "dist_in", [[0.5, 0, -15.0]], [[0, 0, 1.0]])[0] == math.inf


def test_tube_sector_planes():
    # quarter sector [0, pi/2]: from (3, -1) moving +y hits the start plane y = 0 after 1
    prm = (1.0, 5.0, 4.0, 0.0, math.pi / 2)
    assert abs(oracle.solid_eval(TUBE, prm, TOL, "dist_in", [[3.0, -1.0, 0]], [[0, 1.0, 0]])[0] - 1.0) < 1e-14
    # from inside at (2,2) moving -x exits through x = 0 (end plane) after 2
    assert abs(oracle.solid_eval(TUBE, prm, TOL, "dist_out", [[2.0, 2.0, 0]], [[-1.0, 0, 0]])[0] - 2.0) < 1e-14
    # the extension of the start plane beyond the axis is not part of the solid
    assert oracle.solid_eval(TUBE, prm, TOL, "dist_in", [[-3.0, -1.0, 0]], [[0, 1.0, 0]])[0] == math.inf


# ---- brute force -----------------------------------------------------------------------------------
SOLIDS = [
    (BOX, (3.0, 4.0, 5.0), lambda p: member_box((3.0, 4.0, 5.0), p), 12.0),
    (TUBE, (0.0, 4.0, 5.0, 0.0, 2 * math.pi), lambda p: member_tube(0.0, 4.0, 5.0, 0.0, 2 * math.pi, p), 12.0),
    (TUBE, (2.0, 4.0, 5.0, 0.0, 2 * math.pi), lambda p: member_tube(2.0, 4.0, 5.0, 0.0, 2 * math.pi, p), 12.0),
    (TUBE, (200.0, 400.0, 25.0, -math.pi / 32, math.pi / 16), lambda p: member_tube(200.0, 400.0, 25.0, -math.pi / 32, math.pi / 16, p), 900.0),
    (TUBE, (1.5, 4.0, 5.0, 0.4, 2.5), lambda p: member_tube(1.5, 4.0, 5.0, 0.4, 2.5, p), 12.0),
    (TUBE, (0.0, 4.0, 5.0, -1.0, math.pi), lambda p: member_tube(0.0, 4.0, 5.0, -1.0, math.pi, p), 12.0),
]


@pytest.mark.parametrize("k", range(len(SOLIDS)))
def test_distances_against_ray_marching(k):
    stype, prm, member, ext = SOLIDS[k]
    rng = np.random.default_rng(100 + k)
    n = 400
    p = rng.uniform(-ext, ext, size=(n, 3))
    if stype == TUBE and prm[1] > 100:      # put the points near the thin sector
        p = np.stack([rng.uniform(150, 450, n), rng.uniform(-80, 80, n), rng.uniform(-60, 60, n)], axis=1)
    v = unit(rng, n)
    # aim half of the rays at a random interior-ish point so that many of them hit
    aim = p.copy()
    if stype == BOX:
        aim = rng.uniform(-1, 1, size=(n, 3)) * np.asarray(prm[:3])
    else:
        rr = rng.uniform(prm[0], prm[1], n); aa = prm[3] + rng.uniform(0, min(prm[4], 2 * math.pi), n)
        aim = np.stack([rr * np.cos(aa), rr * np.sin(aa), rng.uniform(-prm[2], prm[2], n)], axis=1)
    d = aim - p; nd = np.linalg.norm(d, axis=1, keepdims=True)
    v[: n // 2] = (d / nd)[: n // 2]
    inside = member(p)
    cls = oracle.solid_eval(stype, prm, TOL, "inside", p)
    assert np.array_equal(cls == 0, inside)            # random points are never on a surface
    din = oracle.solid_eval(stype, prm, TOL, "dist_in", p, v)
    dout = oracle.solid_eval(stype, prm, TOL, "dist_out", p, v)
    tmax = 4 * ext
    checked = 0
    for i in range(n):
        t = march(member, p[i], v[i], tmax)
        got = dout[i] if inside[i] else din[i]
        if math.isinf(t) or math.isinf(got):
            if math.isinf(t) != math.isinf(got):
                # a crossing the march cannot see (chord shorter than its step) or a graze within tolerance
                fine = march(member, p[i], v[i], tmax, n=400001)
                assert math.isinf(fine) == math.isinf(got) or abs(fine - got) < 1e-6, (i, t, fine, got)
            continue
        if abs(t - got) > 1e-7 * max(1.0, t):
            fine = march(member, p[i], v[i], tmax, n=400001)   # the coarse march skipped a thin chord
            assert abs(fine - got) < 1e-7 * max(1.0, fine), (i, t, fine, got)
        checked += 1
    assert checked > n // 3


@pytest.mark.parametrize("k", [0, 1])
def test_convex_round_trip(k):
    stype, prm, member, ext = SOLIDS[k]
    rng = np.random.default_rng(7 + k)
    n = 2000
    p = rng.uniform(-1, 1, size=(n, 3)) * (np.asarray(prm[:3]) if stype == BOX else np.array([2.5, 2.5, 4.5]))
    v = unit(rng, n)
    t = oracle.solid_eval(stype, prm, TOL, "dist_out", p, v)
    s = rng.uniform(0.1, 3.0, n)
    q = p + (t + s)[:, None] * v
    back = oracle.solid_eval(stype, prm, TOL, "dist_in", q, -v)
    assert np.max(np.abs(back - s)) < 1e-11


def test_fp32_agrees_with_fp64_on_distances():
    rng = np.random.default_rng(5)
    for stype, prm, member, ext in SOLIDS[:3]:
        p = rng.uniform(-ext, ext, size=(3000, 3)).astype(np.float32)
        v = unit(rng, 3000).astype(np.float32)
        tol32 = float(np.float32(ext * 2.0 ** -18))
        a = oracle.solid_eval(stype, prm, tol32, "dist_in", p, v, precision=32)
        b = oracle.solid_eval(stype, prm, tol32, "dist_in", p.astype(np.float64), v.astype(np.float64), precision=64)
        fin = np.isfinite(a) & np.isfinite(b)
        assert np.mean(np.isfinite(a) == np.isfinite(b)) > 0.995
        assert np.max(np.abs(a[fin] - b[fin]) / np.maximum(b[fin], 1.0)) < 2e-4


def test_unsupported_solids_are_rejected():
    with pytest.raises(RuntimeError):
        oracle.solid_eval(TUBE, (0.0, 1.0, 1.0, 0.0, 4.0), TOL, "inside", [[0.0, 0, 0]])   # pi < dphi < 2pi
    with pytest.raises(RuntimeError):
        oracle.solid_eval(5, (1.0, 1.0, 1.0), TOL, "inside", [[0.0, 0, 0]])
