"""Pins for the oracle's orb solid and for the paper's own benchmark: Algorithm 1 with attenuation only
(Eq. 9) on the "Spheres" geometry with the "Random" and "Regular" particle sets
(PAPER.md L152-160).

Nothing here calls the navigator to make its expectations: the orb is pinned to closed forms and to dense ray marching
of the set |p| <= r, and the free paths to a closed form written out in numpy -- every ray from the centre is
intersected analytically with every ball, the chords are sorted and the optical depth mu_Al * length is accumulated
until it reaches Y (Eq. 5-8)."""
import math

import numpy as np
import pytest

import oracle
from paper_1209_5235_b200 import workloads as W

TOL = 1e-9
ORB = 2


def unit(rng, n):
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


# ---- orb ----------------------------------------------------------------------------------------------
def test_orb_inside_classification():
    r = 100.0
    p = np.array([[0, 0, 0], [99.0, 0, 0], [0, 100.0, 0], [0, 0, 100.0 + 4e-10], [0, 0, 100.0 + 6e-10], [60.0, 80.0, 0.0], [101.0, 0, 0]])
    got = oracle.solid_eval(ORB, [r], TOL, "inside", p)
    assert got.tolist() == [0, 0, 1, 1, 2, 1, 2]


def test_orb_radial_and_chord_closed_forms():
    rng = np.random.default_rng(3)
    r = 70.0
    n = 2000
    u = unit(rng, n)
    rho = rng.uniform(0, r * 0.999, n)
    p = u * rho[:, None]
    # radial rays from an inner point: outward r - rho, inward r + rho
    assert np.allclose(oracle.solid_eval(ORB, [r], TOL, "dist_out", p, u), r - rho, rtol=1e-13, atol=1e-11)
    assert np.allclose(oracle.solid_eval(ORB, [r], TOL, "dist_out", p, -u), r + rho, rtol=1e-13, atol=1e-11)
    # from outside with impact parameter b: entry at sqrt(d^2 - b^2) - sqrt(r^2 - b^2), miss when b > r
    d = rng.uniform(r * 1.01, 5 * r, n)
    v = unit(rng, n)
    q = -v * d[:, None]                                   # ray through the centre
    assert np.allclose(oracle.solid_eval(ORB, [r], TOL, "dist_in", q, v), d - r, rtol=1e-13, atol=1e-11)
    e = np.cross(v, unit(rng, n)); e /= np.linalg.norm(e, axis=1, keepdims=True)
    b = rng.uniform(0, 1.5 * r, n)
    q2 = q + e * b[:, None]
    want = np.where(b < r, d - np.sqrt(np.maximum(r * r - b * b, 0)), np.inf)
    got = oracle.solid_eval(ORB, [r], TOL, "dist_in", q2, v)
    near = np.abs(b - r) < 1e-3                           # grazing band: tolerance rules decide
    assert np.allclose(got[~near], want[~near], rtol=1e-12, atol=1e-9)
    # moving away: never enters
    assert np.all(np.isinf(oracle.solid_eval(ORB, [r], TOL, "dist_in", q, -v)))
    # chord through the ball = dist_out from the entry point
    ent = q2[b < 0.99 * r] + v[b < 0.99 * r] * got[b < 0.99 * r][:, None]
    chord = oracle.solid_eval(ORB, [r], TOL, "dist_out", ent, v[b < 0.99 * r])
    assert np.allclose(chord, 2 * np.sqrt(r * r - b[b < 0.99 * r] ** 2), rtol=1e-9, atol=1e-7)


def test_orb_ray_marching_and_round_trip():
    rng = np.random.default_rng(5)
    r = 40.0

    def member(p):
        return np.sum(p * p, axis=-1) <= r * r

    def march(p, v, tmax, n=20001):
        ts = np.linspace(0.0, tmax, n)
        m = member(p[None, :] + ts[:, None] * v[None, :])
        ch = np.nonzero(m[1:] != m[:-1])[0]
        if len(ch) == 0:
            return math.inf
        lo, hi, m0 = ts[ch[0]], ts[ch[0] + 1], m[ch[0]]
        for _ in range(60):
            mid = 0.5 * (lo + hi)
            if member((p + mid * v)[None, :])[0] == m0:
                lo = mid
            else:
                hi = mid
        return 0.5 * (lo + hi)

    n = 300
    pin = unit(rng, n) * rng.uniform(0, 0.98 * r, n)[:, None]
    pout = unit(rng, n) * rng.uniform(1.05 * r, 3 * r, n)[:, None]
    v = unit(rng, n)
    dout = oracle.solid_eval(ORB, [r], TOL, "dist_out", pin, v)
    din = oracle.solid_eval(ORB, [r], TOL, "dist_in", pout, v)
    for i in range(n):
        assert abs(dout[i] - march(pin[i], v[i], 2.2 * r)) < 1e-6
        m = march(pout[i], v[i], 5 * r)
        if not math.isinf(m):                             # (a miss, or a graze below the marching resolution, pins nothing)
            assert abs(din[i] - m) < 1e-6
        else:
            b = np.linalg.norm(np.cross(pout[i], v[i]))   # impact parameter: a clear miss must be +inf
            if b > r + 1e-3 or pout[i] @ v[i] > 0:
                assert math.isinf(din[i])
    # round trip (convex solid): leave by t, step s beyond, come back: DistanceToIn(-v) = s
    s = rng.uniform(0.1, 30.0, n)
    back = pin + v * (dout + s)[:, None]
    assert np.allclose(oracle.solid_eval(ORB, [r], TOL, "dist_in", back, -v), s, rtol=1e-9, atol=1e-8)


# ---- free paths: closed form in numpy ------------------------------------------------------------------
def analytic_free_paths(centres, radius, mu, d, Y, half):
    """T for rays from the origin (outside every ball): sorted chords, mu * length accumulated until Y (Eq. 7)."""
    n = d.shape[0]
    T = np.full(n, np.inf)
    for i in range(n):
        tca = centres @ d[i]
        d2 = np.einsum("ij,ij->i", centres, centres) - tca * tca
        hit = (d2 < radius * radius) & (tca > 0)
        thc = np.sqrt(radius * radius - d2[hit])
        t0, t1 = tca[hit] - thc, tca[hit] + thc
        texit = np.min(np.where(d[i] != 0, (np.sign(d[i]) * half) / np.where(d[i] != 0, d[i], 1), np.inf))   # world box exit
        order = np.argsort(t0)
        S = 0.0
        for a, b in zip(t0[order], t1[order]):
            if a >= texit:
                break
            b = min(b, texit)
            if S + mu * (b - a) >= Y[i]:
                T[i] = a + (Y[i] - S) / mu
                break
            S += mu * (b - a)
    return T


def sphere_centres(n_side=20, cube=5000.0):
    pitch = cube / n_side
    c = -cube / 2 + pitch * (np.arange(n_side) + 0.5)
    iz, iy, ix = np.meshgrid(c, c, c, indexing="ij")
    return np.stack([ix.reshape(-1), iy.reshape(-1), iz.reshape(-1)], axis=1)


@pytest.mark.parametrize("which", ["random", "regular"])
def test_free_path_equals_sorted_chord_closed_form(which):
    geom = W.spheres_geometry()
    og = oracle.OracleGeometry(geom)
    if which == "random":
        pos, d, Y = W.random_particles(1500, seed=21)
    else:
        pos, d, Y = W.regular_particles(50, 30, pixel=33.0)
    mu = 2.699 * W.MU_MASS_AL_1MEV / 10.0                  # 1/mm  (Eq. 9)
    T, ns = og.free_path(pos, d, Y, W.MU_MASS_AL_1MEV, 64)
    want = analytic_free_paths(sphere_centres(), 100.0, mu, d.astype(np.float64), Y.astype(np.float64), 2500.0)
    both_inf = np.isinf(T) & np.isinf(want)
    assert np.array_equal(np.isinf(T), np.isinf(want))
    assert np.allclose(T[~both_inf], want[~both_inf], rtol=1e-10, atol=1e-7)
    assert both_inf.sum() > 0 and (~both_inf).sum() > 100
    assert ns.min() >= 1 and ns.max() > 3
    # the voxel-accelerated locate changes nothing
    T2, ns2 = og.free_path(pos, d, Y, W.MU_MASS_AL_1MEV, 64, use_grid=False)
    assert np.array_equal(T, T2) and np.array_equal(ns, ns2)


def test_free_path_in_one_homogeneous_ball_is_y_over_mu():
    """Eq. 5 with constant mu: T = Y / mu exactly (up to rounding) while the particle stays inside."""
    b = W._Builder("one_ball")
    world = b.place(-1, b.box(1000, 1000, 1000), "vacuum")
    b.place(world, b.orb(900.0), "aluminium")
    og = oracle.OracleGeometry(b.finish())
    rng = np.random.default_rng(2)
    n = 500
    d = unit(rng, n); pos = np.zeros((n, 3)); Y = rng.exponential(1.0, n)
    mu = 2.699 * W.MU_MASS_AL_1MEV / 10.0
    T, ns = og.free_path(pos, d, Y, W.MU_MASS_AL_1MEV, 64)
    inside = Y / mu < 900.0
    assert np.allclose(T[inside], Y[inside] / mu, rtol=1e-14)
    assert np.all(np.isinf(T[~inside])) and (ns[inside] == 1).all()
    # survival fraction beyond x follows exp(-mu x)  (Eq. 2)
    x = 300.0
    frac = np.mean(T > x)
    assert abs(frac - math.exp(-mu * x)) < 4 * math.sqrt(math.exp(-mu * x) * (1 - math.exp(-mu * x)) / n)


def test_free_path_fp32_tracks_fp64():
    geom = W.spheres_geometry(n_side=6, cube=1500.0, radius=100.0)
    og = oracle.OracleGeometry(geom)
    pos, d, Y = W.random_particles(3000, seed=4, dtype=np.float32)
    T32, _ = og.free_path(pos, d, Y, W.MU_MASS_AL_1MEV, 32)
    T64, _ = og.free_path(pos.astype(np.float64), d.astype(np.float64), Y.astype(np.float64), W.MU_MASS_AL_1MEV, 64)
    fin = np.isfinite(T32) & np.isfinite(T64)
    assert (np.isfinite(T32) == np.isfinite(T64)).mean() > 0.999
    assert np.allclose(T32[fin], T64[fin], rtol=2e-5, atol=5e-3)
