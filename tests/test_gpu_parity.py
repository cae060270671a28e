"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Bars (BASELINE.json north_star): locate / next-volume indices bit-exact; ComputeStep
distances bit-exact against the same-precision oracle (canonical arithmetic), and fp32 against the fp64
oracle within 1e-5 relative or 1e-6 mm where fp32 can represent that (reading 10: the failing
fraction is printed and must stay below 2 %, the failures are bounded in ulp32 of the largest coordinate
involved -- 99.9 % quantile <= 32, maximum < 0.05 mm); >= 99.9 % identical histories in fp64; per-volume
edep within 1e-3 of the aggregate."""
import math

import numpy as np
import pytest

import oracle
from paper_1209_5235_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available()
    from paper_1209_5235_b200 import build, binding
    build.build()
    return binding


def unit(rng, n):
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def cuda(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


GEOMS = {
    "slab": lambda: W.slab_geometry(1),
    "phantom12": lambda: W.phantom_geometry(12, 2.0, seed=3, world_half=150.0),
    "calorimeter": lambda: W.calorimeter_geometry(8),
    "detector": lambda: W.detector_geometry(seed=4, n_phi=16, n_z=8, barrels=((200, 400), (450, 650))),
    "lattice": lambda: W.lattice_geometry(4, seed=7),
    "mixed": lambda: W.mixed_solids_geometry(),          # boxes, tubes, cones, balls, rotated, nested balls
    "cmslike": lambda: W.cms_like_geometry(),            # six-level detector hierarchy of all four solids (8(f) NEXT-2)
}


def deep_centres(geom, nodes):
    """Global positions of the origins of `nodes` (composition of the placement translations / rotations, test-side numpy)."""
    out = []
    for i in nodes:
        x = np.zeros(3)
        while i > 0:
            tr = geom.transforms[geom.placements[i, 3]]
            x = tr[:9].reshape(3, 3) @ x + tr[9:]
            i = geom.placements[i, 0]
        out.append(x)
    return np.array(out)


def query_points(geom, rng, n):
    h = W.world_half_extent(geom)
    p = rng.uniform(-1, 1, size=(n, 3)) * h * 1.02
    s = int(geom.placements[1, 1]); q = geom.solid_params[s]
    ext = np.array([q[0], q[1], q[2]]) if geom.solid_type[s] == 0 else np.array([q[1], q[1], q[2]])
    c = geom.transforms[int(geom.placements[1, 3]), 9:]
    if geom.name.startswith("lattice") or geom.name.startswith("mixed"):
        ext, c = h * 0.9, np.zeros(3)
    if geom.name.startswith("cmslike"):                 # half of the points around the deepest branch (crystal / cone / ball)
        deep = np.nonzero(geom.solid_type[geom.placements[:, 1]] == 3)[0]
        deep = deep[geom.placements[deep, 0] > 0]       # the cones inside the crystals (the end caps hang off the world)
        cg = deep_centres(geom, deep)
        p[: n // 2] = cg[rng.integers(0, len(cg), n // 2)] + rng.normal(size=(n // 2, 3)) * 60.0
        return p
    p[: n // 2] = c + rng.uniform(-1, 1, size=(n // 2, 3)) * ext * 1.05
    if geom.name.startswith("config3"):                 # points exactly on voxel faces / edges / corners
        k = n // 8
        p[:k] = np.round(p[:k] / 2.0) * 2.0
        p[k:2 * k, 2] = np.round(p[k:2 * k, 2] / 2.0) * 2.0
    return p


@pytest.mark.parametrize("name", list(GEOMS))
@pytest.mark.parametrize("precision", [64, 32])
def test_nav_bit_exact(B, name, precision):
    geom = GEOMS[name]()
    og = oracle.OracleGeometry(geom); g = B.Geometry(geom)
    rng = np.random.default_rng(101)
    n = 100003                                          # several blocks and a ragged tail
    R = np.float64 if precision == 64 else np.float32
    p = query_points(geom, rng, n).astype(R); v = unit(rng, n).astype(R)
    tp, tv = cuda(p), cuda(v)
    vol = B.nav_locate(g, tp, tv).cpu().numpy()
    ref = og.locate(p, v, precision)
    assert np.array_equal(vol, ref)
    assert np.array_equal(B.nav_locate(g, tp, None).cpu().numpy(), og.locate(p, None, precision))
    step, nxt = B.nav_compute_step(g, tp, tv, cuda(ref))
    rstep, rnxt = og.compute_step(p, v, ref, None, precision)
    assert np.array_equal(nxt.cpu().numpy(), rnxt)
    assert np.array_equal(step.cpu().numpy(), rstep)    # canonical arithmetic: 0 ulp, hence <= 1e-12 relative
    # with a step limit
    ms = rng.uniform(0, 300, n).astype(R)
    step, nxt = B.nav_compute_step(g, tp, tv, cuda(ref), cuda(ms))
    rstep, rnxt = og.compute_step(p, v, ref, ms, precision)
    assert np.array_equal(nxt.cpu().numpy(), rnxt) and np.array_equal(step.cpu().numpy(), rstep)
    assert len(np.unique(ref)) > min(4, geom.n_places - 1) and (ref == -1).any()


@pytest.mark.parametrize("name", list(GEOMS))
@pytest.mark.parametrize("precision", [64, 32])
def test_safety_bit_exact(B, name, precision):
    """isotropic safety distance -- canonical arithmetic only (+ - * sqrt max |.|), so 0 ulp against the
    oracle's linear scan; and no ComputeStep of the CUDA path from the same point is shorter."""
    geom = GEOMS[name]()
    og = oracle.OracleGeometry(geom); g = B.Geometry(geom)
    rng = np.random.default_rng(202)
    n = 20011 if name == "phantom12" else 50021         # several blocks and a ragged tail (the oracle scans every daughter)
    R = np.float64 if precision == 64 else np.float32
    p = query_points(geom, rng, n).astype(R); v = unit(rng, n).astype(R)
    tp, tv = cuda(p), cuda(v)
    vol = B.nav_locate(g, tp, None)
    ref_vol = og.locate(p, None, precision)
    assert np.array_equal(vol.cpu().numpy(), ref_vol)
    s = B.nav_compute_safety(g, tp, vol).cpu().numpy()
    ref = og.compute_safety(p, ref_vol, precision)
    assert np.array_equal(s, ref)
    assert np.all(s[ref_vol < 0] == 0) and (s > 0).mean() > 0.5 and np.isfinite(s).all()
    # arbitrary (wrong) volumes are still the same function on both sides; -1 and out-of-range give 0
    wrong = rng.integers(-1, geom.n_places, n).astype(np.int32)
    assert np.array_equal(B.nav_compute_safety(g, tp, cuda(wrong)).cpu().numpy(), og.compute_safety(p, wrong, precision))
    # lower bound of every step from the same point (the volume a step starts in depends on the direction on surfaces)
    vol_d = B.nav_locate(g, tp, tv)
    step, _ = B.nav_compute_step(g, tp, tv, vol_d)
    same = (vol_d == vol).cpu().numpy() & (ref_vol >= 0)
    slack = 1e-9 if precision == 64 else 1e-3
    assert np.all(step.cpu().numpy()[same] >= s[same] - slack)
    assert B.nav_compute_safety(g, tp[:0], vol[:0]).numel() == 0


def test_voxel_walk_matches_linear_scan_oracle(B):
    """The sparse lattice puts 64 solids in a voxelised vacuum world: ComputeStep from the mother walks the
    grid; the oracle's ComputeStep is the plain linear scan over all daughters."""
    geom = GEOMS["lattice"]()
    og = oracle.OracleGeometry(geom); g = B.Geometry(geom)
    assert g.voxel_info()["grids"] >= 1
    rng = np.random.default_rng(5)
    n = 50000
    p = rng.uniform(-1, 1, size=(n, 3)) * W.world_half_extent(geom); v = unit(rng, n)
    for precision in (64, 32):
        R = np.float64 if precision == 64 else np.float32
        P, V = p.astype(R), v.astype(R)
        ref = og.locate(P, V, precision, use_grid=False)
        in_world = ref == 0
        assert in_world.sum() > n // 3
        step, nxt = B.nav_compute_step(g, cuda(P), cuda(V), cuda(ref))
        rstep, rnxt = og.compute_step(P, V, ref, None, precision, use_grid=False)
        assert np.array_equal(step.cpu().numpy(), rstep) and np.array_equal(nxt.cpu().numpy(), rnxt)
        assert (rnxt[in_world] > 0).sum() > 1000         # many rays do hit a daughter through the walk


def test_points_in_the_tolerance_band_of_voxel_faces(B):
    """The voxel grid lists a daughter only in the cells its own box overlaps and probes the neighbouring cells
    when the point is within 1.25 delta of a cell boundary.  Points at k * delta from voxel faces, edges and
    corners (k on both sides of every threshold in that argument) must locate and step exactly as the oracle."""
    geom = GEOMS["phantom12"]()
    og = oracle.OracleGeometry(geom); g = B.Geometry(geom)
    rng = np.random.default_rng(77)
    n = 60000
    for precision in (32, 64):
        R = np.float64 if precision == 64 else np.float32
        delta = g.tolerance(precision) / 2
        base = np.round(rng.uniform(-12, 12, size=(n, 3)) / 2.0) * 2.0              # voxel corners (2 mm pitch)
        free = rng.uniform(-12, 12, size=(n, 3))
        on = rng.integers(0, 2, size=(n, 3)).astype(bool); on[:, 0] |= ~on.any(axis=1)   # which coordinates sit on a face
        k = rng.choice([-3.0, -2.0, -1.3, -1.2, -1.0, -0.9, -0.5, 0.0, 0.5, 0.9, 1.0, 1.2, 1.3, 2.0, 3.0], size=(n, 3))
        p = np.where(on, base + k * delta, free).astype(R)
        v = unit(rng, n).astype(R)
        v[: n // 4] = np.where(on[: n // 4], 0.0, v[: n // 4]).astype(R)            # some rays run along the faces
        nz = np.linalg.norm(v, axis=1) == 0
        v[nz] = np.array([0, 0, 1], R)
        v = (v / np.linalg.norm(v, axis=1, keepdims=True)).astype(R)
        tp, tv = cuda(p), cuda(v)
        ref = og.locate(p, v, precision)
        assert np.array_equal(B.nav_locate(g, tp, tv).cpu().numpy(), ref)
        assert np.array_equal(B.nav_locate(g, tp, None).cpu().numpy(), og.locate(p, None, precision))
        step, nxt = B.nav_compute_step(g, tp, tv, cuda(ref))
        rstep, rnxt = og.compute_step(p, v, ref, None, precision)
        assert np.array_equal(nxt.cpu().numpy(), rnxt) and np.array_equal(step.cpu().numpy(), rstep)


def test_steps_that_end_near_the_edges_of_barrel_sectors(B):
    """Sibling hints (store.h NODE_HINT): a photon that leaves a barrel sector through one z or phi face, farther than two
    probe distances from its other faces, is relocated by testing only the sibling across that face.  Rays are aimed at points
    on the z faces, the phi planes and the radial surfaces of sectors, at offsets of 0 .. 3 probe distances from a SECOND face
    (on both sides of the threshold of that rule, and onto edges and corners), so the shortcut and the general search meet;
    step lengths and volumes entered must be the oracle's bit for bit."""
    geom = GEOMS["detector"]()                  # 2 barrels x 16 phi x 8 z sectors, r 200-400 and 450-650, hz 1600
    og = oracle.OracleGeometry(geom); g = B.Geometry(geom)
    rng = np.random.default_rng(91)
    n = 60000
    dphi, hz_s = 2 * np.pi / 16, 1600.0 / 8
    for precision in (32, 64):
        R = np.float64 if precision == 64 else np.float32
        probe = 1.25 * g.tolerance(precision) / 2 + 4 * 2000.0 * (2.0 ** -23 if precision == 32 else 2.0 ** -52)
        k = rng.choice([0.0, 0.5, 1.0, 1.9, 2.1, 3.0, 30.0], size=(n, 3)) * rng.choice([-1.0, 1.0], size=(n, 3)) * probe
        barrel = rng.integers(0, 2, n)
        rlo, rhi = np.where(barrel == 0, 200.0, 450.0), np.where(barrel == 0, 400.0, 650.0)
        # target point: on a z face (kind 0), a phi plane (1) or a radial surface (2); the other two coordinates are either
        # free or sit at an offset k from another face
        kind = rng.integers(0, 3, n)
        near2 = rng.random((n, 2)) < 0.6
        r_face = np.where(rng.random(n) < 0.5, rlo, rhi)
        z_face = -1600.0 + hz_s * 2 * rng.integers(0, 9, n)
        phi_face = dphi * (rng.integers(0, 16, n) + 0.5)                  # sector j spans (j - 1/2, j + 1/2) dphi
        r = np.where(kind == 2, r_face + k[:, 0], np.where(near2[:, 0], r_face + k[:, 0], rng.uniform(rlo + 1, rhi - 1)))
        z = np.where(kind == 0, z_face + k[:, 1], np.where(near2[:, 1], z_face + k[:, 1], rng.uniform(-1590, 1590, n)))
        phi = np.where(kind == 1, phi_face + k[:, 2] / r, np.where(np.where(kind == 0, near2[:, 1], near2[:, 0]), phi_face + k[:, 2] / r, rng.uniform(0, 2 * np.pi, n)))
        target = np.stack([r * np.cos(phi), r * np.sin(phi), z], axis=1)
        v = unit(rng, n)
        origin = target - v * rng.uniform(1.0, 30.0, size=(n, 1))
        p, v = origin.astype(R), v.astype(R)
        v = (v / np.linalg.norm(v.astype(np.float64), axis=1, keepdims=True)).astype(R)
        tp, tv = cuda(p), cuda(v)
        ref = og.locate(p, v, precision)
        assert np.array_equal(B.nav_locate(g, tp, tv).cpu().numpy(), ref)
        step, nxt = B.nav_compute_step(g, tp, tv, cuda(ref))
        rstep, rnxt = og.compute_step(p, v, ref, None, precision)
        assert np.array_equal(nxt.cpu().numpy(), rnxt) and np.array_equal(step.cpu().numpy(), rstep)
        # a second query from where the first step ended: points on (or within rounding of) the boundary just reached
        alive = np.isfinite(rstep) & (rnxt >= 0)
        p2 = (p[alive] + rstep[alive, None] * v[alive]).astype(R)
        v2 = v[alive]
        ref2 = og.locate(p2, v2, precision)
        assert np.array_equal(B.nav_locate(g, cuda(p2), cuda(v2)).cpu().numpy(), ref2)
        step2, nxt2 = B.nav_compute_step(g, cuda(p2), cuda(v2), cuda(ref2))
        rstep2, rnxt2 = og.compute_step(p2, v2, ref2, None, precision)
        assert np.array_equal(nxt2.cpu().numpy(), rnxt2) and np.array_equal(step2.cpu().numpy(), rstep2)
        in_sector = np.isin(ref, np.arange(3, geom.n_places))            # world = 0, barrels = 1, 2
        assert in_sector.mean() > 0.5 and (rnxt[in_sector] >= 3).mean() > 0.3


@pytest.mark.parametrize("name", ["detector", "cmslike", "mixed"])
def test_locate_level_by_level_every_tile_width(B, name):
    """gn_nav_locate on general geometries walks the placement tree level by level inside each warp, on tiles of 32 ... 256
    queries per warp chosen from the batch size (locate_levels_kernel): every tile width, single queries,
    ragged tiles and ragged last warps against the oracle, element by element, with and without directions."""
    geom = GEOMS[name]()
    og = oracle.OracleGeometry(geom); g = B.Geometry(geom)
    rng = np.random.default_rng(77)
    warps = 148 * 64
    sizes = [1, 31, 33, 255, 257, warps * 32 + 5, warps * 40 + 3, warps * 100 + 7, warps * 130 + 1, warps * 170 - 3, warps * 200 + 1, warps * 250 + 3]
    n_max = max(sizes)
    p = query_points(geom, rng, n_max).astype(np.float32); v = unit(rng, n_max).astype(np.float32)
    ref = og.locate(p, v, 32); ref0 = og.locate(p, None, 32)
    assert (ref == -1).any() and len(np.unique(ref)) > 4
    tp, tv = cuda(p), cuda(v)
    for n in sizes:
        o = int(rng.integers(0, n_max - n + 1))                      # a different slice of the same queries each time
        assert np.array_equal(B.nav_locate(g, tp[o:o + n], tv[o:o + n]).cpu().numpy(), ref[o:o + n]), n
        assert np.array_equal(B.nav_locate(g, tp[o:o + n], None).cpu().numpy(), ref0[o:o + n]), n
    pd = p[:warps * 40 + 3].astype(np.float64); vd = v[:warps * 40 + 3].astype(np.float64)
    assert np.array_equal(B.nav_locate(g, cuda(pd), cuda(vd)).cpu().numpy(), og.locate(pd, vd, 64))


def test_nav_edge_cases(B):
    import torch
    geom = GEOMS["slab"]()
    g = B.Geometry(geom)
    for dt in (torch.float32, torch.float64):
        e = torch.empty((0, 3), dtype=dt, device="cuda")
        assert B.nav_locate(g, e, e).numel() == 0
        s, n = B.nav_compute_step(g, e, e, torch.empty(0, dtype=torch.int32, device="cuda"))
        assert s.numel() == 0 and n.numel() == 0
        p = torch.tensor([[0, 0, -500.0], [0, 0, 0], [600.0, 0, 0], [0, 0, -500.0]], dtype=dt, device="cuda")
        v = torch.tensor([[0, 0, 1.0], [0, 0, 1.0], [0, 0, 1.0], [0, 0, -1.0]], dtype=dt, device="cuda")
        vol = B.nav_locate(g, p, v).cpu().tolist()
        assert vol[0] == 0 and vol[1] >= 1 and vol[2] == -1 and vol[3] == -1
        assert B.nav_locate(g, p, None).cpu().tolist()[3] == 0              # surface counts as inside without a direction
        vin = torch.tensor([0, -1, 99999, 0], dtype=torch.int32, device="cuda")
        s, n = B.nav_compute_step(g, p, v, vin)
        s, n = s.cpu().tolist(), n.cpu().tolist()
        assert s[0] == 450.0 and n[0] == 1
        assert math.isinf(s[1]) and n[1] == -1 and math.isinf(s[2]) and n[2] == -1
        s, n = B.nav_compute_step(g, p[:1], v[:1], vin[:1], torch.tensor([449.0], dtype=dt, device="cuda"))
        assert math.isinf(s.item()) and n.item() == 0
        s, n = B.nav_compute_step(g, p[:1], v[:1], vin[:1], torch.tensor([450.0], dtype=dt, device="cuda"))
        assert s.item() == 450.0 and n.item() == 1                           # tie -> boundary
    with pytest.raises(B.GammaNavError):
        B.nav_locate(g, torch.zeros((4, 3)), None)                           # host tensor: refused, no CPU path
    with pytest.raises(B.GammaNavError):
        B.Geometry(W.Geometry(geom.materials, geom.solid_type, geom.solid_params, geom.placements[::-1].copy(), geom.transforms))


def test_fp32_distances_against_fp64_oracle(B):
    """C10: fp32 GPU vs fp64 oracle on the same (rounded) geometry and queries: |d| <= 1e-5 d or 1e-6 mm.
    The literal criterion is not attainable for every query in fp32 (C10 itself says so: the inputs carry
    representation error of a few ulp32 of the largest coordinate, amplified by 1 / sin(incidence) on near-tangent
    cylinder hits -- DESIGN.md reading 10).  Asserted here: at least 98 % of the queries meet the literal criterion, the
    99.9 % quantile of error / ulp32(largest coordinate involved) is <= 32, the largest error is < 0.05 mm, and the
    volumes agree on > 99.99 % of the queries.  The measured values are printed."""
    geom = GEOMS["detector"]()
    og = oracle.OracleGeometry(geom); g = B.Geometry(geom)
    rng = np.random.default_rng(9)
    n = 200000
    p = query_points(geom, rng, n).astype(np.float32); v = unit(rng, n).astype(np.float32)
    vol32 = B.nav_locate(g, cuda(p), cuda(v))
    step32, nxt32 = B.nav_compute_step(g, cuda(p), cuda(v), vol32)
    vol64 = og.locate(p.astype(np.float64), v.astype(np.float64), 64)
    agree = vol32.cpu().numpy() == vol64
    assert agree.mean() > 0.9999
    step64, nxt64 = og.compute_step(p.astype(np.float64), v.astype(np.float64), vol64, None, 64)
    s32 = step32.cpu().numpy().astype(np.float64)
    ok = agree & np.isfinite(step64) & np.isfinite(s32)
    d = np.abs(s32[ok] - step64[ok])
    passed = (d <= 1e-5 * step64[ok]) | (d <= 1e-6)
    scale = np.maximum(np.max(np.abs(p[ok]), axis=1).astype(np.float64), step64[ok])
    ulp = np.spacing(scale.astype(np.float32)).astype(np.float64)
    # failures are representation error of the fp32 inputs: a few ulp32 of the largest coordinate involved, amplified by
    # 1 / sin(incidence) on near-tangent hits of the cylinders (unbounded in principle, so bound a high quantile and the max)
    ratio = d / ulp
    print(f"fp32-vs-fp64 distance criterion: failing fraction {1 - passed.mean():.2e}, volume agreement {agree.mean():.6f}, "
          f"error/ulp32 median {np.median(ratio):.2f} p99.9 {np.quantile(ratio, 0.999):.1f} max {ratio.max():.1f} ({d.max():.2e} mm)")
    assert np.quantile(ratio, 0.999) <= 32 and d.max() < 0.05
    assert passed.mean() > 0.98


TRANSPORT_CASES = {
    "config1": lambda: (W.slab_geometry(1), W.slab_source(), 10000, 1),
    "calorimeter": lambda: (W.calorimeter_geometry(10), W.calorimeter_source(), 20000, 2),
    "phantom16": lambda: (W.phantom_geometry(16, 2.0, 3), W.phantom_source(16, half_angle_deg=0.8), 20000, 3),
    "detector": lambda: (W.detector_geometry(seed=4, n_phi=16, n_z=8, barrels=((200, 400), (450, 650))), W.detector_source(), 20000, 4),
    "lattice": lambda: (W.lattice_geometry(4, seed=7), W.Source(W.SRC_ISOTROPIC, (3.0, 2.0, 1.0), (0, 0, 1.0), W.E_LOGUNIFORM, 0.05, 20.0), 20000, 5),
    "cmslike": lambda: (W.cms_like_geometry(), W.Source(W.SRC_ISOTROPIC, (0.0, 0.0, 0.0), (0, 0, 1.0), W.E_LOGUNIFORM, 0.1, 1000.0), 20000, 6),
}


def compare_transport(B, geom, src, n, seed, precision, min_identical, opts=None, oracle_opts=None, allow_stuck=False):
    og = oracle.OracleGeometry(geom, **(oracle_opts or {})); g = B.Geometry(geom, **(opts or {}))
    got = B.transport_run(g, src, seed, n, precision, per_photon=True)
    ref = og.transport(src, seed, n, precision, per_photon=True)
    hg = got["hash"].cpu().numpy().view(np.uint64); ng = got["nsteps"].cpu().numpy().astype(np.uint32)
    same = (hg == ref["hash"]) & (ng == ref["nsteps"])
    ef = got["efinal"].cpu().numpy()
    same &= np.abs(ef - ref["efinal"]) <= (1e-9 if precision == 64 else 1e-4) * np.abs(ref["efinal"])
    edep = got["edep"].cpu().numpy()
    tot = ref["edep"].sum()
    assert same.mean() >= min_identical, same.mean()
    assert abs(edep.sum() - tot) <= 1e-3 * tot
    assert np.abs(edep - ref["edep"]).sum() <= (1e-3 if precision == 64 else 2e-2) * tot
    s, r = got["stats"], ref["stats"]
    assert s["n_photons"] == n and (allow_stuck or s["n_stuck"] <= max(1, n // 10 ** 6))
    book = edep.sum() + s["e_escaped"] + s["e_stuck"]
    assert abs(book / s["e_source"] - 1) < (1e-12 if precision == 64 else 2e-6)
    assert int(ng.sum()) == s["n_steps"]
    if same.mean() == 1.0:
        for k in ("n_steps", "n_compton", "n_pe", "n_pair", "n_cut", "n_escaped", "n_stuck"):
            assert s[k] == r[k], k
    return got, ref, same.mean()


@pytest.mark.parametrize("name", list(TRANSPORT_CASES))
def test_transport_fp64_histories_identical(B, name):
    geom, src, n, seed = TRANSPORT_CASES[name]()
    compare_transport(B, geom, src, n, seed, 64, 0.999)


@pytest.mark.parametrize("name", list(TRANSPORT_CASES))
def test_transport_fp32_aggregate(B, name):
    geom, src, n, seed = TRANSPORT_CASES[name]()
    # fp32: parity is on the aggregate (libm float functions differ between host and device); histories are
    # still overwhelmingly identical because both sides consume the same Philox draws in the same order
    got, ref, frac = compare_transport(B, geom, src, n, seed, 32, 0.97)
    print(f"{name} fp32 identical histories: {frac:.5f}")


def _layer_stack(axis, thicknesses=(2.0, 4.0, 6.0, 2.0), periods=6, half=150.0):
    """Layers of several thicknesses (multiples of the thinnest) stacked along `axis` in a mother box: the voxel grid's pitch is
    the thinnest layer, so the thin layers are regular voxels and the others regular slabs of 2 and 3 cells (store.h NODE_SLAB)."""
    from paper_1209_5235_b200.workloads import _Builder
    b = _Builder(f"layer_stack_axis{axis}")
    L = periods * sum(thicknesses)
    def dims(t):
        h = [half, half, half]; h[axis] = t / 2
        return h
    world = b.place(-1, b.box(400.0, 400.0, 400.0), "air")
    mh = [half, half, half]; mh[axis] = L / 2
    mother = b.place(world, b.box(*mh), "air")
    solids = [b.box(*dims(t)) for t in thicknesses]
    mats = ["lead", "scint", "iron", "water"]
    u = -L / 2
    for _ in range(periods):
        for k, t in enumerate(thicknesses):
            T = [0.0, 0.0, 0.0]; T[axis] = u + t / 2
            b.place(mother, solids[k], mats[k % len(mats)], T=tuple(T)); u += t
    return b.finish()


@pytest.mark.parametrize("schedule", ["tail", "wavefront"])
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_regular_slabs_along_every_axis(B, axis, precision, schedule):
    """The slab rule of the regular-voxel step kernel (nav.cuh regular_step<.., SLABS>): stacks along x, y and z whose layers
    are 1, 2 and 3 grid cells thick, entered obliquely so that photons cross layers both ways, leave through the sides (the
    general step) and change solid at every boundary.  Histories against the oracle as for every other geometry."""
    geom = _layer_stack(axis)
    d = [0.25, 0.15, 0.15]; d[axis] = 1.0
    o = [3.0, -2.0, 1.0]; o[axis] = -300.0
    src = W.Source(W.SRC_GAUSS_PENCIL, tuple(o), tuple(d), W.E_MONO, 3.0, 0.0, 8.0)
    # "tail": source pass + run-to-completion pass (20000 photons are below tail_photons); "wavefront": the voxel schedule's
    # voxel_pass / general_pass / interact_pass in short passes until a single photon is left
    opts = dict(steps_per_pass=3, tail_photons=1) if schedule == "wavefront" else None
    got, ref, frac = compare_transport(B, geom, src, 20000, 11 + axis, precision, 0.999 if precision == 64 else 0.97, opts=opts)
    assert got["stats"]["n_steps"] > 20000 * 10 and got["stats"]["n_escaped"] > 0 and (got["edep"].cpu().numpy()[2:] > 0).sum() >= 20


# ---- stuck guard (reading 7): the EV_STUCK branch on every schedule ----------------------------
def _big_water():
    from paper_1209_5235_b200.workloads import _Builder
    b = _Builder("big_water")
    b.place(-1, b.box(1e7, 1e7, 1e7), "water")
    return b.finish()


SCHEDULES = {"tail": {}, "wavefront": dict(steps_per_pass=2, tail_photons=1), "refill": dict(refill=1)}


@pytest.mark.parametrize("schedule", list(SCHEDULES))
@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("limit", [1, 3])
def test_stuck_guard_every_step_short(B, schedule, precision, limit):
    """The oracle's pinned construction (tests/test_oracle_hash_stuck.py): a 2e7 mm water world with tol = 1e6 mm, so every
    step is an interaction step shorter than delta and every photon not absorbed first is killed after `limit` steps, after
    that step's Compton scatter.  Hashes (event word STUCK), step counts, n_stuck and E_stuck must equal the oracle's."""
    n = 20000
    tol = {"tol64": 1e6} if precision == 64 else {"tol32": 1e6}
    src = W.Source(W.SRC_PENCIL, (0.0, 0.0, 0.0), (0.0, 0.0, 1.0), W.E_MONO, 1.0)
    got, ref, frac = compare_transport(B, _big_water(), src, n, 7, precision, 0.999 if precision == 64 else 0.97,
                                       opts=dict(stuck_limit=limit, **tol, **SCHEDULES[schedule]), oracle_opts=dict(stuck_limit=limit, **tol), allow_stuck=True)
    s, r = got["stats"], ref["stats"]
    assert s["n_stuck"] == r["n_stuck"] and s["n_stuck"] >= n - 200 and s["n_escaped"] == 0
    assert abs(s["e_stuck"] - r["e_stuck"]) <= (1e-9 if precision == 64 else 1e-4) * r["e_source"]
    assert abs(s["e_stuck"] - (s["e_source"] - float(got["edep"].sum()))) <= (1e-9 if precision == 64 else 1e-4) * s["e_source"]
    ns = got["nsteps"].cpu().numpy()
    assert ns.max() == limit and s["n_steps"] == int(ns.sum())


@pytest.mark.parametrize("schedule", list(SCHEDULES))
@pytest.mark.parametrize("limit", [1, 2])
def test_stuck_guard_zero_length_boundary_steps(B, schedule, limit):
    """A tolerance that is a fifth of the voxel size makes zero-length BOUNDARY steps common (entries snapped to 0, exits after
    a direction change next to a face): with stuck_limit 1 / 2 some photons are killed at boundaries.  Same histories,
    n_stuck and E_stuck as the oracle on every schedule."""
    geom = W.phantom_geometry(16, 2.0, 3); src = W.phantom_source(16, half_angle_deg=0.8)
    got, ref, frac = compare_transport(B, geom, src, 20000, 3, 64, 0.999, opts=dict(tol64=0.4, stuck_limit=limit, **SCHEDULES[schedule]),
                                       oracle_opts=dict(tol64=0.4, stuck_limit=limit), allow_stuck=True)
    s, r = got["stats"], ref["stats"]
    assert s["n_stuck"] == r["n_stuck"] and s["n_stuck"] > 20
    assert abs(s["e_stuck"] - r["e_stuck"]) <= 1e-9 * r["e_source"]
    assert s["n_pe"] + s["n_pair"] + s["n_cut"] + s["n_escaped"] + s["n_stuck"] == 20000


def test_stuck_limit_above_the_counter_width_is_refused(B):
    with pytest.raises(B.GammaNavError):
        B.Geometry(W.slab_geometry(1), stuck_limit=256)
    g = B.Geometry(W.slab_geometry(1), stuck_limit=255)
    assert g.n_places == 6


# ---- SURVEY 8(f) NEXT-3, the rest: Rayleigh scattering and the tabulated photoelectric coefficient -----------------------------
OPTIONAL_PHYSICS = {
    "rayleigh": dict(rayleigh=1),
    "rayleigh_strong": dict(rayleigh=1, sigma_r0=0.5),                    # coherent scattering as frequent as Compton in the light materials
    "pe_table": dict(pe_table_per_decade=256),
    "pe_table_k_edge": dict(pe_table_per_decade=64, pe_k_edge=1),
    "all": dict(rayleigh=1, pe_table_per_decade=128, pe_k_edge=1, secondaries=1),
}
PHYSICS_GEOMS = {
    "config1_300keV": lambda: (W.slab_geometry(1), W.Source(W.SRC_PENCIL, (0.0, 0.0, -500.0), (0.0, 0.0, 1.0), W.E_MONO, 0.3), 20000, 1),
    "phantom16": lambda: TRANSPORT_CASES["phantom16"](),
    "detector": lambda: TRANSPORT_CASES["detector"](),
}


@pytest.mark.parametrize("schedule", ["tail", "wavefront"])
@pytest.mark.parametrize("geo_name", list(PHYSICS_GEOMS))
@pytest.mark.parametrize("physics", list(OPTIONAL_PHYSICS))
def test_optional_physics_fp64_histories_identical(B, physics, geo_name, schedule):
    """gn_opts.rayleigh / pe_table_per_decade / pe_k_edge (readings 18, 19): same Philox draws, same process choice, same
    rejection loops as the oracle -> identical fp64 histories, event word 7 for a Rayleigh scatter, n_rayleigh equal."""
    geom, src, n, seed = PHYSICS_GEOMS[geo_name]()
    opts = OPTIONAL_PHYSICS[physics]
    got, ref, frac = compare_transport(B, geom, src, n, seed, 64, 0.999, opts=dict(opts, **SCHEDULES[schedule]), oracle_opts=opts)
    s, r = got["stats"], ref["stats"]
    assert s["n_rayleigh"] == r["n_rayleigh"]
    if not opts.get("rayleigh"):
        assert s["n_rayleigh"] == 0
    elif physics == "rayleigh_strong" or geo_name == "config1_300keV":       # (at 6 MeV the default cross-section is negligible)
        assert s["n_rayleigh"] > 20
    ends = s["n_pe"] + s["n_pair"] + s["n_cut"] + s["n_escaped"] + s["n_stuck"]
    assert ends == n + (2 * s["n_pair"] if opts.get("secondaries") else 0)


@pytest.mark.parametrize("physics", ["rayleigh_strong", "all"])
def test_optional_physics_fp32_and_refill(B, physics):
    geom, src, n, seed = PHYSICS_GEOMS["detector"]()
    opts = dict(OPTIONAL_PHYSICS[physics]); opts.pop("secondaries", None)
    got, ref, frac = compare_transport(B, geom, src, n, seed, 32, 0.97, opts=opts, oracle_opts=opts)
    assert abs(got["stats"]["n_rayleigh"] - ref["stats"]["n_rayleigh"]) <= 0.02 * ref["stats"]["n_rayleigh"] + 5
    got2, _, _ = compare_transport(B, geom, src, n, seed, 64, 0.999, opts=dict(opts, refill=1), oracle_opts=opts)
    assert got2["stats"]["n_rayleigh"] > 20


def test_optional_physics_leaves_the_default_untouched(B):
    """Options off: the new terms are exact zeros -- same hashes as a library that never heard of them (the oracle's default run)."""
    geom, src, n, seed = TRANSPORT_CASES["phantom16"]()
    a = B.transport_run(B.Geometry(geom), src, seed, n, 64, per_photon=True)
    b = B.transport_run(B.Geometry(geom, rayleigh=0, pe_table_per_decade=0, no_voxel_pass=1), src, seed, n, 64, per_photon=True)
    assert np.array_equal(a["hash"].cpu().numpy(), b["hash"].cpu().numpy()) and a["stats"]["n_rayleigh"] == 0
    with pytest.raises(B.GammaNavError):
        B.Geometry(geom, pe_table_per_decade=5000)


def _four_walls():
    from paper_1209_5235_b200.workloads import _Builder
    b = _Builder("four_walls")
    world = b.place(-1, b.box(1000.0, 1000.0, 1000.0), "vacuum")
    b.place(world, b.box(0.25, 0.25, 4.0), "lead")
    wall_x, wall_y = b.box(50.0, 150.0, 900.0), b.box(50.0, 50.0, 900.0)
    for solid, T in ((wall_x, (150.0, 0, 0)), (wall_x, (-150.0, 0, 0)), (wall_y, (0, 150.0, 0)), (wall_y, (0, -150.0, 0))):
        b.place(world, solid, "lead", T=T)
    return b.finish()


def _pencil(E):
    return W.Source(W.SRC_PENCIL, (0.0, 0.0, -500.0), (0.0, 0.0, 1.0), W.E_MONO, E)


SECONDARY_CASES = {
    # thick lead, 20 MeV: most primaries end in a pair event, so the annihilation photons need more than one batch of cap / 2 pairs
    "lead_slab_20MeV": lambda: (W.homogeneous_slab("lead", half=(200.0, 200.0, 10.0), world_half=1000.0), _pencil(20.0), 20000, 3),
    "four_walls": lambda: (_four_walls(), _pencil(8.0), 20000, 21),
    "calorimeter": lambda: (W.calorimeter_geometry(10), W.calorimeter_source(), 20000, 2),
    "phantom16_6MeV": lambda: (W.phantom_geometry(16, 2.0, 3), W.phantom_source(16, half_angle_deg=0.8), 20000, 3),
    "detector": lambda: (W.detector_geometry(seed=4, n_phi=16, n_z=8, barrels=((200, 400), (450, 650))), W.detector_source(), 20000, 4),
    "cmslike": lambda: (W.cms_like_geometry(), W.Source(W.SRC_ISOTROPIC, (0.0, 0.0, 0.0), (0, 0, 1.0), W.E_LOGUNIFORM, 0.1, 1000.0), 20000, 6),
}


@pytest.mark.parametrize("wavefront", [False, True])
@pytest.mark.parametrize("name", list(SECONDARY_CASES))
def test_secondary_photons_fp64_histories_identical(B, name, wavefront):
    """pair events leave two annihilation photons (Philox stream tags 1 / 2), followed in batches of
    their own after the primaries; per-photon hash and step count are sums over the primary and its secondaries.
    wavefront: tail_photons = 1 and short passes, so the secondaries go through the lean passes, the compaction and the
    interaction wavefront as well (default for this n: source pass, then one run-to-completion pass)."""
    geom, src, n, seed = SECONDARY_CASES[name]()
    opts = dict(secondaries=1, **(dict(steps_per_pass=5, tail_photons=1) if wavefront else {}))
    got, ref, _ = compare_transport(B, geom, src, n, seed, 64, 0.999, opts=opts, oracle_opts=dict(secondaries=1))
    s, r = got["stats"], ref["stats"]
    assert s["n_pair"] == r["n_pair"] and s["n_pair"] > 100
    # every photon ends exactly once; each pair event adds two photons
    assert s["n_pe"] + s["n_pair"] + s["n_cut"] + s["n_escaped"] + s["n_stuck"] == n + 2 * s["n_pair"]
    if name == "lead_slab_20MeV":
        assert 2 * s["n_pair"] > n                                   # more than one batch of annihilation photons


@pytest.mark.parametrize("name", ["lead_slab_20MeV", "calorimeter", "detector"])
def test_secondary_photons_fp32_aggregate(B, name):
    geom, src, n, seed = SECONDARY_CASES[name]()
    got, ref, frac = compare_transport(B, geom, src, n, seed, 32, 0.97, opts=dict(secondaries=1), oracle_opts=dict(secondaries=1))
    print(f"{name} fp32 with secondaries, identical histories: {frac:.5f}")


def test_secondary_photons_without_per_photon_outputs_and_below_threshold(B):
    geom, src, n, seed = SECONDARY_CASES["four_walls"]()
    g1 = B.Geometry(geom, secondaries=1)
    a = B.transport_run(g1, src, seed, n, 64, per_photon=True)
    b = B.transport_run(g1, src, seed, n, 64)                        # the lean (untracked) kernels
    assert np.allclose(a["edep"].cpu().numpy(), b["edep"].cpu().numpy(), rtol=1e-12, atol=1e-12)
    for k in ("n_steps", "n_compton", "n_pe", "n_pair", "n_cut", "n_escaped", "n_stuck", "n_photons"):
        assert a["stats"][k] == b["stats"][k], k
    # below 2 me c^2 the option changes nothing
    g0 = B.Geometry(geom)
    c = B.transport_run(g0, _pencil(1.0), seed, 5000, 64, per_photon=True)
    d = B.transport_run(g1, _pencil(1.0), seed, 5000, 64, per_photon=True)
    assert np.array_equal(c["hash"].cpu().numpy(), d["hash"].cpu().numpy())
    assert np.allclose(c["edep"].cpu().numpy(), d["edep"].cpu().numpy(), rtol=1e-12, atol=1e-12)      # fp64 atomics: order of the adds
    assert d["stats"]["n_pair"] == 0 and d["stats"]["n_steps"] == c["stats"]["n_steps"]
    # sharding by photon-id ranges (the multi-GPU split): secondaries follow their parents' ids
    lo = B.transport_run(g1, src, seed, 7000, 64, first_photon_id=0, per_photon=True)
    hi = B.transport_run(g1, src, seed, n - 7000, 64, first_photon_id=7000, per_photon=True)
    assert np.array_equal(np.concatenate([lo["hash"].cpu().numpy(), hi["hash"].cpu().numpy()]), a["hash"].cpu().numpy())
    assert np.array_equal(np.concatenate([lo["nsteps"].cpu().numpy(), hi["nsteps"].cpu().numpy()]), a["nsteps"].cpu().numpy())
    assert np.allclose((lo["edep"] + hi["edep"]).cpu().numpy(), a["edep"].cpu().numpy(), rtol=1e-12, atol=1e-12)
    # one photon (queue capacity 2): its pair, if any, still fits
    e = B.transport_run(g1, _pencil(8.0), seed, 1, 64, per_photon=True)
    r = oracle.OracleGeometry(geom, secondaries=1).transport(_pencil(8.0), seed, 1, 64, per_photon=True)
    assert int(e["hash"].cpu().numpy().view(np.uint64)[0]) == int(r["hash"][0])


@pytest.mark.parametrize("name", list(TRANSPORT_CASES))
def test_refill_kernel_same_histories(B, name):
    """SURVEY 8(f) NEXT-4 / PAPER.md L195: the persistent refill kernel (gn_opts.refill) follows the same photons with the
    same Philox streams as the wavefront passes -- identical fp64 histories against the oracle, same statistics as the default path."""
    geom, src, n, seed = TRANSPORT_CASES[name]()
    got, ref, frac = compare_transport(B, geom, src, n, seed, 64, 0.999, opts=dict(refill=1))
    assert got["stats"]["n_kernel_launches"] == 1
    d = B.transport_run(B.Geometry(geom), src, seed, n, 64, per_photon=True)
    assert np.array_equal(d["hash"].cpu().numpy(), got["hash"].cpu().numpy())
    for k in ("n_steps", "n_compton", "n_pe", "n_pair", "n_cut", "n_escaped", "n_stuck", "n_photons"):
        assert d["stats"][k] == got["stats"][k], k
    assert np.allclose(d["edep"].cpu().numpy(), got["edep"].cpu().numpy(), rtol=1e-12, atol=1e-12)
    # fp32, untracked kernels, more photons than lanes on the chip (every lane refills many times)
    g = B.Geometry(geom, refill=1)
    a = B.transport_run(g, src, seed, 400000, 32)
    b = B.transport_run(B.Geometry(geom), src, seed, 400000, 32)
    for k in ("n_steps", "n_compton", "n_pe", "n_pair", "n_cut", "n_escaped", "n_stuck", "n_photons"):
        assert a["stats"][k] == b["stats"][k], k
    assert np.allclose(a["edep"].cpu().numpy(), b["edep"].cpu().numpy(), rtol=1e-9, atol=1e-9)
    with pytest.raises(Exception):
        B.transport_run(B.Geometry(geom, refill=1, secondaries=1), src, seed, 100, 64)


def test_transport_is_independent_of_steps_per_pass_and_sharding(B):
    import torch
    geom, src, n, seed = TRANSPORT_CASES["phantom16"]()
    runs = []
    # tail_photons=1: no run-to-completion pass before a single photon is left, so the wavefront passes, the
    # compaction and the front/back partition of the queues are all exercised; the default (one tail pass after
    # the first, since n is small) must give the same histories
    for K, tail in ((1, 1), (7, 1), (64, 1), (16, 0)):
        g = B.Geometry(geom, steps_per_pass=K, tail_photons=tail)
        r = B.transport_run(g, src, seed, n, 64, per_photon=True)
        runs.append((r["hash"].cpu().numpy(), r["edep"].cpu().numpy(), r["stats"]))
        assert r["stats"]["n_passes"] >= (2 if (K == 64 or tail == 0) else 8)
    for h, e, s in runs[1:]:
        assert np.array_equal(h, runs[0][0]) and np.allclose(e, runs[0][1], rtol=1e-12, atol=1e-12)
        assert s["n_steps"] == runs[0][2]["n_steps"]
    g = B.Geometry(geom)
    a = B.transport_run(g, src, seed, 7000, 64, first_photon_id=0, per_photon=True)
    b = B.transport_run(g, src, seed, n - 7000, 64, first_photon_id=7000, per_photon=True)
    assert np.array_equal(np.concatenate([a["hash"].cpu().numpy(), b["hash"].cpu().numpy()]), runs[0][0])
    assert np.allclose((a["edep"] + b["edep"]).cpu().numpy(), runs[0][1], rtol=1e-12, atol=1e-12)
    # the callee zeroes edep: reusing a dirty buffer gives the same tally
    buf = torch.full((g.n_places,), 123.0, dtype=torch.float64, device="cuda")
    c = B.transport_run(g, src, seed, n, 64, edep=buf)
    assert np.allclose(c["edep"].cpu().numpy(), runs[0][1], rtol=1e-12, atol=1e-12)
    # empty run
    z = B.transport_run(g, src, seed, 0, 64)
    assert z["stats"]["n_steps"] == 0 and float(z["edep"].sum()) == 0.0


def test_host_buffer_entry_points(B):
    geom, src, n, seed = TRANSPORT_CASES["config1"]()
    g = B.Geometry(geom)
    dev = B.transport_run(g, src, seed, n, 64)
    host = B.transport_run_host(g, src, seed, n, 64)
    assert np.allclose(host["edep"], dev["edep"].cpu().numpy(), rtol=1e-12, atol=1e-12)
    assert host["stats"]["n_steps"] == dev["stats"]["n_steps"]
    og = oracle.OracleGeometry(geom)
    pos, dirs = W.nav_queries(geom, 10001, seed=5, dtype=np.float64)
    vol, step, nxt = B.nav_query_host(g, pos, dirs, 64)
    rv = og.locate(pos, dirs, 64); rs, rn = og.compute_step(pos, dirs, rv, None, 64)
    assert np.array_equal(vol, rv) and np.array_equal(step, rs) and np.array_equal(nxt, rn)


def test_batching_across_the_queue_capacity(B):
    """More photons than one batch (2^24): ids beyond the boundary keep their own Philox streams."""
    geom, src, _, seed = TRANSPORT_CASES["config1"]()
    g = B.Geometry(geom)
    n = (1 << 24) + 50000
    got = B.transport_run(g, src, seed, n, 32, per_photon=True)
    og = oracle.OracleGeometry(geom)
    first = (1 << 24) - 20000
    ref = og.transport(src, seed, 40000, 32, first_id=first, per_photon=True)
    hg = got["hash"][first:first + 40000].cpu().numpy().view(np.uint64)
    assert (hg == ref["hash"]).mean() > 0.99
    assert got["stats"]["n_photons"] == n and int(got["nsteps"].sum().item()) == got["stats"]["n_steps"]


def test_batching_across_the_queue_capacity_with_secondaries(B):
    """Two batches of primaries, each followed by its own batches of annihilation photons (the pair-vertex list is reused
    per batch; 20 MeV in lead: more pairs than half a queue, so the secondaries of the first batch need two chunks)."""
    geom, src, _, seed = SECONDARY_CASES["lead_slab_20MeV"]()
    g = B.Geometry(geom, secondaries=1)
    n = (1 << 24) + 30000
    got = B.transport_run(g, src, seed, n, 64, per_photon=True)
    og = oracle.OracleGeometry(geom, secondaries=1)
    first = (1 << 24) - 15000
    ref = og.transport(src, seed, 30000, 64, first_id=first, per_photon=True)
    hg = got["hash"][first:first + 30000].cpu().numpy().view(np.uint64)
    ng = got["nsteps"][first:first + 30000].cpu().numpy().astype(np.uint32)
    assert ((hg == ref["hash"]) & (ng == ref["nsteps"])).mean() >= 0.999
    s = got["stats"]
    assert s["n_photons"] == n and 2 * s["n_pair"] > n and int(got["nsteps"].to(torch_int64()).sum().item()) == s["n_steps"]
    assert s["n_pe"] + s["n_pair"] + s["n_cut"] + s["n_escaped"] + s["n_stuck"] == n + 2 * s["n_pair"]
    book = float(got["edep"].sum()) + s["e_escaped"] + s["e_stuck"]
    assert abs(book / s["e_source"] - 1) < 1e-9


def torch_int64():
    import torch
    return torch.int64


# ---- BASELINE.json full-size geometries, in the launch configuration bench.py times ---------------------------
def test_config3_full_size_sampled(B):
    """Config 3 as bench.py runs it (64^3 voxels, 1e7 photons, fp32): oracle on a sampled id range; book-keeping,
    stuck count and step totals as size-independent properties."""
    wl = W.config(3)
    g = B.Geometry(wl.geometry)
    assert g.voxel_info()["cells"] == 64 ** 3
    got = B.transport_run(g, wl.source, wl.seed, wl.n, 32, per_photon=True)
    s = got["stats"]
    assert s["n_photons"] == wl.n and s["n_stuck"] <= wl.n // 10 ** 6
    edep = got["edep"]
    book = float(edep.sum().item()) + s["e_escaped"] + s["e_stuck"]
    assert abs(book / s["e_source"] - 1) < 2e-6
    assert int(got["nsteps"].to("cuda").sum(dtype=__import__("torch").int64).item()) == s["n_steps"]
    assert s["n_steps"] > 30 * wl.n
    og = oracle.OracleGeometry(wl.geometry)
    first, m = 5_000_000, 30000
    ref = og.transport(wl.source, wl.seed, m, 32, first_id=first, per_photon=True)
    hg = got["hash"][first:first + m].cpu().numpy().view(np.uint64)
    ng = got["nsteps"][first:first + m].cpu().numpy().astype(np.uint32)
    same = (hg == ref["hash"]) & (ng == ref["nsteps"])
    print(f"config 3 full size: identical fp32 histories on the sample {same.mean():.5f}")
    assert same.mean() > 0.98
    # aggregate edep: GPU total scaled to the sample vs oracle sample, within MC noise
    per_photon_gpu = float(edep.sum().item()) / wl.n
    per_photon_ref = ref["edep"].sum() / m
    assert abs(per_photon_gpu / per_photon_ref - 1) < 0.05


def test_config3_full_geometry_edep_criterion(B):
    """SURVEY 8(c) C10, literally, on the full 64^3 geometry in fp32: the CUDA path and the oracle transport the SAME photon
    ids (5e6 .. 8e6 of the 1e7); (i) |sum_v edep_gpu - sum_v edep_oracle| <= 1e-3 sum_v edep_oracle, and for every block of
    16^3 voxels with >= 1e4 deposits the relative difference is <= 1e-3 + 3 sigma_MC, sigma_MC^2 = sum of the squared deposits
    of the block (oracle's tally) over the square of its sum.  Also: fp32 histories identical on > 99.5 % of the ids."""
    wl = W.config(3)
    g = B.Geometry(wl.geometry); og = oracle.OracleGeometry(wl.geometry)
    first, m = 5_000_000, 3_000_000                      # ~1.2e4 deposits per 16^3 block
    got = B.transport_run(g, wl.source, wl.seed, m, 32, first_photon_id=first, per_photon=True)
    ref = og.transport(wl.source, wl.seed, m, 32, first_id=first, per_photon=True, tally=True)
    edep = got["edep"].cpu().numpy()
    tot = ref["edep"].sum()
    assert abs(edep.sum() - tot) <= 1e-3 * tot
    same = (got["hash"].cpu().numpy().view(np.uint64) == ref["hash"]) & (got["nsteps"].cpu().numpy().astype(np.uint32) == ref["nsteps"])
    n = 64
    v = np.arange(n ** 3)
    block = (v % n) // 16 + 4 * (((v // n) % n) // 16 + 4 * ((v // (n * n)) // 16))
    bsum = lambda a: np.bincount(block, weights=a[2:], minlength=64)
    eg, er, e2, nd = bsum(edep), bsum(ref["edep"]), bsum(ref["edep_sq"]), bsum(ref["n_dep"].astype(np.float64))
    big = nd >= 1e4
    assert big.sum() >= 16, nd
    rel = np.abs(eg[big] - er[big]) / er[big]
    sigma = np.sqrt(e2[big]) / er[big]
    print(f"config 3 full geometry, {m} shared ids: identical fp32 histories {same.mean():.5f}; total edep diff {abs(edep.sum() - tot) / tot:.2e}; "
          f"{big.sum()} blocks with >= 1e4 deposits, max relative diff {rel.max():.2e} (sigma_MC {sigma.min():.1e} .. {sigma.max():.1e}); "
          f"L1 over voxels {np.abs(edep - ref['edep']).sum() / tot:.2e}")
    assert np.all(rel <= 1e-3 + 3 * sigma)
    assert same.mean() > 0.995
    # deposits outside the voxels (world, container) are negligible but must agree too
    assert abs(edep[:2].sum() - ref["edep"][:2].sum()) <= 1e-3 * tot


@pytest.mark.parametrize("precision", [32, 64])
def test_config5_full_geometry_sampled(B, precision):
    wl = W.config(5)
    g = B.Geometry(wl.geometry)
    og = oracle.OracleGeometry(wl.geometry)
    n = 2_000_003
    R = np.float32 if precision == 32 else np.float64
    pos, dirs = W.nav_queries(wl.geometry, n, seed=wl.seed, dtype=R)
    tp, tv = cuda(pos), cuda(dirs)
    vol = B.nav_locate(g, tp, tv)
    step, nxt = B.nav_compute_step(g, tp, tv, vol)
    rng = np.random.default_rng(0)
    sel = np.sort(rng.choice(n, 60000, replace=False)); sel[-1] = n - 1
    rv = og.locate(pos[sel], dirs[sel], precision)
    rs, rn = og.compute_step(pos[sel], dirs[sel], rv, None, precision)
    assert np.array_equal(vol.cpu().numpy()[sel], rv)
    assert np.array_equal(step.cpu().numpy()[sel], rs) and np.array_equal(nxt.cpu().numpy()[sel], rn)
    assert len(np.unique(rv)) > 3000


def test_config2_and_config4_reduced_counts(B):
    wl = W.config(2)
    compare_transport(B, wl.geometry, wl.source, 30000, wl.seed, 64, 0.999)
    compare_transport(B, wl.geometry, wl.source, 30000, wl.seed, 32, 0.97)
    wl = W.config(4)
    compare_transport(B, wl.geometry, wl.source, 30000, wl.seed, 32, 0.97)
    compare_transport(B, wl.geometry, wl.source, 30000, wl.seed, 64, 0.999)


def test_inline_division_and_sqrt_are_correctly_rounded(B):
    """navigation may only use correctly rounded operations.  The kernels use their own in-line
    Newton-Raphson division / square root (no out-of-line slow path); on the device they must equal the IEEE
    round-to-nearest intrinsics bit for bit: every fp32 square-root argument, 2^31 division pairs."""
    r = B.selftest_arith(1 << 31)
    assert r["sqrt_mismatches"] == 0, r
    assert r["div_mismatches"] == 0, r


# ---- the paper's own benchmark (attenuation-only Algorithm 1, Spheres geometry) ------------
def spheres_small():
    return W.spheres_geometry(n_side=6, cube=1500.0, radius=100.0)


@pytest.mark.parametrize("precision", [64, 32])
def test_orb_navigation_bit_exact(B, precision):
    """Orb solid: locate and ComputeStep (voxel walk of the vacuum world through 216 balls) equal the oracle's plain
    linear scans bit for bit."""
    geom = spheres_small()
    og = oracle.OracleGeometry(geom); g = B.Geometry(geom)
    assert g.voxel_info()["grids"] == 1
    rng = np.random.default_rng(31)
    n = 60001
    R = np.float64 if precision == 64 else np.float32
    p = (rng.uniform(-1, 1, size=(n, 3)) * 760.0).astype(R); v = unit(rng, n).astype(R)
    # a share of the points on / near ball surfaces
    c = (rng.integers(0, 6, size=(n // 4, 3)) + 0.5) * 250.0 - 750.0
    k = rng.choice([-2.0, -1.0, -0.5, 0.0, 0.5, 1.0, 2.0], size=n // 4)
    p[: n // 4] = (c + unit(rng, n // 4) * (100.0 + k[:, None] * g.tolerance(precision) / 2)).astype(R)
    tp, tv = cuda(p), cuda(v)
    ref = og.locate(p, v, precision, use_grid=False)
    assert np.array_equal(B.nav_locate(g, tp, tv).cpu().numpy(), ref)
    assert np.array_equal(B.nav_locate(g, tp, None).cpu().numpy(), og.locate(p, None, precision, use_grid=False))
    step, nxt = B.nav_compute_step(g, tp, tv, cuda(ref))
    rstep, rnxt = og.compute_step(p, v, ref, None, precision, use_grid=False)
    assert np.array_equal(nxt.cpu().numpy(), rnxt) and np.array_equal(step.cpu().numpy(), rstep)
    assert (ref > 0).sum() > 1000 and (rnxt > 0).sum() > 1000 and (ref == -1).any()


@pytest.mark.parametrize("precision", [64, 32])
@pytest.mark.parametrize("which", ["random", "regular"])
def test_free_path_matches_oracle(B, which, precision):
    """gn_free_path_run (Algorithm 2 phase 5) on the paper's Spheres geometry, N = 1e5 as in the paper for the Random set
    (Regular: 400 x 250): T_i and the number of steps equal the oracle's bit for bit (same canonical arithmetic)."""
    import torch
    geom = W.spheres_geometry()
    og = oracle.OracleGeometry(geom); g = B.Geometry(geom)
    R = np.float64 if precision == 64 else np.float32
    pos, d, Y = (W.random_particles(100000, seed=11, dtype=R) if which == "random" else W.regular_particles(400, 250, dtype=R))
    T, ns = B.free_path_run(g, cuda(pos), cuda(d), cuda(Y), W.MU_MASS_AL_1MEV)
    T = T.cpu().numpy(); ns = ns.cpu().numpy().astype(np.uint32)
    # the oracle's ComputeStep scans all 8000 balls per step: compare a seeded sample of 4000 particles
    idx = np.random.default_rng(1).choice(len(Y), 4000, replace=False)
    rT, rns = og.free_path(pos[idx], d[idx], Y[idx], W.MU_MASS_AL_1MEV, precision)
    assert np.array_equal(T[idx], rT) and np.array_equal(ns[idx], rns)
    assert np.isinf(T).any() and np.isfinite(T).sum() > len(Y) // 2
    # whole-set property: every finite free path ends inside a ball (mu = 0 in the vacuum), checked in fp64
    fin = np.isfinite(T)
    end = pos[fin].astype(np.float64) + d[fin].astype(np.float64) * T[fin].astype(np.float64)[:, None]
    rel = np.mod(end + 2500.0, 250.0) - 125.0
    assert np.all(np.linalg.norm(rel, axis=1) <= 100.0 + (1e-6 if precision == 64 else 2e-2))
    # empty input
    e3 = torch.empty((0, 3), dtype=torch.float64 if precision == 64 else torch.float32, device="cuda")
    Te, _ = B.free_path_run(g, e3, e3, e3[:, 0].contiguous(), W.MU_MASS_AL_1MEV)
    assert Te.numel() == 0


# ---- surface normal of the boundary crossed ---------------------------------
@pytest.mark.parametrize("name", list(GEOMS) + ["spheres"])
@pytest.mark.parametrize("precision", [64, 32])
def test_step_normals_bit_exact(B, name, precision):
    """gn_nav_compute_step_normal: step, next volume and the outward normal of the surface that ends the step equal the
    oracle's (plain linear scan, so the voxel walk's tie rule for the daughter hit is checked too)."""
    geom = spheres_small() if name == "spheres" else GEOMS[name]()
    og = oracle.OracleGeometry(geom); g = B.Geometry(geom)
    rng = np.random.default_rng(202)
    n = 40003
    R = np.float64 if precision == 64 else np.float32
    p = query_points(geom, rng, n).astype(R); v = unit(rng, n).astype(R)
    ref = og.locate(p, v, precision, use_grid=False)
    step, nxt, nrm = B.nav_compute_step_normal(g, cuda(p), cuda(v), cuda(ref))
    rstep, rnxt, rnrm = og.compute_step_normal(p, v, ref, None, precision, use_grid=False)
    assert np.array_equal(step.cpu().numpy(), rstep) and np.array_equal(nxt.cpu().numpy(), rnxt)
    assert np.array_equal(nrm.cpu().numpy(), rnrm)
    fin = np.isfinite(rstep)
    assert np.allclose(np.linalg.norm(rnrm[fin].astype(np.float64), axis=1), 1.0, atol=1e-5) and np.all(rnrm[~fin] == 0)
    ms = rng.uniform(0, 300, n).astype(R)
    step, nxt, nrm = B.nav_compute_step_normal(g, cuda(p), cuda(v), cuda(ref), cuda(ms))
    rstep, rnxt, rnrm = og.compute_step_normal(p, v, ref, ms, precision, use_grid=False)
    assert np.array_equal(step.cpu().numpy(), rstep) and np.array_equal(nxt.cpu().numpy(), rnxt) and np.array_equal(nrm.cpu().numpy(), rnrm)


# ---- BASELINE.json's full sizes, in the launch configuration bench.py times, on sampled outputs ------------------
@pytest.mark.parametrize("k,precision,min_same", [(2, 64, 0.999), (2, 32, 0.97), (4, 32, 0.97)])
def test_config2_config4_full_size_sampled(B, k, precision, min_same):
    wl = W.config(k)
    g = B.Geometry(wl.geometry)
    got = B.transport_run(g, wl.source, wl.seed, wl.n, precision, per_photon=True)
    s = got["stats"]
    assert s["n_photons"] == wl.n and s["n_stuck"] <= max(1, wl.n // 10 ** 6)
    book = float(got["edep"].sum().item()) + s["e_escaped"] + s["e_stuck"]
    assert abs(book / s["e_source"] - 1) < (1e-11 if precision == 64 else 2e-6)
    assert int(got["nsteps"].sum(dtype=__import__("torch").int64).item()) == s["n_steps"]
    og = oracle.OracleGeometry(wl.geometry)
    first, m = wl.n // 2, 20000
    ref = og.transport(wl.source, wl.seed, m, precision, first_id=first, per_photon=True)
    hg = got["hash"][first:first + m].cpu().numpy().view(np.uint64)
    ng = got["nsteps"][first:first + m].cpu().numpy().astype(np.uint32)
    ef = got["efinal"][first:first + m].cpu().numpy()
    same = (hg == ref["hash"]) & (ng == ref["nsteps"]) & (np.abs(ef - ref["efinal"]) <= (1e-9 if precision == 64 else 1e-4) * np.abs(ref["efinal"]))
    print(f"config {k} fp{precision} full size: identical histories on the sample {same.mean():.5f}")
    assert same.mean() >= min_same


@pytest.mark.parametrize("precision", [32, 64])
def test_config5_full_size_sampled(B, precision):
    """1e8 queries (fp32; 5e7 in fp64 to stay within a few seconds), generated on the device as bench.py does; the oracle
    checks a seeded sample of 40000 of them bit for bit."""
    import torch
    wl = W.config(5)
    g = B.Geometry(wl.geometry)
    og = oracle.OracleGeometry(wl.geometry)
    n = wl.n if precision == 32 else wl.n // 2
    dt = torch.float32 if precision == 32 else torch.float64
    pos, dirs = W.nav_queries_torch(wl.geometry, n, wl.seed, dt, torch.device("cuda"))
    vol = B.nav_locate(g, pos, dirs)
    step, nxt = B.nav_compute_step(g, pos, dirs, vol)
    sel = torch.from_numpy(np.sort(np.random.default_rng(3).choice(n, 40000, replace=False))).cuda()
    p = pos[sel].cpu().numpy(); v = dirs[sel].cpu().numpy()
    rv = og.locate(p, v, precision)
    rs, rn = og.compute_step(p, v, rv, None, precision)
    assert np.array_equal(vol[sel].cpu().numpy(), rv)
    assert np.array_equal(step[sel].cpu().numpy(), rs) and np.array_equal(nxt[sel].cpu().numpy(), rn)
    # every point of the world box is located, except those within the tolerance of its surface that head outwards (C3)
    assert n - int((vol >= 0).sum().item()) < n // 10 ** 5


@pytest.mark.parametrize("precision", [64, 32])
def test_cones_and_balls_dense_queries(B, precision):
    """queries concentrated in and around every solid of the mixed geometry (boxes, tube sectors, balls,
    three cone shapes incl. one with its apex on an end plane, all randomly rotated, some with a nested ball), a share of
    them exactly on the solids' bounding spheres' tangent directions: locate, ComputeStep and the surface normal equal the
    oracle's linear scans bit for bit."""
    geom = W.mixed_solids_geometry()
    og = oracle.OracleGeometry(geom); g = B.Geometry(geom)
    rng = np.random.default_rng(77)
    R = np.float64 if precision == 64 else np.float32
    centres = geom.transforms[geom.placements[1:65, 3], 9:]                   # the 64 top-level solids
    n = 120000
    c = centres[rng.integers(0, len(centres), n)]
    p = (c + unit(rng, n) * rng.uniform(0, 40.0, n)[:, None]).astype(R)
    v = unit(rng, n)
    aim = rng.random(n) < 0.5                                                  # half of the rays aim at the solid's region
    tgt = c + unit(rng, n) * rng.uniform(0, 25.0, n)[:, None]
    dv = tgt - p.astype(np.float64); nv = np.linalg.norm(dv, axis=1, keepdims=True)
    v = np.where(aim[:, None] & (nv > 1e-6), dv / np.maximum(nv, 1e-300), v).astype(R)
    v = (v.astype(np.float64) / np.linalg.norm(v.astype(np.float64), axis=1, keepdims=True)).astype(R)
    tp, tv = cuda(p), cuda(v)
    ref = og.locate(p, v, precision, use_grid=False)
    assert np.array_equal(B.nav_locate(g, tp, tv).cpu().numpy(), ref)
    stype = geom.solid_type[geom.placements[np.maximum(ref, 0), 1]]
    assert (stype[ref > 0] == 3).sum() > 5000 and (stype[ref > 0] == 2).sum() > 3000
    step, nxt, nrm = B.nav_compute_step_normal(g, tp, tv, cuda(ref))
    rstep, rnxt, rnrm = og.compute_step_normal(p, v, ref, None, precision, use_grid=False)
    assert np.array_equal(step.cpu().numpy(), rstep) and np.array_equal(nxt.cpu().numpy(), rnxt) and np.array_equal(nrm.cpu().numpy(), rnrm)
    s2, n2 = B.nav_compute_step(g, tp, tv, cuda(ref))
    assert np.array_equal(s2.cpu().numpy(), rstep) and np.array_equal(n2.cpu().numpy(), rnxt)
    # second leg from the crossing points (on the surfaces): relocation and the next step
    fin = np.isfinite(rstep) & (rnxt >= 0)
    x2 = oracle.move(p[fin], v[fin], rstep[fin], precision)
    r2s, r2n, r2m = og.compute_step_normal(x2, v[fin], rnxt[fin], None, precision, use_grid=False)
    g2s, g2n, g2m = B.nav_compute_step_normal(g, cuda(x2), cuda(v[fin]), cuda(rnxt[fin]))
    assert np.array_equal(g2s.cpu().numpy(), r2s) and np.array_equal(g2n.cpu().numpy(), r2n) and np.array_equal(g2m.cpu().numpy(), r2m)
