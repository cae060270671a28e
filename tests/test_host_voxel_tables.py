"""Host logic of gn_geometry_create, checked on the CPU through gn_host_voxel_tables (the same builder with every CUDA call
left out): voxel candidate lists (reading 5: listed by the solid, not by its bounding box -- they must still hold
every daughter that can contain a point of the cell), regular-voxel / regular-slab flags, and the sibling hints of segmented
barrels.  The truth comes from elsewhere: the oracle's brute-force locate (linear scan, no grid) and the placements themselves."""
import numpy as np
import pytest

import oracle
from paper_1209_5235_b200 import workloads as W

NODE_HINT, NODE_IDENTITY, NODE_REGULAR, NODE_SLAB = 1 << 31, 1 << 30, 1 << 29, 1 << 28


@pytest.fixture(scope="module")
def B():
    from paper_1209_5235_b200 import build, binding
    build.build()
    return binding


def flags(info):
    return info.astype(np.int64) & 0xFFFFFFFF


def global_frames(B, geom):
    """Per node: M (global -> local rotation, 3 x 3) and T (global position of the local origin): x_local = M (x - T)."""
    import ctypes as C
    V = geom.placements.shape[0]
    M = np.empty((V, 9)); T = np.empty((V, 3))
    pl = np.ascontiguousarray(geom.placements, np.int32); tr = np.ascontiguousarray(geom.transforms, np.float64)
    rc = B.lib().gn_host_compose_transforms(pl.ctypes.data_as(C.c_void_p), C.c_int32(V), tr.ctypes.data_as(C.c_void_p), C.c_int32(tr.shape[0]),
                                            M.ctypes.data_as(C.c_void_p), T.ctypes.data_as(C.c_void_p))
    assert rc == 0
    return M.reshape(V, 3, 3), T


def detector():
    return W.detector_geometry(seed=4, n_phi=16, n_z=8, barrels=((200, 400), (450, 650)))


GEOMS = {"detector": detector, "cmslike": W.cms_like_geometry, "mixed": W.mixed_solids_geometry, "lattice": lambda: W.lattice_geometry(4, seed=7),
         "spheres": lambda: W.spheres_geometry(6, 1500.0, 100.0)}


@pytest.mark.parametrize("name", list(GEOMS))
def test_candidate_lists_hold_the_daughter_that_contains_the_point(B, name):
    """Random points of every voxelised mother: the daughter that brute force finds there must be listed in the point's cell."""
    geom = GEOMS[name]()
    t = B.host_voxel_tables(geom)
    assert len(t["grids"]) >= 1
    og = oracle.OracleGeometry(geom)
    M, T = global_frames(B, geom)
    parent = geom.placements[:, 0]
    rng = np.random.default_rng(5)
    checked = 0
    for G in t["grids"]:
        mother = int(G[0]); gmin, w, n, base = G[1:4], G[4:7], G[7:10].astype(int), int(G[10])
        m = 40000
        u = rng.random((m, 3))
        pl = gmin + u * (w * n)                                            # mother frame
        f = (pl - gmin) / w
        keep = np.all(np.abs(f - np.round(f)) > 1e-6, axis=1)             # not on a cell boundary
        pl, f = pl[keep], f[keep]
        x = pl @ M[mother] + T[mother]                                    # x = M^T p + T
        vol = og.locate(x, None, 64, use_grid=False)
        # the daughter of `mother` on the way down to the located volume (none: the point is in the mother itself or outside)
        d = vol.copy()
        for _ in range(8):
            up = (d >= 0) & (parent[np.maximum(d, 0)] != mother) & (d != mother)
            d = np.where(up, parent[np.maximum(d, 0)], d)
        ok = (d >= 0) & (d != mother) & (parent[np.maximum(d, 0)] == mother)
        cell = base + (f[:, 0].astype(int) + n[0] * (f[:, 1].astype(int) + n[1] * f[:, 2].astype(int)))
        for c, dd in zip(cell[ok], d[ok]):
            lst = t["cand"][t["cell_start"][c]:t["cell_start"][c + 1]]
            assert dd in lst, (name, mother, c, dd, lst)
            assert np.all(np.diff(lst) > 0)                               # ascending: the lists merge in index order
        checked += int(ok.sum())
    assert checked > 400


def test_lists_by_the_solid_are_shorter_than_lists_by_the_bounding_box(B):
    """A tube sector at 45 degrees fills half of its bounding box: the barrels' cells hold fewer candidates than the boxes cover."""
    geom = detector()
    t = B.host_voxel_tables(geom)
    M, T = global_frames(B, geom)
    for G in t["grids"]:
        mother = int(G[0]); gmin, w, n, base = G[1:4], G[4:7], G[7:10].astype(int), int(G[10])
        ncell = int(np.prod(n))
        counts = np.diff(t["cell_start"][base:base + ncell + 1])
        refs = counts.sum()
        # references a bounding-box rule would make: count the cells each daughter's box overlaps (test-side, from the corner
        # points of the sector in the mother's frame)
        box_refs = 0
        for d in np.nonzero(geom.placements[:, 0] == mother)[0]:
            rmin, rmax, hz, sphi, dphi = geom.solid_params[geom.placements[d, 1]]
            tr = geom.transforms[geom.placements[d, 3]]; R = tr[:9].reshape(3, 3); Tl = tr[9:]
            ph = np.linspace(sphi, sphi + dphi, 33)
            pts = np.array([[r * np.cos(a), r * np.sin(a), z] for r in (rmin, rmax) for a in ph for z in (-hz, hz)]) @ R.T + Tl
            lo = np.floor((pts.min(0) + 1e-9 - gmin) / w).astype(int).clip(0, n - 1); hi = np.floor((pts.max(0) - 1e-9 - gmin) / w).astype(int).clip(0, n - 1)
            box_refs += int(np.prod(hi - lo + 1))
        assert refs < 0.8 * box_refs, (refs, box_refs)
        assert refs / max(1, (counts > 0).sum()) < 2.5


def test_sibling_hints_of_a_segmented_barrel(B):
    """hint[d] = the sector across the lower / upper z face and the start / end phi plane of sector d, from the placements."""
    n_phi, n_z = 16, 8
    geom = detector()
    t = B.host_voxel_tables(geom)
    info = flags(t["info"])
    parent = geom.placements[:, 0]
    barrels = [1, 2]
    assert all(geom.solid_type[geom.placements[b, 1]] == W.TUBE for b in barrels)
    sectors = np.nonzero(np.isin(parent, barrels))[0]
    assert len(sectors) == 2 * n_phi * n_z
    assert np.all(info[sectors] & NODE_HINT) and not np.any(np.delete(info, sectors) & NODE_HINT)
    dphi, hz_s = 2 * np.pi / n_phi, 1600.0 / n_z
    where = {}
    for d in sectors:
        tr = geom.transforms[geom.placements[d, 3]]
        j = int(round((np.arctan2(tr[3], tr[0]) % (2 * np.pi)) / dphi)) % n_phi
        iz = int(round((tr[11] + 1600.0 - hz_s) / (2 * hz_s)))
        where[(int(parent[d]), iz, j)] = int(d)
    assert len(where) == len(sectors)
    for (b, iz, j), d in where.items():
        want = [where.get((b, iz - 1, j), -1), where.get((b, iz + 1, j), -1), where[(b, iz, (j - 1) % n_phi)], where[(b, iz, (j + 1) % n_phi)]]
        assert list(t["hint"][d]) == want, (d, b, iz, j)
    # and geometrically: a point just beyond the end plane of sector d, at mid radius and mid z, is inside hint[d][3]
    og = oracle.OracleGeometry(geom)
    M, T = global_frames(B, geom)
    pts, exp = [], []
    for (b, iz, j), d in where.items():
        rmin, rmax, hz, sphi, _ = geom.solid_params[geom.placements[d, 1]]
        for which, ang in ((3, sphi + dphi + 1e-3), (2, sphi - 1e-3)):
            pl = np.array([0.5 * (rmin + rmax) * np.cos(ang), 0.5 * (rmin + rmax) * np.sin(ang), 0.3 * hz])
            pts.append(pl @ M[d] + T[d]); exp.append(t["hint"][d][which])
        for which, z in ((1, hz + 1e-3), (0, -hz - 1e-3)):
            if t["hint"][d][which] >= 0:
                pl = np.array([0.5 * (rmin + rmax) * np.cos(sphi + 0.3 * dphi), 0.5 * (rmin + rmax) * np.sin(sphi + 0.3 * dphi), z])
                pts.append(pl @ M[d] + T[d]); exp.append(t["hint"][d][which])
    vol = og.locate(np.array(pts), None, 64, use_grid=False)
    d = np.where(np.isin(parent[vol], barrels), vol, parent[vol])        # a module inside the neighbour counts as the neighbour
    assert np.array_equal(d, np.array(exp))


def test_no_hints_without_a_lattice(B):
    for name in ("cmslike", "mixed", "lattice"):
        t = B.host_voxel_tables(GEOMS[name]())
        info = flags(t["info"])
        hinted = np.nonzero(info & NODE_HINT)[0]
        assert np.all(t["hint"][np.setdiff1d(np.arange(len(info)), hinted)] == -1)


def test_regular_voxels_of_a_phantom(B):
    geom = W.phantom_geometry(12, 2.0, seed=3, world_half=150.0)
    t = B.host_voxel_tables(geom)
    info = flags(t["info"])
    voxels = np.nonzero(geom.placements[:, 0] == 1)[0]
    assert len(voxels) == 12 ** 3 and np.all(info[voxels] & NODE_REGULAR) and not np.any(info[voxels] & NODE_SLAB)
    assert len(t["grids"]) == 1 and list(t["grids"][0][7:10]) == [12, 12, 12]
    cells = t["link"][voxels]
    assert sorted(cells) == list(range(12 ** 3))                          # one voxel per cell ...
    assert np.array_equal(np.diff(t["cell_start"]), np.ones(12 ** 3, np.int32))
    assert np.array_equal(t["cand"][cells], voxels)                       # ... and the cell lists exactly that voxel
    # the cell of a voxel is where its centre is
    gmin, w = t["grids"][0][1:4], t["grids"][0][4:7]
    c = np.floor((geom.transforms[geom.placements[voxels, 3]][:, 9:] - gmin) / w).astype(int)
    assert np.array_equal(cells, c[:, 0] + 12 * (c[:, 1] + 12 * c[:, 2]))
    walls = (info[voxels] >> 22) & 0x3F
    for k in range(3):
        assert np.array_equal((walls >> (2 * k)) & 1, (c[:, k] == 0).astype(int)) and np.array_equal((walls >> (2 * k + 1)) & 1, (c[:, k] == 11).astype(int))


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_regular_slabs_of_a_layer_stack(B, axis):
    """Layers of 2, 4, 6, 2 mm in a 2 mm grid: the thin ones are regular voxels, the others slabs of 2 and 3 cells."""
    thick = (2.0, 4.0, 6.0, 2.0); periods = 6; half = 150.0
    b = W._Builder("stack")
    L = periods * sum(thick)
    mh = [half] * 3; mh[axis] = L / 2
    b.place(-1, b.box(400.0, 400.0, 400.0), "air")
    mother = b.place(0, b.box(*mh), "air")
    solids = []
    for th in thick:
        h = [half] * 3; h[axis] = th / 2
        solids.append(b.box(*h))
    u = -L / 2; lows = []
    for _ in range(periods):
        for k, th in enumerate(thick):
            T = [0.0] * 3; T[axis] = u + th / 2
            b.place(mother, solids[k], ["lead", "scint", "iron", "water"][k], T=tuple(T)); lows.append(u + L / 2); u += th
    geom = b.finish()
    t = B.host_voxel_tables(geom)
    info = flags(t["info"])
    assert len(t["grids"]) == 1
    n = t["grids"][0][7:10].astype(int); wcell = t["grids"][0][4 + axis]
    assert n[axis] == int(round(L / 2.0)) and abs(wcell - 2.0) < 1e-12 and np.prod(n) == n[axis]
    layers = np.arange(2, 2 + periods * len(thick))
    for i, d in enumerate(layers):
        th = thick[i % len(thick)]
        cells = int(round(th / 2.0))
        assert bool(info[d] & NODE_REGULAR) == (cells == 1) and bool(info[d] & NODE_SLAB) == (cells > 1), (d, th)
        assert t["link"][d] == int(round(lows[i] / 2.0))                  # its lowest cell
        for q in range(cells):                                            # alone in every cell of its row
            c = t["link"][d] + q
            assert list(t["cand"][t["cell_start"][c]:t["cell_start"][c + 1]]) == [d]
        walls = (info[d] >> 22) & 0x3F
        assert ((walls >> (2 * axis)) & 1) == (i == 0) and ((walls >> (2 * axis + 1)) & 1) == (i == len(layers) - 1)
