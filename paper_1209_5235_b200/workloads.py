"""Seeded synthetic input generators (geometries, sources, navigation queries).

This module serves BOTH the CUDA library's Python binding and the CPU oracle's tests.  It holds none
of the method's arithmetic: no navigation, no physics, no RNG of the method -- only descriptions of
inputs as plain numpy arrays in the layout both C interfaces take:

    materials    (n_mats, 3)  float64   Z, A, rho [g/cm3]
    solid_type   (n_solids,)  int32     0 = BOX, 1 = TUBE, 2 = ORB, 3 = CONE
    solid_params (n_solids,5) float64   BOX: hx,hy,hz,0,0 [mm]; TUBE: rmin,rmax,hz [mm], sphi,dphi [rad]; ORB: r,0,0,0,0; CONE: r1 (at -hz),r2 (at +hz),hz,0,0
    placements   (n_places,4) int32     parent (-1 for node 0 = world; parent < child), solid, material, transform
    transforms   (n_tr, 12)   float64   R row-major (local->parent) then T [mm]

The five configurations are the synthetic stand-ins BASELINE.json names (configs 1..5 in file order;
SURVEY.md section 8(d) fixes the open choices); the paper's own workloads (Spheres, CMS)
are not available.  Everything is seeded with numpy default_rng.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

BOX, TUBE, ORB, CONE = 0, 1, 2, 3
SRC_PENCIL, SRC_GAUSS_PENCIL, SRC_CONE, SRC_ISOTROPIC = 0, 1, 2, 3
E_MONO, E_LOGUNIFORM = 0, 1

# (Z, A, rho).  A from Z/A where BASELINE.json gives only Z_eff.
MATERIALS = {
    "vacuum": (1.0, 1.0, 0.0),
    "air": (7.3, 7.3 / 0.49919, 1.2e-3),
    "lead": (82.0, 207.2, 11.35),
    "water": (7.4, 7.4 / 0.55508, 1.0),
    "lung": (7.4, 7.4 / 0.55508, 0.3),
    "bone": (13.8, 13.8 / 0.51478, 1.85),
    "scint": (5.7, 5.7 / 0.54141, 1.03),
    "iron": (26.0, 55.845, 7.87),
    "silicon": (14.0, 28.0855, 2.33),
    "aluminium": (13.0, 26.9815, 2.699),
}


@dataclasses.dataclass
class Geometry:
    materials: np.ndarray
    solid_type: np.ndarray
    solid_params: np.ndarray
    placements: np.ndarray
    transforms: np.ndarray
    name: str = ""
    material_names: tuple = ()

    @property
    def n_places(self) -> int:
        return int(self.placements.shape[0])


@dataclasses.dataclass
class Source:
    kind: int
    origin: tuple
    axis: tuple
    energy_kind: int = E_MONO
    e0: float = 1.0
    e1: float = 0.0
    sigma: float = 0.0
    half_angle: float = 0.0


@dataclasses.dataclass
class Workload:
    name: str
    geometry: Geometry
    source: Optional[Source]
    n: int                      # photons (configs 1-4) or queries (config 5)
    precisions: tuple
    seed: int


class _Builder:
    def __init__(self, name):
        self.name = name
        self.mat_names, self.mats = [], []
        self.stype, self.sparams = [], []
        self.places, self.trs = [], []

    def material(self, name):
        if name not in self.mat_names:
            self.mat_names.append(name)
            self.mats.append(MATERIALS[name])
        return self.mat_names.index(name)

    def box(self, hx, hy, hz):
        self.stype.append(BOX); self.sparams.append((hx, hy, hz, 0.0, 0.0)); return len(self.stype) - 1

    def tube(self, rmin, rmax, hz, sphi=0.0, dphi=2 * math.pi):
        self.stype.append(TUBE); self.sparams.append((rmin, rmax, hz, sphi, dphi)); return len(self.stype) - 1

    def orb(self, r):
        self.stype.append(ORB); self.sparams.append((r, 0.0, 0.0, 0.0, 0.0)); return len(self.stype) - 1

    def cone(self, r1, r2, hz):
        self.stype.append(CONE); self.sparams.append((r1, r2, hz, 0.0, 0.0)); return len(self.stype) - 1

    def place(self, parent, solid, material, R=None, T=(0.0, 0.0, 0.0)):
        R = np.eye(3) if R is None else np.asarray(R, dtype=np.float64)
        self.trs.append(np.concatenate([R.reshape(9), np.asarray(T, dtype=np.float64)]))
        self.places.append((parent, solid, self.material(material) if isinstance(material, str) else material, len(self.trs) - 1))
        return len(self.places) - 1

    def finish(self) -> Geometry:
        return Geometry(
            materials=np.ascontiguousarray(np.array(self.mats, dtype=np.float64).reshape(-1, 3)),
            solid_type=np.ascontiguousarray(np.array(self.stype, dtype=np.int32)),
            solid_params=np.ascontiguousarray(np.array(self.sparams, dtype=np.float64).reshape(-1, 5)),
            placements=np.ascontiguousarray(np.array(self.places, dtype=np.int32).reshape(-1, 4)),
            transforms=np.ascontiguousarray(np.array(self.trs, dtype=np.float64).reshape(-1, 12)),
            name=self.name, material_names=tuple(self.mat_names))


def rot_z(angle):
    c, s = math.cos(angle), math.sin(angle)
    return np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]])


def random_rotation(rng):
    q = rng.normal(size=4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


# ----------------------------------------------------------------------------------------------
def slab_geometry(seed=1) -> Geometry:
    """Config 1: 1 m air world, 10 cm lead box at the origin, 4 water boxes of 2 cm inside it."""
    rng = np.random.default_rng(seed)
    b = _Builder("config1_tiny_slab")
    world = b.place(-1, b.box(500, 500, 500), "air")
    lead = b.place(world, b.box(50, 50, 50), "lead")
    wsolid = b.box(10, 10, 10)
    centres = []
    while len(centres) < 4:
        c = rng.uniform(-39.0, 39.0, size=3)
        if all(np.max(np.abs(c - o)) >= 21.0 for o in centres):
            centres.append(c)
    for c in centres:
        b.place(lead, wsolid, "water", T=c)
    return b.finish()


def slab_source() -> Source:
    return Source(SRC_PENCIL, (0.0, 0.0, -500.0), (0.0, 0.0, 1.0), E_MONO, 1.0)


def homogeneous_slab(material="water", half=(1000.0, 1000.0, 50.0), world_half=2000.0) -> Geometry:
    """One slab of one material in a vacuum world: the exp(-mu x) transmission pin (Eq. 2-5)."""
    b = _Builder("homogeneous_slab")
    world = b.place(-1, b.box(world_half, world_half, world_half), "vacuum")
    b.place(world, b.box(*half), material)
    return b.finish()


def calorimeter_geometry(n_pairs=50, t_lead=2.0, t_scint=5.0, half_xy=500.0) -> Geometry:
    """Config 2: n_pairs alternating lead / scintillator layers (lead first, lowest z) in a mother box."""
    b = _Builder("config2_sampling_calorimeter")
    hz = n_pairs * (t_lead + t_scint) / 2
    world = b.place(-1, b.box(2 * half_xy, 2 * half_xy, 2 * half_xy), "air")
    mother = b.place(world, b.box(half_xy, half_xy, hz), "air")
    s_pb, s_sc = b.box(half_xy, half_xy, t_lead / 2), b.box(half_xy, half_xy, t_scint / 2)
    z = -hz
    for _ in range(n_pairs):
        b.place(mother, s_pb, "lead", T=(0, 0, z + t_lead / 2)); z += t_lead
        b.place(mother, s_sc, "scint", T=(0, 0, z + t_scint / 2)); z += t_scint
    return b.finish()


def calorimeter_source() -> Source:
    return Source(SRC_GAUSS_PENCIL, (0.0, 0.0, -500.0), (0.0, 0.0, 1.0), E_MONO, 10.0, sigma=10.0)


def phantom_geometry(n=64, voxel=2.0, seed=3, world_half=1200.0) -> Geometry:
    """Config 3: n^3 grid of `voxel` mm boxes filling a water container; material per voxel seeded
    categorical 70 % water / 20 % bone / 10 % lung.  index = ix + n (iy + n iz) + 2."""
    rng = np.random.default_rng(seed)
    b = _Builder(f"config3_voxel_phantom_{n}")
    half = n * voxel / 2
    world = b.place(-1, b.box(world_half, world_half, world_half), "air")
    cont = b.place(world, b.box(half, half, half), "water")
    vs = b.box(voxel / 2, voxel / 2, voxel / 2)
    mats = [b.material("water"), b.material("bone"), b.material("lung")]
    choice = rng.choice(3, size=n * n * n, p=[0.7, 0.2, 0.1])
    # vectorised construction (262 144 placements at n = 64)
    idx = np.arange(n * n * n)
    ix, iy, iz = idx % n, (idx // n) % n, idx // (n * n)
    T = np.stack([-half + voxel * (ix + 0.5), -half + voxel * (iy + 0.5), -half + voxel * (iz + 0.5)], axis=1)
    g = b.finish()
    tr = np.zeros((n ** 3, 12)); tr[:, 0] = tr[:, 4] = tr[:, 8] = 1.0; tr[:, 9:] = T
    nt0 = g.transforms.shape[0]
    pl = np.empty((n ** 3, 4), dtype=np.int32)
    pl[:, 0] = cont; pl[:, 1] = vs; pl[:, 2] = np.array(mats, dtype=np.int32)[choice]; pl[:, 3] = nt0 + idx
    g.transforms = np.ascontiguousarray(np.concatenate([g.transforms, tr]))
    g.placements = np.ascontiguousarray(np.concatenate([g.placements, pl]))
    return g


def phantom_source(n=64, voxel=2.0, distance=1000.0, half_angle_deg=5.0, energy=6.0) -> Source:
    return Source(SRC_CONE, (0.0, 0.0, -(n * voxel / 2 + distance)), (0.0, 0.0, 1.0), E_MONO, energy,
                  half_angle=math.radians(half_angle_deg))


def detector_geometry(seed=4, n_phi=32, n_z=64, barrels=((200, 400), (450, 650), (700, 900), (950, 1150)),
                      hz=1600.0, module_every=4, module_half=(10.0, 10.0, 20.0)) -> Geometry:
    """Config 4: world -> full-tube barrels -> n_phi x n_z tube sectors -> box modules (random rotation
    about z) in every `module_every`-th sector.  Materials of sectors and modules seeded uniform from
    {lead, iron, silicon, air}."""
    rng = np.random.default_rng(seed)
    b = _Builder(f"config4_detector_{len(barrels)}x{n_phi}x{n_z}")
    world = b.place(-1, b.box(1500, 1500, 2000), "air")
    pool = ["lead", "iron", "silicon", "air"]
    dphi = 2 * math.pi / n_phi
    hz_s = hz / n_z
    barrel_ids, sector_solids = [], []
    for (r0, r1) in barrels:
        barrel_ids.append(b.place(world, b.tube(r0, r1, hz), "air"))
        sector_solids.append(b.tube(r0, r1, hz_s, -dphi / 2, dphi))
    sectors = []
    for bi, (r0, r1) in enumerate(barrels):
        for iz in range(n_z):
            for j in range(n_phi):
                s = b.place(barrel_ids[bi], sector_solids[bi], pool[rng.integers(4)], R=rot_z(j * dphi),
                            T=(0, 0, -hz + hz_s * (2 * iz + 1)))
                sectors.append((s, 0.5 * (r0 + r1)))
    msolid = b.box(*module_half)
    for k, (s, rmid) in enumerate(sectors):
        if k % module_every == 0:
            b.place(s, msolid, pool[rng.integers(4)], R=rot_z(rng.uniform(0, 2 * math.pi)), T=(rmid, 0, 0))
    return b.finish()


def detector_source() -> Source:
    return Source(SRC_ISOTROPIC, (0.0, 0.0, 0.0), (0.0, 0.0, 1.0), E_LOGUNIFORM, 0.1, 1000.0)


def lattice_geometry(n=4, seed=7, pitch=100.0, fill="aluminium") -> Geometry:
    """Spheres-like test geometry (solids on a regular grid in a vacuum cube): n^3 cells of
    `pitch` mm, each holding a randomly rotated box, holed tube or tube sector that fits its cell; every
    third solid holds a rotated daughter box.  Exercises rotations, tubes and the sparse voxel walk."""
    rng = np.random.default_rng(seed)
    b = _Builder(f"lattice_{n}")
    half = n * pitch / 2
    world = b.place(-1, b.box(half + 50, half + 50, half + 50), "vacuum")
    rmax = 0.5 * pitch / math.sqrt(3) * 0.95          # circumscribed sphere fits the cell
    solids = [
        b.box(rmax * 0.55, rmax * 0.5, rmax * 0.6),
        b.tube(0.0, rmax * 0.7, rmax * 0.7),
        b.tube(rmax * 0.3, rmax * 0.7, rmax * 0.7),
        b.tube(rmax * 0.25, rmax * 0.7, rmax * 0.7, 0.3, 2.1),
        b.tube(0.0, rmax * 0.7, rmax * 0.7, -0.4, math.pi),
    ]
    inner = b.box(rmax * 0.12, rmax * 0.1, rmax * 0.3)
    k = 0
    hosts = []
    for iz in range(n):
        for iy in range(n):
            for ix in range(n):
                s = int(rng.integers(len(solids)))
                c = (-half + pitch * (ix + 0.5), -half + pitch * (iy + 0.5), -half + pitch * (iz + 0.5))
                node = b.place(world, solids[s], fill, R=random_rotation(rng), T=c)
                if k % 3 == 0:
                    hosts.append((node, s))
                k += 1
    for node, s in hosts:
        # daughter box placed where every host solid has material: at radius 0.5 rmax, angle 1.0 rad
        r = rmax * 0.5
        pos = (r * math.cos(1.0), r * math.sin(1.0), 0.0) if s != 0 else (0.0, 0.0, 0.0)
        b.place(node, inner, "lead", R=rot_z(rng.uniform(0, 6.28)), T=pos)
    return b.finish()


def mixed_solids_geometry(n=4, seed=9, pitch=100.0) -> Geometry:
    """All four solid types the paper names (boxes, tubes, cones, spheres) on a regular grid in a vacuum
    cube, randomly rotated; every fourth solid holds a small ball.  Test geometry for the orb and cone solids."""
    rng = np.random.default_rng(seed)
    b = _Builder(f"mixed_{n}")
    half = n * pitch / 2
    world = b.place(-1, b.box(half + 40, half + 40, half + 40), "vacuum")
    rmax = 0.5 * pitch / math.sqrt(3) * 0.95
    solids = [
        b.box(rmax * 0.55, rmax * 0.5, rmax * 0.6),
        b.tube(rmax * 0.3, rmax * 0.7, rmax * 0.7, 0.3, 2.1),
        b.orb(rmax * 0.8),
        b.cone(rmax * 0.2, rmax * 0.7, rmax * 0.65),
        b.cone(rmax * 0.7, 0.0, rmax * 0.5),
        b.cone(rmax * 0.6, rmax * 0.6, rmax * 0.6),
    ]
    inner = b.orb(rmax * 0.1)
    k = 0
    for iz in range(n):
        for iy in range(n):
            for ix in range(n):
                s = int(rng.integers(len(solids)))
                c = (-half + pitch * (ix + 0.5), -half + pitch * (iy + 0.5), -half + pitch * (iz + 0.5))
                node = b.place(world, solids[s], "aluminium", R=random_rotation(rng), T=c)
                if k % 4 == 0:
                    # on the axis at z = -0.3 hz for cones (inside every frustum above), at a radius with material for the tube
                    pos = (rmax * 0.5 * math.cos(1.3), rmax * 0.5 * math.sin(1.3), 0.0) if s == 1 else (0.0, 0.0, -0.1 * rmax)
                    b.place(node, inner, "lead", T=pos)
                k += 1
    return b.finish()


def cms_like_geometry(seed=13, n_rings=8, n_phi=16) -> Geometry:
    """A synthetic collider-detector hierarchy, six levels deep, of all four solid types (the paper's second test geometry is
    the CMS detector; that model is not available, SURVEY 8(f) NEXT-2 asks for a "deeper CMS-like synthetic
    hierarchy").  world box -> { beam pipe, tracker tube with silicon layers, ECAL barrel -> z rings -> phi sectors -> rotated
    crystal boxes -> rotated cones -> balls; HCAL barrel -> phi sectors -> radial layers; two end-cap cones (one flipped) with
    a ring and a ball each; twelve rotated muon boxes with layer boxes and a transverse drift tube }.  Daughters lie strictly
    inside their mothers and siblings do not overlap (checked against the brute-force locate in tests/)."""
    rng = np.random.default_rng(seed)
    b = _Builder(f"cmslike_{n_rings}x{n_phi}")
    world = b.place(-1, b.box(3000, 3000, 3000), "air")
    b.place(world, b.tube(0.0, 30.0, 2700.0), "vacuum")                                  # beam pipe
    tracker = b.place(world, b.tube(40.0, 1100.0, 2700.0), "air")
    for r in (100.0, 250.0, 400.0, 600.0, 800.0, 1000.0):
        b.place(tracker, b.tube(r, r + 4.0, 2600.0), "silicon")
    # ECAL: barrel -> rings -> sectors -> crystal -> cone -> ball
    ecal = b.place(world, b.tube(1200.0, 1500.0, 2700.0), "air")
    hz_r = 2700.0 / n_rings
    dphi = 2 * math.pi / n_phi
    ring_solid = b.tube(1205.0, 1495.0, hz_r - 2.0)
    sector_solid = b.tube(1210.0, 1490.0, hz_r - 4.0, -dphi / 2 + 0.004, dphi - 0.008)
    crystal = b.box(110.0, min(150.0, 1220.0 * math.tan(dphi / 2 - 0.01) - 5.0), min(200.0, hz_r - 10.0))
    cone = b.cone(20.0, 60.0, 80.0)
    ball = b.orb(25.0)
    for iz in range(n_rings):
        ring = b.place(ecal, ring_solid, "air", T=(0, 0, -2700.0 + hz_r * (2 * iz + 1)))
        for j in range(n_phi):
            sec = b.place(ring, sector_solid, "scint", R=rot_z(j * dphi))
            cr = b.place(sec, crystal, "lead", R=rot_z(rng.uniform(-0.05, 0.05)), T=(1350.0, 0, 0))
            co = b.place(cr, cone, "iron", R=random_rotation(rng))
            b.place(co, ball, "silicon", T=(0, 0, 10.0))
    # HCAL: barrel -> sectors -> radial layers (tube sectors of the same opening, inset)
    hcal = b.place(world, b.tube(1600.0, 2400.0, 2700.0), "air")
    n_h = 12
    dph = 2 * math.pi / n_h
    hsec = b.tube(1605.0, 2395.0, 2690.0, -dph / 2 + 0.003, dph - 0.006)
    layers = [b.tube(r, r + 150.0, 2680.0, -dph / 2 + 0.006, dph - 0.012) for r in (1620.0, 1820.0, 2020.0, 2220.0)]
    for j in range(n_h):
        s = b.place(hcal, hsec, "scint", R=rot_z(j * dph))
        for k, lay in enumerate(layers):
            b.place(s, lay, "iron" if k % 2 == 0 else "lead")
    # end caps: frustums opening away from the centre, the one at -z flipped about x
    cap = b.cone(400.0, 1500.0, 120.0)
    flip = np.array([[1.0, 0.0, 0.0], [0.0, -1.0, 0.0], [0.0, 0.0, -1.0]])
    ring_in_cap = b.tube(150.0, 350.0, 100.0)
    for sgn, Rm in ((1.0, None), (-1.0, flip)):
        c = b.place(world, cap, "iron", R=Rm, T=(0, 0, sgn * 2850.0))
        b.place(c, ring_in_cap, "lead")
        b.place(c, b.orb(40.0), "silicon", T=(0.0, 0.0, -50.0))
    # muon chambers: boxes around the barrel, rotated about z; three layer boxes and a drift tube across each
    chamber = b.box(100.0, 500.0, 2500.0)
    layer = b.box(15.0, 480.0, 2400.0)
    drift = b.tube(0.0, 12.0, 450.0)
    rot_x90 = np.array([[1.0, 0.0, 0.0], [0.0, 0.0, -1.0], [0.0, 1.0, 0.0]])         # tube axis along the chamber's y
    for j in range(12):
        a = j * math.pi / 6 + 0.02
        ch = b.place(world, chamber, "air", R=rot_z(a), T=(2700.0 * math.cos(a), 2700.0 * math.sin(a), 0.0))
        for x in (-70.0, -20.0, 30.0):
            b.place(ch, layer, "aluminium", T=(x, 0, 0))
        b.place(ch, drift, "air", R=rot_x90, T=(80.0, 0.0, 2450.0 * rng.uniform(-1, 1)))
    return b.finish()


# ----------------------------------------------------------------------------------------------
# ---- the paper's own benchmark inputs (section 3.5) ----------------------------
MU_MASS_AL_1MEV = 0.06146       # cm^2/g


def spheres_geometry(n_side=20, cube=5000.0, radius=100.0) -> Geometry:
    """"Spheres": n_side^3 aluminium balls on a regular grid in a vacuum cube (8000 balls, 5 m cube).
    The paper does not print the radius; 100 mm (pitch 250 mm) is this repo's choice."""
    b = _Builder(f"spheres{n_side}")
    world = b.place(-1, b.box(cube / 2, cube / 2, cube / 2), "vacuum")
    ball = b.orb(radius)
    pitch = cube / n_side
    for iz in range(n_side):
        for iy in range(n_side):
            for ix in range(n_side):
                b.place(world, ball, "aluminium", T=(-cube / 2 + pitch * (ix + 0.5), -cube / 2 + pitch * (iy + 0.5), -cube / 2 + pitch * (iz + 0.5)))
    return b.finish()


def random_particles(n=100000, seed=11, dtype=np.float64, origin=(0.0, 0.0, 0.0)):
    """"Random" set: directions uniform on the unit sphere, lifetimes Y ~ Exp(1); all particles start
    from the centre of the geometry (L160).  Generated on the host as in Algorithm 2 steps 2-3 (numpy PCG64 here, the
    paper used Boost's Mersenne Twister)."""
    rng = np.random.default_rng(seed)
    d = rng.normal(size=(n, 3)); d /= np.linalg.norm(d, axis=1, keepdims=True)
    Y = rng.exponential(1.0, size=n)
    pos = np.tile(np.asarray(origin, dtype=np.float64), (n, 1))
    d = d.astype(dtype); d64 = d.astype(np.float64)
    d = (d64 / np.linalg.norm(d64, axis=1, keepdims=True)).astype(dtype)
    return pos.astype(dtype), d, Y.astype(dtype)


def regular_particles(nx=400, ny=250, dtype=np.float64, origin=(0.0, 0.0, 0.0), screen_z=1000.0, pixel=4.0):
    """"Regular" set: the particles travel towards a regular nx x ny grid, input in column-major order,
    all with lifetime Y = 1 -- the output is a volume-raytraced bitmap.  The screen is this repo's choice: pixel centres
    of an nx x ny raster with `pixel` mm pitch on the plane z = screen_z, centred on the axis."""
    ix, iy = np.meshgrid(np.arange(nx), np.arange(ny), indexing="ij")        # column-major: iy fastest
    px = (ix.reshape(-1) - (nx - 1) / 2.0) * pixel; py = (iy.reshape(-1) - (ny - 1) / 2.0) * pixel
    d = np.stack([px, py, np.full(px.shape, screen_z)], axis=1)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    n = nx * ny
    pos = np.tile(np.asarray(origin, dtype=np.float64), (n, 1))
    return pos.astype(dtype), d.astype(dtype), np.ones(n, dtype=dtype)


def world_half_extent(geom: Geometry) -> np.ndarray:
    s = int(geom.placements[0, 1])
    p = geom.solid_params[s]
    if geom.solid_type[s] == BOX:
        return np.array([p[0], p[1], p[2]])
    return np.array([p[1], p[1], p[2]])


def nav_queries(geom: Geometry, n: int, seed: int = 5, dtype=np.float64, first: int = 0):
    """Config 5 queries: point uniform in the world bounding box, direction uniform on the sphere.
    Query i depends only on (seed, first + i) chunk position, so ranges can be sharded."""
    h = world_half_extent(geom)
    chunk = 1 << 20
    pos = np.empty((n, 3), dtype=dtype); dirs = np.empty((n, 3), dtype=dtype)
    done = 0
    while done < n:
        m = min(chunk - (first + done) % chunk, n - done)
        c = (first + done) // chunk
        rng = np.random.default_rng([seed, c])
        u = rng.random((chunk, 5))
        o = (first + done) % chunk
        u = u[o:o + m]
        pos[done:done + m] = ((2 * u[:, :3] - 1) * h).astype(dtype)
        ct = 1 - 2 * u[:, 3]; st = np.sqrt(np.maximum(0.0, 1 - ct * ct)); ph = 2 * math.pi * u[:, 4]
        d = np.stack([st * np.cos(ph), st * np.sin(ph), ct], axis=1)
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        d = d.astype(dtype)
        if dtype == np.float32:       # renormalise in the target precision
            d /= np.linalg.norm(d.astype(np.float64), axis=1, keepdims=True).astype(np.float32)
        dirs[done:done + m] = d
        done += m
    return pos, dirs


def nav_queries_torch(geom: Geometry, n: int, seed: int, dtype, device):
    """Same distribution as nav_queries, generated on `device` with torch's generator (plumbing only;
    used by bench.py at the full 1e8-query size where a host-side numpy array would take minutes)."""
    import torch
    g = torch.Generator(device=device); g.manual_seed(seed)
    h = torch.tensor(world_half_extent(geom), dtype=torch.float64, device=device)
    pos = torch.empty((n, 3), dtype=dtype, device=device); dirs = torch.empty((n, 3), dtype=dtype, device=device)
    chunk = 1 << 24
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        u = torch.rand((m, 5), generator=g, device=device, dtype=torch.float64)
        pos[s:s + m] = ((2 * u[:, :3] - 1) * h).to(dtype)
        ct = 1 - 2 * u[:, 3]; st = torch.sqrt(torch.clamp(1 - ct * ct, min=0)); ph = 2 * math.pi * u[:, 4]
        d = torch.stack([st * torch.cos(ph), st * torch.sin(ph), ct], dim=1)
        d = d / d.norm(dim=1, keepdim=True)
        dirs[s:s + m] = d.to(dtype)
    return pos, dirs


def config(k: int, scale: float = 1.0) -> Workload:
    """The five BASELINE.json configurations (1-based).  scale < 1 shrinks only the photon/query count."""
    if k == 1:
        return Workload("config1_tiny_slab", slab_geometry(1), slab_source(), int(1e4 * scale), (64,), 1)
    if k == 2:
        return Workload("config2_sampling_calorimeter", calorimeter_geometry(), calorimeter_source(), int(1e6 * scale), (64, 32), 2)
    if k == 3:
        return Workload("config3_voxel_phantom", phantom_geometry(64), phantom_source(64), int(1e7 * scale), (32,), 3)
    if k == 4:
        return Workload("config4_detector", detector_geometry(), detector_source(), int(1e7 * scale), (32,), 4)
    if k == 5:
        return Workload("config5_nav_queries", detector_geometry(), None, int(1e8 * scale), (32, 64), 5)
    raise ValueError("config must be 1..5")
