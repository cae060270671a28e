// store.h -- device-resident geometry store (what the kernels see).
//
// One GeoView<Real> per precision; built once by gn_geometry_create (geometry.cu) and passed to the
// kernels by value.  Layout (all arrays in HBM, L2-resident for every BASELINE.json config):
//   node[i]   NodeRec: everything a visit to node i needs in ONE 32-byte sector (fp32; 48 B in fp64):
//               parent, solid | flags, material, number of daughters, link, Tg[3]
//             link >= 0: first index into dlist (daughters in index order); link < 0: ~(voxel grid id)
//             flag NODE_IDENTITY: the composed rotation is exactly the identity, so p_local = x - Tg and
//             v_local = w (the general fma chain gives the same values; only the sign of zeros can differ,
//             which no comparison in the navigator can see) and `rot` is never read for this node
//             flag NODE_REGULAR (leaf boxes only): the box coincides with exactly one cell of its mother's voxel grid,
//             is that cell's only candidate and is not rotated against the mother; link = index of its cell in the mother's
//             grid (ix + nx (iy + ny iz)); bits 16..21 of info = id of that grid, bits 22..27 = "wall" bits: bit 22 + 2 k
//             (+ 1) is set when the cell is the first (last) one of the grid along axis k, i.e. no neighbour cell there.
//             A photon leaving it through a face or an edge finds the candidates in the neighbouring cells directly,
//             without the general cell lookup (nav.cuh: settle, regular_step; box-only kernels).  Only mothers that are
//             unrotated boxes whose grid spans them exactly hand out this flag, so a point within the probe distance of
//             the voxel whose neighbour cell on that side exists is inside the mother by more than delta
//             flag NODE_SLAB (leaf boxes only): the same for a box that coincides with a ROW of cells along one axis, alone in
//             each (a calorimeter layer in a grid whose pitch divides every layer thickness); link = index of its lowest
//             cell; the axis and the number of cells of the row are in its solid record (cS, sS of a box); wall bits for the
//             two ends of the row and the sides.  A photon leaving it through one of the two end faces finds its candidate in
//             the cell beyond that end (nav.cuh: regular_step<.., SLABS>)
//             flag NODE_HINT (tube sectors on a cylindrical lattice inside a full tube of the same radii -- a segmented
//             barrel): hint[4 i ..] names the sibling across each z face and phi plane.  A photon that leaves the sector
//             through one of those faces, farther than 2 probe distances from all its other faces, is in that sibling or in
//             the mother: relocation tests just that one (nav.cuh: settle_flat), the result is the general search's
//   rot[i]    M (row-major, global->local rotation), 9 Real padded to 12 (fp32, three 16-byte loads) /
//             10 (fp64, five 16-byte loads);  p_local = M (x - Tg)
//   solids, mats, grids: small tables (staged to shared memory by every kernel)
//   cells[c]  int2 {x, count}: count == 1 -> x is the candidate daughter itself; else x = offset into cand
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace gn {

enum : int { SOLID_BOX = 0, SOLID_TUBE = 1, SOLID_ORB = 2, SOLID_CONE = 3 };
enum : int { TUBE_SECTOR = 1, TUBE_HOLE = 2 };
enum : int { NODE_HINT = (int)0x80000000u, NODE_IDENTITY = 1 << 30, NODE_REGULAR = 1 << 29, NODE_SLAB = 1 << 28, NODE_SOLID_MASK = 0xffff, NODE_GRID_SHIFT = 16, NODE_GRID_MASK = 0x3f, NODE_WALL_SHIFT = 22, NODE_WALL_MASK = 0x3f };

template <class R> struct SolidRec {
    R a, b, c;            // BOX: hx hy hz      TUBE: rmin rmax hz      ORB: r - -      CONE: r0 = (r1 + r2)/2, slope m, hz
    R cS, sS, cE, sE;     // trig of sphi and sphi + dphi (host libm, fp64, rounded once);  CONE: cS = 1/sqrt(1 + m^2);
                          // BOX: cS = axis of its regular slabs (-1: none), sS = cells per slab (NODE_SLAB)
    int type, flags;
};

template <class R> struct MatRec { R aPE, aC, aP, capZ; };

template <class R> struct NodeRec;
template <> struct alignas(16) NodeRec<float> { int parent, info, mat, ndau; int link; float t[3]; };
template <> struct alignas(16) NodeRec<double> { int parent, info, mat, ndau; int link, pad; double t[3]; };
static_assert(sizeof(NodeRec<float>) == 32 && sizeof(NodeRec<double>) == 48, "node record layout");
template <class R> struct RotStride;
template <> struct RotStride<float> { static constexpr int value = 12; };
template <> struct RotStride<double> { static constexpr int value = 10; };

// header of one voxel grid; laid out so that the fields a cell lookup needs come in 16-byte words
template <class R> struct alignas(16) GridRec {
    R gmin[3], eps0;      // eps = probe half-width in cell units (padded), split over the three words
    R inv_w[3], eps1;
    int n[3];
    int cell_base;        // offset of this grid's cells in `cells`
    R w[3], eps2;
    int sy, sz;           // cell strides along y and z: n[0], n[0] n[1]
    int dense;            // >= 0: every cell holds exactly one candidate, the regular voxel with node index dense + cell index
                          // (the candidate of a cell needs no look-up); -1 otherwise
    int gpad;
    __host__ __device__ R eps(int k) const { return k == 0 ? eps0 : (k == 1 ? eps1 : eps2); }
};

template <class R> struct GeoView {
    const NodeRec<R>* node;
    const R* rot;
    const int* dlist;
    const int* dfirst;    // node -> offset of its daughters in dlist (every node, voxelised or not; the safety scan)
    const int* hint;      // 4 per node: sibling across the lower / upper z face, the start / end phi plane of a NODE_HINT tube sector
    const SolidRec<R>* solids;
    const MatRec<R>* mats;
    const double* rho;    // density per material [g/cm3] (attenuation-only mode: mu = rho * mu_mass)
    const R* mat_r;       // Rayleigh factor per material, n sigma_R0 (Z/13)^2 / 10 (gn_opts.rayleigh; reading 18)
    const R* pe_tab;      // tabulated photoelectric coefficient, n_mats x pe_points (gn_opts.pe_table_per_decade; reading 19)
    const GridRec<R>* grids;
    const int2* cells;
    const int* cand;
    R tol, delta, probe;  // surface tolerance, tol/2, voxel probe half-width
    R e_cut;
    int n_nodes, n_solids, n_mats, n_grids, stuck_limit;
    int rayleigh, pe_per_decade, pe_points;       // optional physics; 0 = off
};

}  // namespace gn
