// store.h -- device-resident structure-of-arrays geometry store (what the kernels see).
//
// One GeoView<Real> per precision; built once by gn_geometry_create (geometry.cu) and passed to the
// kernels by value.  Layout (all arrays in HBM, L2-resident for every BASELINE.json config):
//   node[i]   int4  {parent, solid | flags, material, number of daughters}      16 B / node
//             flag NODE_IDENTITY: the composed rotation is exactly the identity, so p_local = x - Tg and
//             v_local = w (the general fma chain gives the same values; only the sign of zeros can differ,
//             which no comparison in the navigator can see)
//   kids[i]   int2  {first index into dlist (daughters in index order), voxel grid id or -1}
//   xf[i]     12 Real: M (row-major, global->local rotation) then Tg; p_local = M (x - Tg)
//             48 B (fp32, three 16-byte loads) / 96 B (fp64, six 16-byte loads); Tg sits in the last 16 / 32 B
//   solids, mats: tiny tables (staged to shared memory by every kernel)
//   grids[g]  header of the voxel grid of one mother
//   cells[c]  int2 {x, count}: count == 1 -> x is the candidate daughter itself; else x = offset into cand
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace gn {

enum : int { SOLID_BOX = 0, SOLID_TUBE = 1 };
enum : int { TUBE_SECTOR = 1, TUBE_HOLE = 2 };
enum : int { NODE_IDENTITY = 1 << 30, NODE_SOLID_MASK = (1 << 30) - 1 };

template <class R> struct SolidRec {
    R a, b, c;            // BOX: hx hy hz      TUBE: rmin rmax hz
    R cS, sS, cE, sE;     // trig of sphi and sphi + dphi (host libm, fp64, rounded once)
    int type, flags;
};

template <class R> struct MatRec { R aPE, aC, aP, capZ; };

template <class R> struct GridRec {
    R gmin[3], inv_w[3], w[3], eps[3];   // eps = probe half-width in cell units (padded)
    int n[3];
    int cell_base;        // offset of this grid's cells in `cells`
};

template <class R> struct GeoView {
    const int4* node;
    const int2* kids;
    const int* dlist;
    const R* xf;
    const SolidRec<R>* solids;
    const MatRec<R>* mats;
    const GridRec<R>* grids;
    const int2* cells;
    const int* cand;
    R tol, delta, probe;  // surface tolerance, tol/2, voxel probe half-width
    R e_cut;
    int n_nodes, n_solids, n_mats, stuck_limit;
};

}  // namespace gn
