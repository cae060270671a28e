// geometry.cu -- gn_geometry_create / destroy: validate the placement tree, compose the affine transforms
// root-down in fp64, build the flattened voxel grids (C5) and upload the
// structure-of-arrays store (store.h) in both precisions.  Host code only; "Load the geometry
// and transfer it to GPU memory".
#include <algorithm>
#include <cmath>
#include <cstring>
#include <string>
#include <vector>
#include "geometry.h"
#include "hostmath.h"

namespace gn {

static thread_local std::string g_last_error;
void set_error(const std::string& msg) { g_last_error = msg; }
int fail(int code, const std::string& msg) { g_last_error = msg; return code; }
const char* last_error_cstr() { return g_last_error.c_str(); }

namespace {

const double kRe = 2.8179403262e-13, kAlpha = 7.2973525693e-3, kNA = 6.02214076e23, kBarn = 1e-24;
const double kPi = 3.14159265358979323846;

struct HostSolid { int type; double a, b, c, sphi, dphi; bool sector; double cS, sS, cE, sE; double rbound; };

struct Uploader {
    gn_geometry* geo; bool dry = false; bool ok = true; std::string err;
    template <class T> const T* put(const std::vector<T>& v) {
        if (!ok || dry) return nullptr;
        void* d = nullptr;
        size_t bytes = std::max<size_t>(v.size(), 1) * sizeof(T);
        cudaError_t e = cudaMalloc(&d, bytes);
        if (e != cudaSuccess) { ok = false; err = std::string("cudaMalloc: ") + cudaGetErrorString(e); return nullptr; }
        geo->allocations.push_back(d); geo->device_bytes += (int64_t)bytes;
        if (!v.empty()) {
            e = cudaMemcpy(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
            if (e != cudaSuccess) { ok = false; err = std::string("cudaMemcpy: ") + cudaGetErrorString(e); return nullptr; }
        }
        return static_cast<const T*>(d);
    }
};

// axis-aligned bounds of an annular sector r in [r0, r1], phi in [p0, p1]
void sector_bounds(double r0, double r1, double p0, double p1, double lo[2], double hi[2]) {
    double xs[12], ys[12]; int n = 0;
    const double ang[2] = {p0, p1}, rr[2] = {r0, r1};
    for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) { xs[n] = rr[j] * std::cos(ang[i]); ys[n] = rr[j] * std::sin(ang[i]); ++n; }
    int k0 = (int)std::ceil(p0 / (kPi / 2) - 1e-12), k1 = (int)std::floor(p1 / (kPi / 2) + 1e-12);
    for (int k = k0; k <= k1 && n < 12; ++k) { xs[n] = r1 * std::cos(k * (kPi / 2)); ys[n] = r1 * std::sin(k * (kPi / 2)); ++n; }
    lo[0] = hi[0] = xs[0]; lo[1] = hi[1] = ys[0];
    for (int i = 1; i < n; ++i) { lo[0] = std::min(lo[0], xs[i]); hi[0] = std::max(hi[0], xs[i]); lo[1] = std::min(lo[1], ys[i]); hi[1] = std::max(hi[1], ys[i]); }
    double pad = 1e-9 * r1;
    lo[0] -= pad; lo[1] -= pad; hi[0] += pad; hi[1] += pad;
}

// bounds of a placed daughter in its mother's frame (R, T: local -> mother)
void daughter_bounds(const HostSolid& s, const double* R, const double* T, double lo[3], double hi[3]) {
    if (s.type == GN_TUBE && s.sector && std::fabs(R[8] - 1.0) < 1e-12 && std::fabs(R[0] * R[4] - R[1] * R[3] - 1.0) < 1e-9) {
        // rotation about z: the sector stays a sector, shifted in angle -- exact bounds
        double th = std::atan2(R[3], R[0]);
        double l2[2], h2[2];
        sector_bounds(s.a, s.b, s.sphi + th, s.sphi + s.dphi + th, l2, h2);
        lo[0] = l2[0] + T[0]; hi[0] = h2[0] + T[0]; lo[1] = l2[1] + T[1]; hi[1] = h2[1] + T[1];
        lo[2] = T[2] - s.c; hi[2] = T[2] + s.c;
        return;
    }
    double l[3], h[3];
    if (s.type == GN_BOX) { l[0] = -s.a; h[0] = s.a; l[1] = -s.b; h[1] = s.b; l[2] = -s.c; h[2] = s.c; }
    else if (s.type == GN_CONE) { l[0] = l[1] = -s.rbound; h[0] = h[1] = s.rbound; l[2] = -s.c; h[2] = s.c; }
    else if (s.type == GN_ORB) {          // rotation invariant
        for (int k = 0; k < 3; ++k) { lo[k] = T[k] - s.a; hi[k] = T[k] + s.a; }
        return;
    } else {
        l[2] = -s.c; h[2] = s.c;
        if (s.sector) sector_bounds(s.a, s.b, s.sphi, s.sphi + s.dphi, l, h);
        else { l[0] = l[1] = -s.b; h[0] = h[1] = s.b; }
    }
    for (int k = 0; k < 3; ++k) { lo[k] = 1e300; hi[k] = -1e300; }
    for (int c = 0; c < 8; ++c) {
        double q[3] = {(c & 1) ? h[0] : l[0], (c & 2) ? h[1] : l[1], (c & 4) ? h[2] : l[2]};
        for (int k = 0; k < 3; ++k) {
            double y = R[3 * k] * q[0] + R[3 * k + 1] * q[1] + R[3 * k + 2] * q[2] + T[k];
            lo[k] = std::min(lo[k], y); hi[k] = std::max(hi[k], y);
        }
    }
}

// Can the placed daughter (R, T: local -> mother) come anywhere near the cell [clo, chi] of its mother's voxel grid?  Returns
// true only when that is PROVABLY not so: some bounding set of the solid (slab, cylinder, hole, half-plane,
// ball, cone -- the solid is their intersection and the outsideness D is the largest signed distance s_k to one of them) stays
// farther than `margin` from every point of the cell, so D > margin on the whole cell.  Planar sets are tested at the eight
// corners (s_k is linear: its minimum over a box is at a corner), curved ones through the centre and the half diagonal rho
// (every s_k is 1-Lipschitz: s_k >= s_k(centre) - rho), the hole through the corners (the distance from the axis is convex:
// its maximum over a box is at a corner).  An axis-aligned bounding box is a poor fit for a tube sector or a rotated box;
// this test keeps such a daughter out of the cells its box covers but the solid does not.
static bool cell_excluded(const HostSolid& s, const double* R, const double* T, const double clo[3], const double chi[3], double margin) {
    double q[8][3], ctr[3] = {0, 0, 0};
    for (int c = 0; c < 8; ++c) {
        const double y[3] = {((c & 1) ? chi[0] : clo[0]) - T[0], ((c & 2) ? chi[1] : clo[1]) - T[1], ((c & 4) ? chi[2] : clo[2]) - T[2]};
        for (int k = 0; k < 3; ++k) { q[c][k] = R[k] * y[0] + R[3 + k] * y[1] + R[6 + k] * y[2]; ctr[k] += q[c][k] / 8; }      // q = R^T y
    }
    const double rho = 0.5 * std::sqrt((chi[0] - clo[0]) * (chi[0] - clo[0]) + (chi[1] - clo[1]) * (chi[1] - clo[1]) + (chi[2] - clo[2]) * (chi[2] - clo[2]));
    auto beyond_plane = [&](double nx, double ny, double nz, double h) {           // n . q - h > margin at every corner
        for (int c = 0; c < 8; ++c) if (!(nx * q[c][0] + ny * q[c][1] + nz * q[c][2] - h > margin)) return false;
        return true;
    };
    if (s.type == GN_ORB) return std::sqrt(ctr[0] * ctr[0] + ctr[1] * ctr[1] + ctr[2] * ctr[2]) - rho - s.a > margin;
    if (s.type == GN_BOX)
        return beyond_plane(1, 0, 0, s.a) || beyond_plane(-1, 0, 0, s.a) || beyond_plane(0, 1, 0, s.b) || beyond_plane(0, -1, 0, s.b) ||
               beyond_plane(0, 0, 1, s.c) || beyond_plane(0, 0, -1, s.c);
    if (beyond_plane(0, 0, 1, s.c) || beyond_plane(0, 0, -1, s.c)) return true;
    const double rc = std::sqrt(ctr[0] * ctr[0] + ctr[1] * ctr[1]);
    if (s.type == GN_CONE) {                                                        // (r - u(z)) cs, u = r0 + m z (a, b of the record)
        const double m = s.b, cs = 1.0 / std::sqrt(1.0 + m * m);
        return (rc - (s.a + m * ctr[2])) * cs - rho > margin;
    }
    if (rc - rho - s.b > margin) return true;                                       // outside the outer cylinder
    if (s.a > 0) {                                                                  // inside the hole
        double rmax = 0;
        for (int c = 0; c < 8; ++c) rmax = std::max(rmax, std::sqrt(q[c][0] * q[c][0] + q[c][1] * q[c][1]));
        if (s.a - rmax > margin) return true;
    }
    if (s.sector && (beyond_plane(s.sS, -s.cS, 0, 0) || beyond_plane(-s.sE, s.cE, 0, 0))) return true;
    return false;
}

template <class R> SolidRec<R> make_solid_rec(const HostSolid& s) {
    SolidRec<R> o;
    o.a = (R)s.a; o.b = (R)s.b; o.c = (R)s.c; o.cS = (R)s.cS; o.sS = (R)s.sS; o.cE = (R)s.cE; o.sE = (R)s.sE;
    o.type = s.type == GN_BOX ? SOLID_BOX : (s.type == GN_ORB ? SOLID_ORB : (s.type == GN_CONE ? SOLID_CONE : SOLID_TUBE));
    o.flags = 0;
    if (s.type == GN_TUBE) { if (s.sector) o.flags |= TUBE_SECTOR; if (o.a > 0) o.flags |= TUBE_HOLE; }
    return o;
}

template <class R> MatRec<R> make_mat_rec(double Z, double A, double rho, double s0) {
    double n = rho * kNA / A;                        // atoms / cm^3; mu [1/mm] = n sigma / 10
    MatRec<R> o;
    o.aPE = (R)(n * (s0 * kBarn * std::pow(Z / 82.0, 5.0)) / 10.0);
    o.aC = (R)(n * (Z * (2.0 * kPi * kRe * kRe)) / 10.0);
    o.aP = (R)(n * (kAlpha * kRe * kRe * Z * Z) / 10.0);
    o.capZ = (R)((28.0 / 9.0) * std::log(183.0 * std::pow(Z, -1.0 / 3.0)) - 2.0 / 27.0);
    return o;
}

// One solid from its type code and five parameters (gammanav.h).  What is stored is what the device formulas of
// nav.cuh read: half-lengths / radii as given; for a phi sector the cosines and sines of its two bounding planes;
// for a cone the mid radius, the slope dr/dz and 1 / sqrt(1 + slope^2).
int parse_solid(int type, const double* q, HostSolid& out, const char** why) {
    out = HostSolid{};
    out.type = type;
    switch (type) {
    case GN_BOX:
        out.a = q[0]; out.b = q[1]; out.c = q[2];
        if (out.a > 0 && out.b > 0 && out.c > 0) return GN_OK;
        *why = "box half-lengths must be positive"; return GN_INVALID_ARGUMENT;
    case GN_ORB:
        out.a = q[0];
        if (out.a > 0) return GN_OK;
        *why = "orb radius must be positive"; return GN_INVALID_ARGUMENT;
    case GN_CONE: {
        const double r_low = q[0], r_high = q[1], half = q[2];
        if (!(r_low >= 0 && r_high >= 0 && r_low + r_high > 0 && half > 0)) { *why = "cone needs r1, r2 >= 0, r1 + r2 > 0, hz > 0"; return GN_INVALID_ARGUMENT; }
        out.a = (r_low + r_high) / 2;
        out.b = (r_high - r_low) / (2 * half);
        out.c = half;
        out.cS = 1 / std::sqrt(1 + out.b * out.b);
        out.rbound = std::max(r_low, r_high);
        return GN_OK;
    }
    case GN_TUBE: {
        out.a = q[0]; out.b = q[1]; out.c = q[2]; out.sphi = q[3]; out.dphi = q[4];
        if (!(out.a >= 0 && out.b > out.a && out.c > 0)) { *why = "tube needs 0 <= rmin < rmax, hz > 0"; return GN_INVALID_ARGUMENT; }
        if (out.dphi >= 2 * kPi) return GN_OK;                        // full tube: no phi planes
        if (!(out.dphi > 0) || out.dphi > kPi) { *why = "tube sector must have 0 < dphi <= pi (or a full tube)"; return GN_UNSUPPORTED_SOLID; }
        const double phi_end = out.sphi + out.dphi;
        out.sector = true;
        out.cS = std::cos(out.sphi); out.sS = std::sin(out.sphi);
        out.cE = std::cos(phi_end); out.sE = std::sin(phi_end);
        return GN_OK;
    }
    default:
        *why = "unknown solid type"; return GN_UNSUPPORTED_SOLID;
    }
}

struct HostGrid { int n[3]; double gmin[3], w[3]; int cell_base; int mother; };

// gn_host_voxel_tables: the host tables of a geometry (voxel grids, candidate lists, node flags, sibling hints) as
// gn_geometry_create builds them, kept instead of uploaded -- the same code path with every CUDA call left out
struct HostTables {
    std::vector<int> info, link, hint, cell_start, cand;
    std::vector<HostGrid> grids;
};
static thread_local HostTables* g_dry = nullptr;

}  // namespace
}  // namespace gn

using namespace gn;

extern "C" int gn_geometry_create(const double* h_materials, int32_t n_mats, const int32_t* h_solid_type,
                                  const double* h_solid_params, int32_t n_solids, const int32_t* h_placements,
                                  int32_t n_places, const double* h_transforms, int32_t n_transforms,
                                  const gn_opts* h_opts, gn_geometry** out) {
    if (!h_materials || !h_solid_type || !h_solid_params || !h_placements || !h_transforms || !out)
        return fail(GN_INVALID_ARGUMENT, "gn_geometry_create: NULL argument");
    if (n_mats <= 0 || n_solids <= 0 || n_places <= 0 || n_transforms <= 0)
        return fail(GN_INVALID_ARGUMENT, "gn_geometry_create: empty table");
    if (n_solids > NODE_SOLID_MASK + 1) return fail(GN_INVALID_ARGUMENT, "gn_geometry_create: at most 65536 solids (the node record keeps 16 bits for the solid index)");
    const bool dry = g_dry != nullptr;                             // host tables only (gn_host_voxel_tables): no device is touched
    int dev_count = 0;
    if (!dry && (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0)) {
        cudaGetLastError();
        return fail(GN_CUDA_ERROR, "gn_geometry_create: no CUDA device (this library has no CPU fallback)");
    }
    for (int i = 0; i < n_mats; ++i) {
        double Z = h_materials[3 * i], A = h_materials[3 * i + 1], rho = h_materials[3 * i + 2];
        if (!(Z > 0 && A > 0 && rho >= 0)) return fail(GN_INVALID_ARGUMENT, "gn_geometry_create: material needs Z > 0, A > 0, rho >= 0");
    }
    std::vector<HostSolid> solids(n_solids);
    for (int i = 0; i < n_solids; ++i) {
        const char* why = nullptr;
        const int rc = parse_solid(h_solid_type[i], h_solid_params + 5 * (size_t)i, solids[i], &why);
        if (rc != GN_OK) return fail(rc, std::string("gn_geometry_create: ") + why);
    }
    const size_t V = (size_t)n_places;
    std::vector<int4> node(V);
    std::vector<double> Rg(9 * V), Tg(3 * V);
    std::vector<int> kid_count(V, 0);
    for (size_t i = 0; i < V; ++i) {
        const int p = h_placements[4 * i], sol = h_placements[4 * i + 1], mat = h_placements[4 * i + 2];
        if (sol < 0 || sol >= n_solids || mat < 0 || mat >= n_mats) return fail(GN_INVALID_ARGUMENT, "gn_geometry_create: placement index out of range");
        node[i] = make_int4(p, sol, mat, -1);
    }
    {
        std::vector<Affine> global;
        const int st = compose_tree(h_placements, n_places, h_transforms, n_transforms, global);     // hostmath.h (C0)
        if (st == 1) return fail(GN_INVALID_ARGUMENT, "gn_geometry_create: placement index out of range");
        if (st == 2) return fail(GN_BAD_TREE, "gn_geometry_create: node 0 must be the world and parent < child");
        if (st == 3) return fail(GN_BAD_TREE, "gn_geometry_create: rotation not orthonormal");
        for (size_t i = 0; i < V; ++i) {
            std::memcpy(&Rg[9 * i], global[i].R.m, 9 * sizeof(double));
            Tg[3 * i] = global[i].T.x; Tg[3 * i + 1] = global[i].T.y; Tg[3 * i + 2] = global[i].T.z;
            if (node[i].x >= 0) kid_count[node[i].x]++;
        }
    }
    // daughters in index order (CSR)
    std::vector<int2> kids(V);
    std::vector<int> dlist(V > 1 ? V - 1 : 0);
    { int acc = 0; for (size_t i = 0; i < V; ++i) { kids[i] = make_int2(acc, 0); acc += kid_count[i]; } }
    for (size_t i = 1; i < V; ++i) { int p = node[i].x; dlist[kids[p].x + kids[p].y] = (int)i; kids[p].y++; }

    gn_geometry* geo = new gn_geometry();
    geo->n_places = n_places; geo->n_solids = n_solids; geo->n_mats = n_mats;
    if (!dry) cudaGetDevice(&geo->device);
    if (!dry) {   // stream-ordered scratch of the query sort: a pool of the handle's own that keeps freed blocks (the device's default
        // pool and its release threshold are the application's, not this library's)
        cudaMemPoolProps props{};
        props.allocType = cudaMemAllocationTypePinned; props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice; props.location.id = geo->device;
        if (cudaMemPoolCreate(&geo->pool, &props) == cudaSuccess) {
            unsigned long long keep = ~0ull;
            cudaMemPoolSetAttribute(geo->pool, cudaMemPoolAttrReleaseThreshold, &keep);
        } else { cudaGetLastError(); geo->pool = nullptr; }
    }
    gn_opts o{}; if (h_opts) o = *h_opts;
    const HostSolid& ws = solids[node[0].y];
    double ext = ws.type == GN_BOX ? std::max(ws.a, std::max(ws.b, ws.c)) : (ws.type == GN_ORB ? ws.a : (ws.type == GN_CONE ? std::max(ws.rbound, ws.c) : std::max(ws.b, ws.c)));
    {   // bounding box of the world solid (schedule only: the cells of the ray-coherent work order)
        const double hxy = ws.type == GN_BOX ? ws.a : (ws.type == GN_ORB ? ws.a : (ws.type == GN_CONE ? ws.rbound : ws.b));
        const double hb[3] = {hxy, ws.type == GN_BOX ? ws.b : hxy, ws.type == GN_ORB ? ws.a : ws.c};
        for (int k = 0; k < 3; ++k) { geo->world_h[k] = (float)hb[k]; geo->world_c[k] = 0.0f; }
    }
    geo->tol64 = o.tol64 > 0 ? o.tol64 : 1e-9;
    geo->tol32 = o.tol32 > 0 ? o.tol32 : (double)(float)(ext * 0x1p-18);
    if (!(o.sigma_pe0 > 0)) o.sigma_pe0 = 1750.0;
    if (!(o.e_cut > 0)) o.e_cut = 0.010;
    if (o.voxel_min_daughters <= 0) o.voxel_min_daughters = 8;
    if (o.stuck_limit <= 0) o.stuck_limit = 8;
    if (!(o.sigma_r0 > 0)) o.sigma_r0 = 7.886e-3;
    if (o.pe_table_per_decade < 0) o.pe_table_per_decade = 0;
    if (o.pe_table_per_decade > 4096) { gn_geometry_destroy(geo); return fail(GN_INVALID_ARGUMENT, "gn_geometry_create: pe_table_per_decade must be <= 4096"); }
    if (o.stuck_limit > 255) { gn_geometry_destroy(geo); return fail(GN_INVALID_ARGUMENT, "gn_geometry_create: stuck_limit must be <= 255 (the per-photon counter of consecutive short steps has 8 bits)"); }
    const bool steps_default = o.steps_per_pass <= 0;
    if (steps_default) o.steps_per_pass = 16;
    if (o.first_pass_steps <= 0) o.first_pass_steps = 1;
    if (o.tail_photons <= 0) o.tail_photons = 148 * 1024;      // measured on configs 2-4: 148 x 512 .. 148 x 4096, best at 1024 (config 2 +7 %)
    const bool regroup_default = o.regroup_percent <= 0;
    o.tol64 = geo->tol64; o.tol32 = geo->tol32;
    geo->opts = o;

    // ---- voxel grids (C5): one uniform 3-D grid per mother = three nested levels of uniform slices, flattened
    std::vector<HostGrid> grids;
    std::vector<int> regular_cell(V, -1);      // leaf box that coincides with one voxel cell of its mother: ix | iy << 10 | iz << 20
    // regular slab: an unrotated leaf box that coincides with a row of cells along ONE axis, alone in each of them (a layer of a
    // sampling calorimeter in a grid whose pitch divides every layer thickness): lowest cell, axis, number of cells, walls
    struct SlabInfo { int cell = -1, axis = 0, span = 0, walls = 0; };
    std::vector<SlabInfo> slab(V);
    std::vector<int> cell_start(1, 0), cand;
    const double shrink = geo->tol64 / 8;
    for (size_t mth = 0; mth < V; ++mth) {
        int nd = kids[mth].y;
        if (nd < o.voxel_min_daughters) continue;
        const HostSolid& ms = solids[node[mth].y];
        double mlo[3], mhi[3];
        if (ms.type == GN_ORB) { mlo[0] = mlo[1] = -ms.a; mhi[0] = mhi[1] = ms.a; }
        else if (ms.type == GN_CONE) { mlo[0] = mlo[1] = -ms.rbound; mhi[0] = mhi[1] = ms.rbound; }
        else if (ms.type == GN_BOX) { mlo[0] = -ms.a; mhi[0] = ms.a; mlo[1] = -ms.b; mhi[1] = ms.b; }
        else { mlo[0] = mlo[1] = -ms.b; mhi[0] = mhi[1] = ms.b; }
        mlo[2] = -ms.c; mhi[2] = ms.c;
        if (ms.type == GN_ORB) { mlo[2] = -ms.a; mhi[2] = ms.a; }
        std::vector<double> blo(3 * (size_t)nd), bhi(3 * (size_t)nd);
        double minext[3] = {1e300, 1e300, 1e300};
        for (int j = 0; j < nd; ++j) {
            int d = dlist[kids[mth].x + j];
            int t = h_placements[4 * (size_t)d + 3];
            const double* Rl = h_transforms + 12 * (size_t)t;
            daughter_bounds(solids[node[d].y], Rl, Rl + 9, &blo[3 * (size_t)j], &bhi[3 * (size_t)j]);
            for (int k = 0; k < 3; ++k) minext[k] = std::min(minext[k], bhi[3 * (size_t)j + k] - blo[3 * (size_t)j + k]);
        }
        HostGrid G;
        double budget = std::max(8.0 * nd, 4096.0);
        for (int k = 0; k < 3; ++k) {
            double L = mhi[k] - mlo[k];
            double f = std::floor(L / std::max(minext[k], L / 1024.0) + 1e-9);
            G.n[k] = (int)std::min(std::max(f, 1.0), 1024.0);
        }
        while ((double)G.n[0] * G.n[1] * G.n[2] > budget) {
            int k = (G.n[0] >= G.n[1] && G.n[0] >= G.n[2]) ? 0 : (G.n[1] >= G.n[2] ? 1 : 2);
            G.n[k] = (G.n[k] + 1) / 2;
        }
        // cell range of daughter j along axis k for a grid of n cells
        auto cell_range = [&](int j, int k, int n, int& a, int& b) {
            const double w = (mhi[k] - mlo[k]) / n, top = n - 1.0;
            double fa = std::floor((blo[3 * (size_t)j + k] + shrink - mlo[k]) / w), fb = std::floor((bhi[3 * (size_t)j + k] - shrink - mlo[k]) / w);
            fa = std::min(std::max(fa, 0.0), top); fb = std::min(std::max(fb, 0.0), top);
            if (fb < fa) fb = fa;
            a = (int)fa; b = (int)fb;
        };
        // daughter j is listed in cell (ix, iy, iz) of a grid of n cells unless the solid itself provably stays clear of it
        // (cell_excluded; margin = 16 delta + rounding, far beyond the 1.25 delta of the probes -- DESIGN.md reading 5)
        const double excl_margin = 8.0 * std::max(geo->tol32, geo->tol64) + 256.0 * ext * 0x1p-23;
        std::vector<char> tight(nd, 1);
        auto in_cell = [&](int j, const int n[3], int ix, int iy, int iz) -> bool {
            if (!tight[j]) return true;
#ifdef GN_AABB_LISTS
            return true;                          // diagnostics: candidate lists by bounding box only
#endif
            const int d = dlist[kids[mth].x + j];
            const double* Rl = h_transforms + 12 * (size_t)h_placements[4 * (size_t)d + 3];
            const int ii[3] = {ix, iy, iz};
            double clo[3], chi[3];
            for (int k = 0; k < 3; ++k) { const double w = (mhi[k] - mlo[k]) / n[k]; clo[k] = mlo[k] + ii[k] * w; chi[k] = mlo[k] + (ii[k] + 1) * w; }
            return !cell_excluded(solids[node[d].y], Rl, Rl + 9, clo, chi, excl_margin);
        };
        // refinement (the smart-voxel idea of choosing the cut that minimises candidate references): while cells hold
        // more than ~1 candidate on average, double the axis whose doubling shortens the lists most, within a budget of
        // 64 cells per daughter.  Short, equally long lists keep the lanes of a warp in step during relocation.
        auto list_stats = [&](const int n[3], double& refs, double& nonempty) {
            std::vector<int> cnt((size_t)n[0] * n[1] * n[2], 0);
            for (int j = 0; j < nd; ++j) {
                int a[3], b[3];
                for (int k = 0; k < 3; ++k) cell_range(j, k, n[k], a[k], b[k]);
                for (int iz = a[2]; iz <= b[2]; ++iz) for (int iy = a[1]; iy <= b[1]; ++iy) for (int ix = a[0]; ix <= b[0]; ++ix)
                    if (in_cell(j, n, ix, iy, iz)) cnt[ix + (size_t)n[0] * (iy + (size_t)n[1] * iz)]++;
            }
            refs = 0; nonempty = 0;
            for (int c : cnt) if (c) { refs += c; nonempty += 1; }
        };
        {
            const double refine_budget = std::max(64.0 * nd, 4096.0);
            double refs, nonempty; list_stats(G.n, refs, nonempty);
            while (nonempty > 0 && refs > 1.25 * nonempty) {
                int best_k = -1; double best_avg = 0.97 * refs / nonempty;
                for (int k = 0; k < 3; ++k) {
                    if (G.n[k] * 2 > 1024 || 2.0 * G.n[0] * G.n[1] * G.n[2] > refine_budget) continue;
                    int t[3] = {G.n[0], G.n[1], G.n[2]}; t[k] *= 2;
                    double r, ne; list_stats(t, r, ne);
                    if (ne > 0 && r / ne < best_avg) { best_avg = r / ne; best_k = k; }
                }
                if (best_k < 0) break;
                G.n[best_k] *= 2;
                list_stats(G.n, refs, nonempty);
            }
        }
        for (int k = 0; k < 3; ++k) { G.gmin[k] = mlo[k]; G.w[k] = (mhi[k] - mlo[k]) / G.n[k]; }
        size_t ncell = (size_t)G.n[0] * G.n[1] * G.n[2];
        G.cell_base = (int)cell_start.size() - 1;
        std::vector<int> count(ncell, 0);
        std::vector<int> c0(3 * (size_t)nd), c1(3 * (size_t)nd);
        for (int j = 0; j < nd; ++j) {
            for (int k = 0; k < 3; ++k) cell_range(j, k, G.n[k], c0[3 * (size_t)j + k], c1[3 * (size_t)j + k]);
            int kept = 0;
            for (int iz = c0[3 * (size_t)j + 2]; iz <= c1[3 * (size_t)j + 2]; ++iz)
                for (int iy = c0[3 * (size_t)j + 1]; iy <= c1[3 * (size_t)j + 1]; ++iy)
                    for (int ix = c0[3 * (size_t)j]; ix <= c1[3 * (size_t)j]; ++ix)
                        kept += in_cell(j, G.n, ix, iy, iz) ? 1 : 0;
            if (kept == 0) tight[j] = 0;          // a daughter outside its mother's grid: listed by its bounding box, as before
            for (int iz = c0[3 * (size_t)j + 2]; iz <= c1[3 * (size_t)j + 2]; ++iz)
                for (int iy = c0[3 * (size_t)j + 1]; iy <= c1[3 * (size_t)j + 1]; ++iy)
                    for (int ix = c0[3 * (size_t)j]; ix <= c1[3 * (size_t)j]; ++ix)
                        if (in_cell(j, G.n, ix, iy, iz)) count[ix + (size_t)G.n[0] * (iy + (size_t)G.n[1] * iz)]++;
        }
        size_t base = cand.size();
        std::vector<size_t> pos(ncell);
        { size_t acc = base; for (size_t c = 0; c < ncell; ++c) { pos[c] = acc; acc += count[c]; cell_start.push_back((int)acc); } cand.resize(acc); }
        for (int j = 0; j < nd; ++j) {           // j ascending = daughter index ascending -> lists stay sorted
            int d = dlist[kids[mth].x + j];
            for (int iz = c0[3 * (size_t)j + 2]; iz <= c1[3 * (size_t)j + 2]; ++iz)
                for (int iy = c0[3 * (size_t)j + 1]; iy <= c1[3 * (size_t)j + 1]; ++iy)
                    for (int ix = c0[3 * (size_t)j]; ix <= c1[3 * (size_t)j]; ++ix)
                        if (in_cell(j, G.n, ix, iy, iz)) cand[pos[ix + (size_t)G.n[0] * (iy + (size_t)G.n[1] * iz)]++] = d;
        }
        // regular voxels: an unrotated leaf box that fills exactly one cell, alone -- in a mother that is a box spanned exactly
        // by the grid (so that cells at the rim are the only ones next to the mother's surface) and whose cells are much
        // wider than the tolerances (the probe distance is a small fraction of a voxel)
        bool regular_mother = ms.type == GN_BOX;
        for (int k = 0; k < 3; ++k) regular_mother = regular_mother && G.w[k] >= 16.0 * std::max(geo->tol32, geo->tol64) + 64.0 * ext * 0x1p-23;
        for (int j = 0; j < nd && regular_mother; ++j) {
            int d = dlist[kids[mth].x + j];
            if (kids[d].y != 0 || solids[node[d].y].type != GN_BOX) continue;
            const double* Rl = h_transforms + 12 * (size_t)h_placements[4 * (size_t)d + 3];
            bool ok = Rl[0] == 1.0 && Rl[4] == 1.0 && Rl[8] == 1.0 && Rl[1] == 0.0 && Rl[2] == 0.0 && Rl[3] == 0.0 && Rl[5] == 0.0 && Rl[6] == 0.0 && Rl[7] == 0.0;
            for (int k = 0; k < 3 && ok; ++k) {
                int a = c0[3 * (size_t)j + k], b = c1[3 * (size_t)j + k];
                ok = a == b && a < 1024 && std::fabs(blo[3 * (size_t)j + k] - (G.gmin[k] + a * G.w[k])) <= geo->tol64 && std::fabs(bhi[3 * (size_t)j + k] - (G.gmin[k] + (a + 1) * G.w[k])) <= geo->tol64;
            }
            if (!ok) continue;
            size_t cell = c0[3 * (size_t)j] + (size_t)G.n[0] * (c0[3 * (size_t)j + 1] + (size_t)G.n[1] * c0[3 * (size_t)j + 2]);
            if (count[cell] != 1) continue;
            regular_cell[d] = c0[3 * (size_t)j] | (c0[3 * (size_t)j + 1] << 10) | (c0[3 * (size_t)j + 2] << 20);
        }
        for (int j = 0; j < nd && regular_mother; ++j) {                   // regular slabs
            int d = dlist[kids[mth].x + j];
            if (regular_cell[d] >= 0 || kids[d].y != 0 || solids[node[d].y].type != GN_BOX) continue;
            const double* Rl = h_transforms + 12 * (size_t)h_placements[4 * (size_t)d + 3];
            bool ok = Rl[0] == 1.0 && Rl[4] == 1.0 && Rl[8] == 1.0 && Rl[1] == 0.0 && Rl[2] == 0.0 && Rl[3] == 0.0 && Rl[5] == 0.0 && Rl[6] == 0.0 && Rl[7] == 0.0;
            int axis = -1, span = 1;
            for (int k = 0; k < 3 && ok; ++k) {
                const int a = c0[3 * (size_t)j + k], b = c1[3 * (size_t)j + k];
                ok = std::fabs(blo[3 * (size_t)j + k] - (G.gmin[k] + a * G.w[k])) <= geo->tol64 && std::fabs(bhi[3 * (size_t)j + k] - (G.gmin[k] + (b + 1) * G.w[k])) <= geo->tol64;
                if (b > a) { ok = ok && axis < 0 && b - a + 1 <= 4096; axis = k; span = b - a + 1; }
            }
            if (!ok || axis < 0) continue;
            int walls = 0;
            for (int k = 0; k < 3; ++k) walls |= (c0[3 * (size_t)j + k] == 0 ? 1 << (2 * k) : 0) | (c1[3 * (size_t)j + k] == G.n[k] - 1 ? 2 << (2 * k) : 0);
            size_t cell0 = c0[3 * (size_t)j] + (size_t)G.n[0] * (c0[3 * (size_t)j + 1] + (size_t)G.n[1] * c0[3 * (size_t)j + 2]);
            const size_t stride = axis == 0 ? 1 : (axis == 1 ? (size_t)G.n[0] : (size_t)G.n[0] * G.n[1]);
            for (int q = 0; q < span && ok; ++q) ok = count[cell0 + q * stride] == 1;
            if (!ok || cell0 + (size_t)span * stride >= (1u << 30)) continue;
            slab[d].cell = (int)cell0; slab[d].axis = axis; slab[d].span = span; slab[d].walls = walls;
        }
        G.mother = (int)mth;
        node[mth].w = (int)grids.size();
        grids.push_back(G);
        geo->n_cells += (int64_t)ncell;
    }
    geo->n_grids = (int64_t)grids.size(); geo->n_cand = (int64_t)cand.size();

    // a solid carries the axis and the number of cells of its regular slabs (SolidRec: cS, sS of a box): every slab placement
    // of one solid must agree, and the mother's grid id must fit the node record; the others stay ordinary boxes
    {
        std::vector<int> s_axis(solids.size(), -1), s_span(solids.size(), 0);
        std::vector<char> s_bad(solids.size(), 0);
        for (size_t i = 0; i < V; ++i) {
            if (slab[i].cell < 0) continue;
            const int si = node[i].y;
            if (node[node[i].x].w > NODE_GRID_MASK) { slab[i].cell = -1; continue; }
            if (s_axis[si] < 0) { s_axis[si] = slab[i].axis; s_span[si] = slab[i].span; }
            else if (s_axis[si] != slab[i].axis || s_span[si] != slab[i].span) s_bad[si] = 1;
        }
        for (size_t i = 0; i < V; ++i) if (slab[i].cell >= 0 && s_bad[node[i].y]) slab[i].cell = -1;
        for (size_t si = 0; si < solids.size(); ++si)
            if (solids[si].type == GN_BOX) { const bool on = s_axis[si] >= 0 && !s_bad[si]; solids[si].cS = on ? s_axis[si] : -1; solids[si].sS = on ? s_span[si] : 1; }
    }

    // ---- sibling hints (store.h NODE_HINT): a full tube whose daughters are one tube-sector solid on a cylindrical lattice --
    // N_phi sectors around, N_z along z, same radii as the mother (a segmented barrel).  A photon that leaves such a sector
    // through ONE of its z or phi faces, farther than 2 probe distances from every other face, can only be in the sibling
    // across that face or in the mother: every other sibling lies behind a second face of the sector left, i.e. farther than
    // delta from the point.  hint[4 d + {0,1,2,3}] = sibling across the lower / upper z face, the start / end phi plane (-1: none)
    std::vector<int> hint(4 * V, -1);
    std::vector<char> hinted(V, 0);
    for (size_t mth = 0; mth < V; ++mth) {
        const int nd = kids[mth].y;
        const HostSolid& ms = solids[node[mth].y];
        if (nd < 8 || ms.type != GN_TUBE || ms.sector || !(ms.a > 0)) continue;
        const int S = node[dlist[kids[mth].x]].y;
        const HostSolid& ss = solids[S];
        const double margin = 2.0 * (1.25 * 0.5 * std::max(geo->tol32, geo->tol64) + 4.0 * ext * 0x1p-23);      // 2 x the fp32 probe distance
        if (ss.type != GN_TUBE || !ss.sector || std::fabs(ss.a - ms.a) > geo->tol64 || std::fabs(ss.b - ms.b) > geo->tol64) continue;
        const double two_pi = 6.283185307179586476925;
        const int n_phi = (int)std::lround(two_pi / ss.dphi), n_z = (int)std::lround(ms.c / ss.c);
        if (n_phi < 3 || n_z < 1 || std::fabs(n_phi * ss.dphi - two_pi) > 1e-9 || std::fabs(n_z * ss.c - ms.c) > geo->tol64) continue;
        if ((size_t)n_phi * n_z > (1u << 24)) continue;
        if (!(2 * ss.c > 16 * margin && ss.b - ss.a > 16 * margin && ss.a * std::sin(ss.dphi) > 16 * margin && ss.dphi < 1.6)) continue;
        std::vector<int> slot((size_t)n_phi * n_z, -1);
        bool ok = true;
        for (int j = 0; j < nd && ok; ++j) {
            const int d = dlist[kids[mth].x + j];
            const double* Rl = h_transforms + 12 * (size_t)h_placements[4 * (size_t)d + 3];
            const double* T = Rl + 9;
            ok = node[d].y == S && std::fabs(Rl[8] - 1.0) < 1e-12 && std::fabs(Rl[2]) < 1e-12 && std::fabs(Rl[5]) < 1e-12 && std::fabs(Rl[6]) < 1e-12 &&
                 std::fabs(Rl[7]) < 1e-12 && std::fabs(Rl[0] - Rl[4]) < 1e-12 && std::fabs(Rl[1] + Rl[3]) < 1e-12 && std::fabs(T[0]) <= geo->tol64 && std::fabs(T[1]) <= geo->tol64;
            if (!ok) break;
            double th = std::atan2(Rl[3], Rl[0]); if (th < 0) th += two_pi;
            const long jj = std::lround(th / ss.dphi);
            const long iz = std::lround((T[2] + ms.c - ss.c) / (2 * ss.c));
            double dth = std::fabs(th - jj * ss.dphi);
            ok = dth < 1e-9 && iz >= 0 && iz < n_z && std::fabs(T[2] - (-ms.c + ss.c * (2 * iz + 1))) <= geo->tol64;
            if (!ok) break;
            int& sl = slot[(size_t)iz * n_phi + (size_t)(jj % n_phi)];
            ok = sl < 0; sl = d;
        }
        if (!ok) continue;
        for (int iz = 0; iz < n_z; ++iz) for (int jp = 0; jp < n_phi; ++jp) {
            const int d = slot[(size_t)iz * n_phi + jp];
            if (d < 0) continue;
            hinted[d] = 1;
            hint[4 * (size_t)d + 0] = iz > 0 ? slot[(size_t)(iz - 1) * n_phi + jp] : -1;
            hint[4 * (size_t)d + 1] = iz + 1 < n_z ? slot[(size_t)(iz + 1) * n_phi + jp] : -1;
            hint[4 * (size_t)d + 2] = slot[(size_t)iz * n_phi + (jp + n_phi - 1) % n_phi];        // across the start plane
            hint[4 * (size_t)d + 3] = slot[(size_t)iz * n_phi + (jp + 1) % n_phi];                // across the end plane
        }
    }
#ifdef GN_NO_HINTS
    std::fill(hinted.begin(), hinted.end(), 0);
#endif

    // ---- per-precision tables (store.h): node records with Tg inline, padded rotations
    std::vector<NodeRec<float>> n32(V); std::vector<NodeRec<double>> n64(V);
    std::vector<float> rot32((size_t)RotStride<float>::value * V, 0.f); std::vector<double> rot64((size_t)RotStride<double>::value * V, 0.0);
    for (size_t i = 0; i < V; ++i) {
        const double* R = &Rg[9 * i];
        bool ident = R[0] == 1.0 && R[4] == 1.0 && R[8] == 1.0 && R[1] == 0.0 && R[2] == 0.0 && R[3] == 0.0 && R[5] == 0.0 && R[6] == 0.0 && R[7] == 0.0;
        for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) {            // M = Rg^T
            rot64[RotStride<double>::value * i + 3 * a + b] = Rg[9 * i + 3 * b + a];
            rot32[RotStride<float>::value * i + 3 * a + b] = (float)Rg[9 * i + 3 * b + a];
        }
        NodeRec<float>& a = n32[i]; NodeRec<double>& b = n64[i];
        a.parent = b.parent = node[i].x;
        a.info = b.info = node[i].y | (ident ? NODE_IDENTITY : 0) | (hinted[i] ? NODE_HINT : 0);
        a.mat = b.mat = node[i].z;
        a.ndau = b.ndau = kids[i].y;
        a.link = b.link = node[i].w >= 0 ? ~node[i].w : kids[i].x;        // voxelised mother: ~grid id
        if (regular_cell[i] >= 0 && node[node[i].x].w <= NODE_GRID_MASK) {
            const int gid = node[node[i].x].w;                              // grid of the mother
            const HostGrid& G = grids[gid];
            const int c[3] = {regular_cell[i] & 1023, (regular_cell[i] >> 10) & 1023, (regular_cell[i] >> 20) & 1023};
            int walls = 0;
            for (int k = 0; k < 3; ++k) walls |= (c[k] == 0 ? 1 << (2 * k) : 0) | (c[k] == G.n[k] - 1 ? 2 << (2 * k) : 0);
            a.info = b.info = a.info | NODE_REGULAR | (gid << NODE_GRID_SHIFT) | (walls << NODE_WALL_SHIFT);
            a.link = b.link = c[0] + G.n[0] * (c[1] + G.n[1] * c[2]);
        } else if (slab[i].cell >= 0) {
            const int gid = node[node[i].x].w;
            a.info = b.info = a.info | NODE_SLAB | (gid << NODE_GRID_SHIFT) | (slab[i].walls << NODE_WALL_SHIFT);
            a.link = b.link = slab[i].cell;
        }
        b.pad = 0;
        for (int k = 0; k < 3; ++k) { b.t[k] = Tg[3 * i + k]; a.t[k] = (float)Tg[3 * i + k]; }
    }
    std::vector<SolidRec<float>> s32; std::vector<SolidRec<double>> s64;
    for (const HostSolid& s : solids) { s32.push_back(make_solid_rec<float>(s)); s64.push_back(make_solid_rec<double>(s)); }
    std::vector<MatRec<float>> m32; std::vector<MatRec<double>> m64;
    for (int i = 0; i < n_mats; ++i) {
        m32.push_back(make_mat_rec<float>(h_materials[3 * i], h_materials[3 * i + 1], h_materials[3 * i + 2], o.sigma_pe0));
        m64.push_back(make_mat_rec<double>(h_materials[3 * i], h_materials[3 * i + 1], h_materials[3 * i + 2], o.sigma_pe0));
    }
    std::vector<GridRec<float>> g32; std::vector<GridRec<double>> g64;
    for (const HostGrid& G : grids) {
        GridRec<float> a; GridRec<double> b;
        const double probe32 = std::max(geo->tol32, (double)(float)(ext * 0x1p-18)), probe64 = geo->tol64;
        for (int k = 0; k < 3; ++k) {
            a.gmin[k] = (float)G.gmin[k]; a.w[k] = (float)G.w[k]; a.inv_w[k] = (float)(1.0 / G.w[k]); a.n[k] = G.n[k];
            b.gmin[k] = G.gmin[k]; b.w[k] = G.w[k]; b.inv_w[k] = 1.0 / G.w[k]; b.n[k] = G.n[k];
            // probe half-width in cell units.  A daughter that is not listed in the cell holding the point can only be
            // occupied / hit if the point (ray) comes within delta = tol / 2 of that cell's boundary: 1.25 delta, plus
            // a guard for the rounding of the index arithmetic itself (a few ulp of the largest cell coordinate).
            const float e32 = (float)(1.25 * 0.5 * probe32 / G.w[k] + 8.0 * G.n[k] * 0x1p-23);
            const double e64 = 1.25 * 0.5 * probe64 / G.w[k] + 8.0 * G.n[k] * 0x1p-52;
            (k == 0 ? a.eps0 : (k == 1 ? a.eps1 : a.eps2)) = e32;
            (k == 0 ? b.eps0 : (k == 1 ? b.eps1 : b.eps2)) = e64;
        }
        a.cell_base = b.cell_base = G.cell_base;
        a.sy = b.sy = G.n[0]; a.sz = b.sz = G.n[0] * G.n[1];
        a.gpad = b.gpad = 0;
        {   // dense: cell c holds exactly the regular voxel with node index base + c
            int base = -1; bool dense = true;
            const size_t ncell = (size_t)G.n[0] * G.n[1] * G.n[2];
            for (size_t c = 0; c < ncell && dense; ++c) {
                const int lo = cell_start[G.cell_base + c], cnt = cell_start[G.cell_base + c + 1] - lo;
                if (cnt != 1) { dense = false; break; }
                const int d = cand[lo];
                if (c == 0) base = d;
                dense = d == base + (int)c && regular_cell[d] >= 0 && (int)c == (regular_cell[d] & 1023) + G.n[0] * (((regular_cell[d] >> 10) & 1023) + G.n[1] * ((regular_cell[d] >> 20) & 1023));
            }
            a.dense = b.dense = dense ? base : -1;
        }
        g32.push_back(a); g64.push_back(b);
    }
    std::vector<int2> cells(cell_start.size() - 1);
    for (size_t c = 0; c + 1 < cell_start.size(); ++c) {
        int cnt = cell_start[c + 1] - cell_start[c];
        cells[c] = make_int2(cnt == 1 ? cand[cell_start[c]] : cell_start[c], cnt);
    }
    {
        bool coherent = true;
        for (size_t i = 0; i < V; ++i) coherent = coherent && solids[node[i].y].type == GN_BOX && (n32[i].info & NODE_IDENTITY);
        for (const int2& c : cells) coherent = coherent && c.y <= 1;
        geo->coherent = coherent;
        size_t n_regular = 0;
        bool has_slabs = false;
        for (size_t i = 0; i < V; ++i) { n_regular += (n32[i].info & (NODE_REGULAR | NODE_SLAB)) ? 1 : 0; has_slabs = has_slabs || (n32[i].info & NODE_SLAB); }
        geo->has_slabs = has_slabs;
        geo->voxel_sched = coherent && 2 * n_regular >= V && geo->opts.no_voxel_pass <= 0 && geo->opts.rayleigh <= 0 && geo->opts.pe_table_per_decade <= 0 && n_solids <= 32 && n_mats <= 32 && grids.size() <= 8 && ext < 0x1p50;      // table sizes: MAX_SMEM_* of common.cuh
        if (regroup_default) geo->opts.regroup_percent = coherent ? 35 : 90;      // swept on configs 2-4 (round 2): 15-50 / 85-95 within 1 %
        if (steps_default && geo->voxel_sched) geo->opts.steps_per_pass = 24;      // the regular-voxel pass is cheap per step: fewer, longer passes (measured)
    }
    if (dry) {
        g_dry->info.resize(V); g_dry->link.resize(V);
        for (size_t i = 0; i < V; ++i) { g_dry->info[i] = n32[i].info; g_dry->link[i] = n32[i].link; }
        g_dry->hint = hint; g_dry->cell_start = cell_start; g_dry->cand = cand; g_dry->grids = grids;
        delete geo;
        *out = nullptr;
        return GN_OK;
    }
    Uploader up{geo};
    const int* d_dlist = up.put(dlist);
    { std::vector<int> dfirst(V); for (size_t i = 0; i < V; ++i) dfirst[i] = kids[i].x; geo->v32.dfirst = geo->v64.dfirst = up.put(dfirst); }
    geo->v32.hint = geo->v64.hint = up.put(hint);
    const int2* d_cells = up.put(cells); const int* d_cand = up.put(cand);
    GeoView<float>& a = geo->v32; GeoView<double>& b = geo->v64;
    a.dlist = b.dlist = d_dlist; a.cells = b.cells = d_cells; a.cand = b.cand = d_cand;
    a.node = up.put(n32); b.node = up.put(n64);
    a.rot = up.put(rot32); b.rot = up.put(rot64);
    a.solids = up.put(s32); b.solids = up.put(s64);
    a.mats = up.put(m32); b.mats = up.put(m64);
    a.grids = up.put(g32); b.grids = up.put(g64);
    a.n_grids = b.n_grids = (int)grids.size();
    {
        std::vector<double> rho(n_mats);
        for (int i = 0; i < n_mats; ++i) rho[i] = h_materials[3 * i + 2];
        a.rho = b.rho = up.put(rho);
    }
    {   // optional physics: Rayleigh factors (reading 18) and the photoelectric table (reading 19), built in
        // fp64 and rounded once per precision
        const int P = o.pe_table_per_decade, points = P > 0 ? 5 * P + 1 : 0;
        std::vector<float> r32(n_mats); std::vector<double> r64(n_mats);
        std::vector<float> t32((size_t)points * n_mats); std::vector<double> t64((size_t)points * n_mats);
        for (int i = 0; i < n_mats; ++i) {
            const double Z = h_materials[3 * i], A = h_materials[3 * i + 1], rho = h_materials[3 * i + 2];
            const double atoms = rho * kNA / A;                            // per cm^3
            r64[i] = atoms * (o.sigma_r0 * kBarn * (Z / 13.0) * (Z / 13.0)) / 10.0; r32[i] = (float)r64[i];
            const double k_edge = 13.6e-6 * (Z - 1.0) * (Z - 1.0);          // MeV
            for (int k = 0; k < points; ++k) {
                const double Ek = 0.01 * std::pow(10.0, (double)k / P);
                double sigma = o.sigma_pe0 * kBarn * std::pow(Z / 82.0, 5.0) * std::pow(0.1 / Ek, 3.5);
                if (o.pe_k_edge > 0 && Ek < k_edge) sigma = sigma / 5.0;  // below the K edge the K shell does not absorb
                t64[(size_t)i * points + k] = atoms * sigma / 10.0; t32[(size_t)i * points + k] = (float)t64[(size_t)i * points + k];
            }
        }
        a.mat_r = up.put(r32); b.mat_r = up.put(r64);
        a.pe_tab = up.put(t32); b.pe_tab = up.put(t64);
        a.rayleigh = b.rayleigh = o.rayleigh > 0 ? 1 : 0;
        a.pe_per_decade = b.pe_per_decade = P; a.pe_points = b.pe_points = points;
    }
    a.tol = (float)geo->tol32; a.delta = a.tol / 2; a.probe = (float)(1.25 * 0.5 * geo->tol32 + 4.0 * ext * 0x1p-23); a.e_cut = (float)o.e_cut;
    b.tol = geo->tol64; b.delta = b.tol / 2; b.probe = 1.25 * 0.5 * geo->tol64 + 4.0 * ext * 0x1p-52; b.e_cut = o.e_cut;
    a.n_nodes = b.n_nodes = n_places; a.n_solids = b.n_solids = n_solids; a.n_mats = b.n_mats = n_mats;
    a.stuck_limit = b.stuck_limit = o.stuck_limit;
    if (!up.ok) {
        std::string e = up.err;
        gn_geometry_destroy(geo);
        return fail(e.find("cudaMalloc") == 0 ? GN_OUT_OF_MEMORY : GN_CUDA_ERROR, "gn_geometry_create: " + e);
    }
    *out = geo;
    return GN_OK;
}

extern "C" int gn_geometry_destroy(gn_geometry* geo) {
    if (!geo) return GN_OK;
    for (void* p : geo->allocations) cudaFree(p);
    if (geo->ws_scratch) cudaFree(geo->ws_scratch);
    if (geo->ws_pinned) cudaFreeHost(geo->ws_pinned);
    if (geo->ws_host_edep) cudaFree(geo->ws_host_edep);
    if (geo->ws_events_ok) for (cudaEvent_t e : geo->ws_events) if (e) cudaEventDestroy(e);
    if (geo->hp_buf) cudaFree(geo->hp_buf);
    if (geo->hp_streams_ok) for (cudaStream_t st : geo->hp_stream) if (st) cudaStreamDestroy(st);
    if (geo->pool) cudaMemPoolDestroy(geo->pool);
    delete geo;
    return GN_OK;
}

extern "C" int32_t gn_geometry_num_places(const gn_geometry* geo) { return geo ? geo->n_places : 0; }
extern "C" double gn_geometry_tolerance(const gn_geometry* geo, int precision) {
    if (!geo) return 0.0;
    return precision == 32 ? geo->tol32 : geo->tol64;
}
extern "C" int gn_geometry_voxel_info(const gn_geometry* geo, int64_t info[4]) {
    if (!geo || !info) return fail(GN_INVALID_ARGUMENT, "gn_geometry_voxel_info: NULL argument");
    info[0] = geo->n_grids; info[1] = geo->n_cells; info[2] = geo->n_cand; info[3] = geo->device_bytes;
    return GN_OK;
}
namespace gn { const char* last_error_cstr(); }
extern "C" const char* gn_last_error(void) { return gn::last_error_cstr(); }
extern "C" const char* gn_version(void) { return "gammanav 0.1 (sm_100a)"; }

// host-only hook (no device needed): the voxel grids, candidate lists, node flags and sibling hints of a geometry, exactly as
// gn_geometry_create builds them, for tests that check them against brute force
extern "C" int gn_host_voxel_tables(const double* h_materials, int32_t n_mats, const int32_t* h_solid_type, const double* h_solid_params,
                                    int32_t n_solids, const int32_t* h_placements, int32_t n_places, const double* h_transforms,
                                    int32_t n_transforms, const gn_opts* h_opts, int64_t counts[3], int32_t* h_node_info,
                                    int32_t* h_node_link, int32_t* h_hint, double* h_grids, int32_t* h_cell_start, int32_t* h_cand) {
    if (!counts) return fail(GN_INVALID_ARGUMENT, "gn_host_voxel_tables: NULL counts");
    HostTables t;
    g_dry = &t;
    gn_geometry* none = nullptr;
    const int rc = gn_geometry_create(h_materials, n_mats, h_solid_type, h_solid_params, n_solids, h_placements, n_places, h_transforms,
                                      n_transforms, h_opts, &none);
    g_dry = nullptr;
    if (rc != GN_OK) return rc;
    counts[0] = (int64_t)t.grids.size(); counts[1] = (int64_t)t.cell_start.size() - 1; counts[2] = (int64_t)t.cand.size();
    if (h_node_info) std::copy(t.info.begin(), t.info.end(), h_node_info);
    if (h_node_link) std::copy(t.link.begin(), t.link.end(), h_node_link);
    if (h_hint) std::copy(t.hint.begin(), t.hint.end(), h_hint);
    if (h_grids) for (size_t i = 0; i < t.grids.size(); ++i) {
        const HostGrid& G = t.grids[i];
        double* o = h_grids + 11 * i;
        o[0] = G.mother; for (int k = 0; k < 3; ++k) { o[1 + k] = G.gmin[k]; o[4 + k] = G.w[k]; o[7 + k] = G.n[k]; }
        o[10] = G.cell_base;
    }
    if (h_cell_start) std::copy(t.cell_start.begin(), t.cell_start.end(), h_cell_start);
    if (h_cand) std::copy(t.cand.begin(), t.cand.end(), h_cand);
    return GN_OK;
}

// host-only hook (no device needed): the composed global -> local transforms the store would hold, M = R_global^T (row-major)
// and T_global per node, for tests that compare them with an independent composition
extern "C" int gn_host_compose_transforms(const int32_t* h_placements, int32_t n_places, const double* h_transforms, int32_t n_transforms,
                                          double* h_M_out, double* h_T_out) {
    if (!h_placements || !h_transforms || !h_M_out || !h_T_out || n_places <= 0 || n_transforms <= 0)
        return fail(GN_INVALID_ARGUMENT, "gn_host_compose_transforms: bad argument");
    std::vector<Affine> global;
    const int st = compose_tree(h_placements, n_places, h_transforms, n_transforms, global);
    if (st != 0) return fail(st == 1 ? GN_INVALID_ARGUMENT : GN_BAD_TREE, "gn_host_compose_transforms: bad placement tree");
    for (int32_t i = 0; i < n_places; ++i) {
        for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) h_M_out[9 * (size_t)i + 3 * a + b] = global[i].R.m[3 * b + a];
        h_T_out[3 * (size_t)i] = global[i].T.x; h_T_out[3 * (size_t)i + 1] = global[i].T.y; h_T_out[3 * (size_t)i + 2] = global[i].T.z;
    }
    return GN_OK;
}
