// hostmath.h -- host-side fp64 set-up arithmetic of the library: small vector / matrix helpers, the source frame
// and the root-down composition of the placement transforms.
// Every sum of three products is evaluated as (p0 + p1) + p2, left to right, so that any other implementation of the
// same definitions that sums in that order gets the same bits.
#pragma once
#include <cmath>
#include <cstddef>
#include <vector>

namespace gn {

struct Vec3d { double x, y, z; };
inline double dot3(const Vec3d& a, const Vec3d& b) { return (a.x * b.x + a.y * b.y) + a.z * b.z; }
inline double norm3(const Vec3d& a) { return std::sqrt(dot3(a, a)); }
inline Vec3d div3(const Vec3d& a, double d) { return Vec3d{a.x / d, a.y / d, a.z / d}; }
inline Vec3d cross3(const Vec3d& a, const Vec3d& b) { return Vec3d{a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
inline double comp3(const Vec3d& a, int k) { return k == 0 ? a.x : (k == 1 ? a.y : a.z); }

// Orthonormal frame of a source: a along the axis; e1 = the coordinate axis nearest to perpendicular (smallest |a_k|,
// ties x < y < z) with its component along a removed, normalised; e2 = a x e1.
struct SourceFrame { Vec3d a, e1, e2; };
inline bool source_frame(const double axis[3], SourceFrame& f) {
    const Vec3d raw{axis[0], axis[1], axis[2]};
    const double len = norm3(raw);
    if (!(len > 0)) return false;
    f.a = div3(raw, len);
    int k = 0;
    for (int i = 1; i < 3; ++i) if (std::fabs(comp3(f.a, i)) < std::fabs(comp3(f.a, k))) k = i;
    const double along = comp3(f.a, k);                               // (unit vector k) . a
    const Vec3d perp{(k == 0 ? 1.0 : 0.0) - along * f.a.x, (k == 1 ? 1.0 : 0.0) - along * f.a.y, (k == 2 ? 1.0 : 0.0) - along * f.a.z};
    f.e1 = div3(perp, norm3(perp));
    f.e2 = cross3(f.a, f.e1);
    return true;
}

// 3 x 3 matrices, row-major
struct Mat3d { double m[9]; };
inline Vec3d row3(const Mat3d& A, int i) { return Vec3d{A.m[3 * i], A.m[3 * i + 1], A.m[3 * i + 2]}; }
inline Vec3d col3(const Mat3d& A, int j) { return Vec3d{A.m[j], A.m[3 + j], A.m[6 + j]}; }
inline Mat3d mul33(const Mat3d& A, const Mat3d& B) {
    Mat3d C;
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) C.m[3 * i + j] = dot3(row3(A, i), col3(B, j));
    return C;
}
inline Vec3d apply3(const Mat3d& A, const Vec3d& v) { return Vec3d{dot3(row3(A, 0), v), dot3(row3(A, 1), v), dot3(row3(A, 2), v)}; }
inline bool orthonormal3(const Mat3d& A, double eps) {
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j)
        if (std::fabs(dot3(row3(A, i), row3(A, j)) - (i == j ? 1.0 : 0.0)) > eps) return false;
    return true;
}

// A placement's own transform (local -> parent) out of the 12-double records: R then T
struct Affine { Mat3d R; Vec3d T; };
inline Affine affine_of(const double* rec) {
    Affine t;
    for (int k = 0; k < 9; ++k) t.R.m[k] = rec[k];
    t.T = Vec3d{rec[9], rec[10], rec[11]};
    return t;
}
// C0: parents come before children, so one sweep composes every node's local -> global transform:
// R_global = R_parent_global R_local, T_global = R_parent_global T_local + T_parent_global.
// status: 0 ok, 1 index out of range, 2 bad tree order, 3 rotation not orthonormal
inline int compose_tree(const int32_t* placements, int32_t n_places, const double* transforms, int32_t n_transforms, std::vector<Affine>& global) {
    global.resize((size_t)n_places);
    for (int32_t i = 0; i < n_places; ++i) {
        const int32_t parent = placements[4 * (size_t)i], t = placements[4 * (size_t)i + 3];
        if (t < 0 || t >= n_transforms) return 1;
        if ((i == 0) != (parent == -1) || parent >= i || parent < -1) return 2;
        const Affine local = affine_of(transforms + 12 * (size_t)t);
        if (!orthonormal3(local.R, 1e-9)) return 3;
        if (parent < 0) { global[i] = local; continue; }
        const Affine& up = global[(size_t)parent];
        const Vec3d moved = apply3(up.R, local.T);
        global[i].R = mul33(up.R, local.R);
        global[i].T = Vec3d{moved.x + up.T.x, moved.y + up.T.y, moved.z + up.T.z};
    }
    return 0;
}

}  // namespace gn
