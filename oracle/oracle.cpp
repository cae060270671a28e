/*
 * oracle.cpp -- plain, slow, single-threaded CPU ORACLE of the gamma transport step loop.
 *
 * TEST INFRASTRUCTURE ONLY (see oracle.h).  Shares nothing with the CUDA path.
 *
 * Every function cites the passage it follows:
 *   P:Lnn      = /root/reference/PAPER.md line nn   (Algorithm 1 = P:L55-76, Eq.1-9 = P:L78-150,
 *                navigation problem statement = P:L120-127, Algorithm 2 = P:L133-144)
 *   S:Cn       = SURVEY.md section 8(c) item Cn     (the readings of what the paper leaves silent)
 *   D:...      = DESIGN.md "Readings" entry
 *
 * Arithmetic is the "canonical arithmetic" of S:C0: only + - * / sqrt, comparisons and |.| in
 * navigation, evaluated left to right as written, compiled with -ffp-contract=off; explicit fma
 * only in the affine transforms and in x + t*w.  Real = float | double per precision mode.
 *
 * Pins (tests/test_oracle_*.py): analytic box/tube distances, dense ray marching of the
 * signed-distance field, brute-force locate with per-level transforms, chained steps vs. sorted
 * analytic crossings, Klein-Nishina quadrature and k->0 limit, Compton energy-momentum
 * conservation, chi^2 of sampled epsilon, slab transmission exp(-mu x), energy book-keeping,
 * Philox vs. cuRAND's host generator, uniform end points; orb closed forms / ray marching and the
 * attenuation-only free paths (the paper's own benchmark) vs. a sorted-chord closed form in numpy
 * (tests/test_oracle_freepath.py); secondary photons (tests/test_oracle_secondaries.py); isotropic safety: points
 * built at a chosen distance off one face of every surface kind, lower bound against DistanceToIn / DistanceToOut in
 * many directions, attained from inside box / tube / orb, never above a ComputeStep (tests/test_oracle_safety.py).
 * PARITY UNPINNED (defined only by SURVEY 8(c)/DESIGN.md, no independent truth exists):
 *   sigma_PE0 normalisation, the capped Bethe-Heitler form, A values, source frame convention,
 *   tolerances, tie-breaks, stuck guard, history hash.
 */
#include "oracle.h"
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#include <algorithm>

namespace {

/* ---- constants (S:C0) ---------------------------------------------------------------- */
const double kMeC2 = 0.51099895;          /* MeV */
const double kRe = 2.8179403262e-13;      /* cm  */
const double kAlpha = 7.2973525693e-3;
const double kNA = 6.02214076e23;
const double kBarn = 1e-24;               /* cm^2 */
const double kPi = 3.14159265358979323846;

template <class R> inline R r_inf() { return std::numeric_limits<R>::infinity(); }
template <class R> inline R r_fma(R a, R b, R c) { return std::fma(a, b, c); }
template <class R> inline R r_abs(R a) { return std::fabs(a); }
template <class R> inline R r_sqrt(R a) { return std::sqrt(a); }
template <class R> inline R r_max(R a, R b) { return a > b ? a : b; }
template <class R> inline R r_min(R a, R b) { return a < b ? a : b; }
/* transcendental functions (physics only; navigation never calls them, S:C0) */
template <class R> inline R r_log(R a) { return std::log(a); }
template <class R> inline R r_exp(R a) { return std::exp(a); }
template <class R> inline R r_cos(R a) { return std::cos(a); }
template <class R> inline R r_sin(R a) { return std::sin(a); }
template <class R> inline R r_pow(R a, R b) { return std::pow(a, b); }

/* ---- operation counter (S:8(d) "instrumented oracle") -------------------------------------------------
 * Counted is a third `Real`: a double whose every operation also bumps a counter, so that one run of the SAME
 * templates gives the algorithmic flops of the workload: + - * / sqrt, compare / min / max / |.| = 1 each,
 * fma = 2, every transcendental = 1 (S:8(d): "a deliberately low count").  Values are plain fp64, so a counted
 * run follows exactly the fp64 histories.  Unary minus, copies and integer index arithmetic are not counted. */
struct OpCounts { uint64_t add, mul, div, sqrt, cmp, fma, trans; };
OpCounts g_ops = {0, 0, 0, 0, 0, 0, 0};
struct Counted {
    double v;
    Counted() = default;
    Counted(double x) : v(x) {}
    explicit operator double() const { return v; }
    Counted operator-() const { return Counted(-v); }
    friend Counted operator+(Counted a, Counted b) { ++g_ops.add; return Counted(a.v + b.v); }
    friend Counted operator-(Counted a, Counted b) { ++g_ops.add; return Counted(a.v - b.v); }
    friend Counted operator*(Counted a, Counted b) { ++g_ops.mul; return Counted(a.v * b.v); }
    friend Counted operator/(Counted a, Counted b) { ++g_ops.div; return Counted(a.v / b.v); }
    friend bool operator<(Counted a, Counted b) { ++g_ops.cmp; return a.v < b.v; }
    friend bool operator>(Counted a, Counted b) { ++g_ops.cmp; return a.v > b.v; }
    friend bool operator<=(Counted a, Counted b) { ++g_ops.cmp; return a.v <= b.v; }
    friend bool operator>=(Counted a, Counted b) { ++g_ops.cmp; return a.v >= b.v; }
    friend bool operator==(Counted a, Counted b) { ++g_ops.cmp; return a.v == b.v; }
    friend bool operator!=(Counted a, Counted b) { ++g_ops.cmp; return a.v != b.v; }
};
template <> inline Counted r_inf<Counted>() { return Counted(std::numeric_limits<double>::infinity()); }
template <> inline Counted r_fma<Counted>(Counted a, Counted b, Counted c) { ++g_ops.fma; return Counted(std::fma(a.v, b.v, c.v)); }
template <> inline Counted r_abs<Counted>(Counted a) { ++g_ops.cmp; return Counted(std::fabs(a.v)); }
template <> inline Counted r_sqrt<Counted>(Counted a) { ++g_ops.sqrt; return Counted(std::sqrt(a.v)); }
template <> inline Counted r_log<Counted>(Counted a) { ++g_ops.trans; return Counted(std::log(a.v)); }
template <> inline Counted r_exp<Counted>(Counted a) { ++g_ops.trans; return Counted(std::exp(a.v)); }
template <> inline Counted r_cos<Counted>(Counted a) { ++g_ops.trans; return Counted(std::cos(a.v)); }
template <> inline Counted r_sin<Counted>(Counted a) { ++g_ops.trans; return Counted(std::sin(a.v)); }
template <> inline Counted r_pow<Counted>(Counted a, Counted b) { ++g_ops.trans; return Counted(std::pow(a.v, b.v)); }
/* the type in which the energy-dependent factors of mu are evaluated (D:"mu factorisation": fp64 in both precision modes) */
template <class R> struct Wide { typedef double type; };
template <> struct Wide<Counted> { typedef Counted type; };
/* operations done in plain double inside an accelerator (grid index arithmetic): counted by hand */
template <class R> inline void note_ops(uint64_t, uint64_t) {}
template <> inline void note_ops<Counted>(uint64_t adds, uint64_t muls) { g_ops.add += adds; g_ops.mul += muls; }

/* ---- geometry store ------------------------------------------------------------------- */
struct SolidD {            /* as given (fp64) */
    int type;
    double a, b, c;        /* BOX: hx,hy,hz   TUBE: rmin,rmax,hz */
    double sphi, dphi;
    bool sector;
    double cS, sS, cE, sE; /* host libm trig of sphi, sphi+dphi (S:C0) */
};
template <class R> struct SolidR {
    int type; R a, b, c; bool sector; R cS, sS, cE, sE;
};
template <class R> struct XformR { R M[9]; R T[3]; };   /* global->local: p = M (x - T)  (S:C0) */

struct Grid {              /* locate accelerator of one mother: uniform grid, padded lists */
    int n[3]; double gmin[3], inv_w[3];
    std::vector<int> start, cand;
};

struct MaterialD { double Z, A, rho; };
template <class R> struct MaterialR { R aPE, aC, aP, capZ; };   /* D:"mu factorisation" */

struct Geo {
    std::vector<MaterialD> mats;
    std::vector<SolidD> solids;
    std::vector<int> parent, solid, material, xform_in;
    std::vector<std::vector<int>> daughters;
    std::vector<double> Rin, Tin;            /* input local->parent transforms per node (9,3) */
    std::vector<XformR<double>> x64; std::vector<XformR<float>> x32;
    std::vector<SolidR<double>> s64; std::vector<SolidR<float>> s32;
    std::vector<MaterialR<double>> m64; std::vector<MaterialR<float>> m32;
    std::vector<XformR<Counted>> xc; std::vector<SolidR<Counted>> sc; std::vector<MaterialR<Counted>> mc;   /* copies of the fp64 tables for the operation counter */
    std::vector<int> grid_of;                /* node -> index in grids or -1 */
    std::vector<Grid> grids;
    double tol64, tol32, sigma_pe0, e_cut; int stuck_limit, grid_min, secondaries;
    int rayleigh = 0, pe_per_decade = 0, pe_k_edge = 0; double sigma_r0 = 0;
    std::vector<double> aR;                       /* Rayleigh material factor n sigma_R0 (Z/13)^2 / 10 [1/mm at 1 MeV], fp64 */
    std::vector<std::vector<double>> pe_tab;      /* per material: mu_PE [1/mm] on the grid E_k = 0.01 MeV 10^(k / P), k = 0 .. 5 P, fp64 */
};

template <class R> struct Sel;
template <> struct Sel<double> {
    static const std::vector<XformR<double>>& x(const Geo& g) { return g.x64; }
    static const std::vector<SolidR<double>>& s(const Geo& g) { return g.s64; }
    static const std::vector<MaterialR<double>>& m(const Geo& g) { return g.m64; }
    static double tol(const Geo& g) { return g.tol64; }
};
template <> struct Sel<Counted> {
    static const std::vector<XformR<Counted>>& x(const Geo& g) { return g.xc; }
    static const std::vector<SolidR<Counted>>& s(const Geo& g) { return g.sc; }
    static const std::vector<MaterialR<Counted>>& m(const Geo& g) { return g.mc; }
    static Counted tol(const Geo& g) { return Counted(g.tol64); }
};
template <> struct Sel<float> {
    static const std::vector<XformR<float>>& x(const Geo& g) { return g.x32; }
    static const std::vector<SolidR<float>>& s(const Geo& g) { return g.s32; }
    static const std::vector<MaterialR<float>>& m(const Geo& g) { return g.m32; }
    static float tol(const Geo& g) { return (float)g.tol32; }
};

/* ---- solids (S:C2) -------------------------------------------------------------------- */
enum { IN = 0, SURFACE = 1, OUT = 2 };

template <class R> inline int classify(R D, R delta) {         /* S:C2 "Inside" */
    if (D > delta) return OUT;
    if (D >= -delta) return SURFACE;
    return IN;
}

/* BOX: s_i = |p_i| - h_i */
template <class R> R box_outsideness(const SolidR<R>& s, const R p[3]) {
    return r_max(r_max(r_abs(p[0]) - s.a, r_abs(p[1]) - s.b), r_abs(p[2]) - s.c);
}
template <class R> int box_inside(const SolidR<R>& s, const R p[3], R delta) { return classify(box_outsideness(s, p), delta); }

/* one planar pair +-h along an axis, exit rule of S:C2: if moving outward and within the band -> 0,
 * else candidate (sign(v) h - p)/v.  Returns false when the answer is 0. */
template <class R> inline bool slab_out(R p, R v, R h, R delta, R& best) {
    if (v > 0) {
        if (p - h >= -delta) return false;
        best = r_min(best, (h - p) / v);
    } else if (v < 0) {
        if (-p - h >= -delta) return false;
        best = r_min(best, (-h - p) / v);
    }
    return true;
}

template <class R> R box_dist_out(const SolidR<R>& s, const R p[3], const R v[3], R delta) {
    R best = r_inf<R>();
    if (!slab_out(p[0], v[0], s.a, delta, best)) return 0;
    if (!slab_out(p[1], v[1], s.b, delta, best)) return 0;
    if (!slab_out(p[2], v[2], s.c, delta, best)) return 0;
    return r_max(best, (R)0);
}

/* S:C2 DistanceToIn BOX: slab method with tolerance */
template <class R> R box_dist_in(const SolidR<R>& s, const R p[3], const R v[3], R delta) {
    const R h[3] = {s.a, s.b, s.c};
    R tmin = -r_inf<R>(), tmax = r_inf<R>();
    for (int i = 0; i < 3; ++i) {
        R si = r_abs(p[i]) - h[i];
        if (si >= -delta && p[i] * v[i] >= 0) return r_inf<R>();
        if (v[i] > 0) {
            tmin = r_max(tmin, (-h[i] - p[i]) / v[i]);
            tmax = r_min(tmax, (h[i] - p[i]) / v[i]);
        } else if (v[i] < 0) {
            tmin = r_max(tmin, (h[i] - p[i]) / v[i]);
            tmax = r_min(tmax, (-h[i] - p[i]) / v[i]);
        }
    }
    if (tmax <= tmin + delta) return r_inf<R>();
    return tmin < delta ? (R)0 : tmin;
}

/* TUBE: rmin=a, rmax=b, hz=c; sector planes s_S = sS x - cS y, s_E = cE y - sE x */
template <class R> R tube_outsideness(const SolidR<R>& s, const R p[3]) {
    R r = r_sqrt(p[0] * p[0] + p[1] * p[1]);
    R D = r_abs(p[2]) - s.c;
    D = r_max(D, r - s.b);
    if (s.a > 0) D = r_max(D, s.a - r);
    if (s.sector) {
        D = r_max(D, s.sS * p[0] - s.cS * p[1]);
        D = r_max(D, s.cE * p[1] - s.sE * p[0]);
    }
    return D;
}
template <class R> int tube_inside(const SolidR<R>& s, const R p[3], R delta) { return classify(tube_outsideness(s, p), delta); }

template <class R> R tube_dist_out(const SolidR<R>& s, const R p[3], const R v[3], R delta) {
    R best = r_inf<R>();
    if (!slab_out(p[2], v[2], s.c, delta, best)) return 0;           /* z planes */
    R a = v[0] * v[0] + v[1] * v[1];
    R b = p[0] * v[0] + p[1] * v[1];
    R r2 = p[0] * p[0] + p[1] * p[1];
    R r = r_sqrt(r2);
    if (a > 0) {
        /* outer cylinder: outward when b > 0; exit = larger root, stable form */
        if (b > 0 && r - s.b >= -delta) return 0;
        R c = r2 - s.b * s.b;
        R Dq = r_max(b * b - a * c, (R)0);
        R t = (b > 0) ? -c / (b + r_sqrt(Dq)) : (-b + r_sqrt(Dq)) / a;
        best = r_min(best, t);
        /* inner cylinder: outward (into the hole) when b < 0; hit = smaller root */
        if (s.a > 0 && b < 0) {
            if (s.a - r >= -delta) return 0;
            R ci = r2 - s.a * s.a;
            R Di = b * b - a * ci;
            if (Di > 0) best = r_min(best, ci / (-b + r_sqrt(Di)));
        }
    }
    if (s.sector) {
        R sS = s.sS * p[0] - s.cS * p[1], dS = s.sS * v[0] - s.cS * v[1];
        if (dS > 0) { if (sS >= -delta) return 0; best = r_min(best, -sS / dS); }
        R sE = s.cE * p[1] - s.sE * p[0], dE = s.cE * v[1] - s.sE * v[0];
        if (dE > 0) { if (sE >= -delta) return 0; best = r_min(best, -sE / dE); }
    }
    return r_max(best, (R)0);
}

template <class R> struct TubeHit {
    const SolidR<R>& s; const R* p; const R* v; R delta;
    R q[3];
    void at(R t) { for (int i = 0; i < 3; ++i) q[i] = r_fma(t, v[i], p[i]); }
    bool ok_z() const { return r_abs(q[2]) <= s.c + delta; }
    bool ok_r() const {
        R r = r_sqrt(q[0] * q[0] + q[1] * q[1]);
        if (r > s.b + delta) return false;
        if (s.a > 0 && r < s.a - delta) return false;
        return true;
    }
    bool ok_phi() const {
        if (!s.sector) return true;
        return (s.sS * q[0] - s.cS * q[1] <= delta) && (s.cE * q[1] - s.sE * q[0] <= delta);
    }
};

/* S:C2 DistanceToIn TUBE: minimum over validated candidates (i)-(iv) */
template <class R> R tube_dist_in(const SolidR<R>& s, const R p[3], const R v[3], R delta) {
    R best = r_inf<R>();
    TubeHit<R> h{s, p, v, delta, {0, 0, 0}};
    R r2 = p[0] * p[0] + p[1] * p[1];
    R r = r_sqrt(r2);
    R a = v[0] * v[0] + v[1] * v[1];
    R b = p[0] * v[0] + p[1] * v[1];
    /* (i) z planes */
    R sz = r_abs(p[2]) - s.c;
    if (sz >= -delta) {
        if (p[2] * v[2] >= 0) return r_inf<R>();
        R t = r_max(sz / r_abs(v[2]), (R)0);
        h.at(t);
        if (h.ok_r() && h.ok_phi()) best = r_min(best, t);
    }
    /* (ii) outer cylinder from outside, must really penetrate the shrunken radius */
    if (a > 0 && b < 0 && r >= s.b - delta) {
        R rs = s.b - delta;
        R cs = r2 - rs * rs;
        if (b * b - a * cs > 0) {
            R c = r2 - s.b * s.b;
            R Dq = b * b - a * c;
            R t = r_max(c / (-b + r_sqrt(Dq)), (R)0);
            h.at(t);
            if (h.ok_z() && h.ok_phi()) best = r_min(best, t);
        }
    }
    /* (iii) inner cylinder: larger root = where the ray leaves the hole */
    if (s.a > 0 && a > 0) {
        R ci = r2 - s.a * s.a;
        R Di = b * b - a * ci;
        if (Di >= 0) {
            R t = (b > 0) ? -ci / (b + r_sqrt(Di)) : (-b + r_sqrt(Di)) / a;
            bool acc = (t >= 0);
            if (!acc && r_abs(r - s.a) <= delta) { acc = true; }
            if (acc) {
                t = r_max(t, (R)0);
                if (b + a * t > 0) {
                    h.at(t);
                    if (h.ok_z() && h.ok_phi()) best = r_min(best, t);
                }
            }
        }
    }
    /* (iv) phi planes */
    if (s.sector) {
        for (int k = 0; k < 2; ++k) {
            R c = k == 0 ? s.cS : s.cE, sn = k == 0 ? s.sS : s.sE;
            R sp = k == 0 ? (s.sS * p[0] - s.cS * p[1]) : (s.cE * p[1] - s.sE * p[0]);
            R dp = k == 0 ? (s.sS * v[0] - s.cS * v[1]) : (s.cE * v[1] - s.sE * v[0]);
            if (sp >= -delta && dp < 0) {
                R t = r_max(sp / (-dp), (R)0);
                h.at(t);
                if (!h.ok_z() || !h.ok_r()) continue;
                if (h.q[0] * c + h.q[1] * sn < 0) continue;          /* correct half of the plane */
                R so = k == 0 ? (s.cE * h.q[1] - s.sE * h.q[0]) : (s.sS * h.q[0] - s.cS * h.q[1]);
                if (so > delta) continue;
                best = r_min(best, t);
            }
        }
    }
    return best;
}

/* ORB (radius a): s = |p| - r.  D:"orb solid" -- the sphere analogue of the S:C2 cylinder rules; the paper only
 * names the solid ("aluminium balls").  Sums are (x.x + y.y) + z.z, left to right. */
template <class R> R orb_outsideness(const SolidR<R>& s, const R p[3]) {
    R rp = r_sqrt((p[0] * p[0] + p[1] * p[1]) + p[2] * p[2]);
    return rp - s.a;
}
template <class R> int orb_inside(const SolidR<R>& s, const R p[3], R delta) { return classify(orb_outsideness(s, p), delta); }
template <class R> R orb_dist_out(const SolidR<R>& s, const R p[3], const R v[3], R delta) {
    R a = (v[0] * v[0] + v[1] * v[1]) + v[2] * v[2];
    R b = (p[0] * v[0] + p[1] * v[1]) + p[2] * v[2];
    R r2 = (p[0] * p[0] + p[1] * p[1]) + p[2] * p[2];
    R rp = r_sqrt(r2);
    if (b > 0 && rp - s.a >= -delta) return 0;                     /* on the surface band, moving outward */
    R c = r2 - s.a * s.a;
    R Dq = r_max(b * b - a * c, (R)0);
    R t = (b > 0) ? -c / (b + r_sqrt(Dq)) : (-b + r_sqrt(Dq)) / a;   /* larger root, cancellation-free form */
    return r_max(t, (R)0);
}
template <class R> R orb_dist_in(const SolidR<R>& s, const R p[3], const R v[3], R delta) {
    R a = (v[0] * v[0] + v[1] * v[1]) + v[2] * v[2];
    R b = (p[0] * v[0] + p[1] * v[1]) + p[2] * v[2];
    R r2 = (p[0] * p[0] + p[1] * p[1]) + p[2] * p[2];
    R rp = r_sqrt(r2);
    if (!(rp >= s.a - delta) || !(b < 0)) return r_inf<R>();       /* inside, or not approaching */
    R rs = s.a - delta;                                            /* the ray must cross the radius shrunk by delta */
    R cs = r2 - rs * rs;
    if (!(b * b - a * cs > 0)) return r_inf<R>();
    R c = r2 - s.a * s.a;
    R Dq = b * b - a * c;
    return r_max(c / (-b + r_sqrt(Dq)), (R)0);                     /* smaller root */
}

/* CONE (solid frustum about z: radius r1 at z = -hz, r2 at z = +hz; the paper names the solid, nothing more).
 * D:"cone solid".  Stored: a = r0 = (r1 + r2)/2, b = m = (r2 - r1)/(2 hz), c = hz, cS = cs = 1/sqrt(1 + m^2) (fp64 on the
 * host, rounded once).  Surface radius u(z) = r0 + m z; s_z = |z| - hz; s_c = (r - u) cs (true distance to the cone).
 * Along a ray, f(t) = r(t)^2 - u(t)^2 = A t^2 + 2 B t + C with du = m v_z, A = (vx^2 + vy^2) - du^2,
 * B = (x vx + y vy) - u du, C = (x^2 + y^2) - u^2; B > 0 <=> moving outward at the surface. */
template <class R> R cone_outsideness(const SolidR<R>& s, const R p[3]) {
    R r = r_sqrt(p[0] * p[0] + p[1] * p[1]);
    R u = s.a + s.b * p[2];
    return r_max(r_abs(p[2]) - s.c, (r - u) * s.cS);
}
template <class R> int cone_inside(const SolidR<R>& s, const R p[3], R delta) { return classify(cone_outsideness(s, p), delta); }
template <class R> R cone_dist_out(const SolidR<R>& s, const R p[3], const R v[3], R delta) {
    R best = r_inf<R>();
    if (!slab_out(p[2], v[2], s.c, delta, best)) return 0;            /* z planes */
    R u = s.a + s.b * p[2], du = s.b * v[2];
    R A = (v[0] * v[0] + v[1] * v[1]) - du * du;
    R B = (p[0] * v[0] + p[1] * v[1]) - u * du;
    R r2 = p[0] * p[0] + p[1] * p[1];
    R C = r2 - u * u;
    if (B > 0 && (r_sqrt(r2) - u) * s.cS >= -delta) return 0;          /* on the cone's band, moving outward */
    R q = r_sqrt(r_max(B * B - A * C, (R)0));
    /* first t > 0 at which f turns positive: -C/(B + q) when B > 0 (any A), else the larger root if A > 0, else never */
    if (B > 0) best = r_min(best, -C / (B + q));
    else if (A > 0) best = r_min(best, (-B + q) / A);
    return r_max(best, (R)0);
}
template <class R> R cone_dist_in(const SolidR<R>& s, const R p[3], const R v[3], R delta) {
    R best = r_inf<R>();
    R u = s.a + s.b * p[2], du = s.b * v[2];
    R r2 = p[0] * p[0] + p[1] * p[1];
    R r = r_sqrt(r2);
    /* (i) end planes: validate against the cone at the hit point */
    R sz = r_abs(p[2]) - s.c;
    if (sz >= -delta) {
        if (p[2] * v[2] >= 0) return r_inf<R>();
        R t = r_max(sz / r_abs(v[2]), (R)0);
        R q[3] = {r_fma(t, v[0], p[0]), r_fma(t, v[1], p[1]), r_fma(t, v[2], p[2])};
        R rq = r_sqrt(q[0] * q[0] + q[1] * q[1]);
        if ((rq - (s.a + s.b * q[2])) * s.cS <= delta) best = r_min(best, t);
    }
    /* (ii) conical surface from outside: the root where f turns from + to - (slope A t + B = -q < 0), i.e.
     * t = (-B - q)/A, evaluated without cancellation: C / (-B + q) when B < 0, (B + q) / (-A) when B >= 0 and A < 0 (a ray
     * steeper than the cone, possibly starting beyond the apex), none otherwise.  The ray must cross the surface moved
     * inwards by delta (no graze loops); z is validated at the hit point (this also rejects the other nappe). */
    if ((r - u) * s.cS >= -delta) {
        R A = (v[0] * v[0] + v[1] * v[1]) - du * du;
        R us = u - delta / s.cS;
        R Bs = (p[0] * v[0] + p[1] * v[1]) - us * du, Cs = r2 - us * us;
        if (Bs * Bs - A * Cs > 0) {
            R B = (p[0] * v[0] + p[1] * v[1]) - u * du, C = r2 - u * u;
            R Dq = B * B - A * C;
            if (Dq > 0) {
                R q = r_sqrt(Dq), t = 0; bool have = false;
                if (B < 0) { t = C / (-B + q); have = true; }
                else if (A < 0) { t = (B + q) / (-A); have = true; }
                if (have) {
                    t = r_max(t, (R)0);
                    R zq = r_fma(t, v[2], p[2]);
                    if (r_abs(zq) <= s.c + delta && (B + A * t) < 0) best = r_min(best, t);      /* moving inward there */
                }
            }
        }
    }
    return best;
}

/* Outward unit normal of the bounding surface a point q (local frame) lies on -- "what is the normal of the boundary
 * surface at that point?".  D:"surface normal": the surface is the one whose signed outsideness s_k(q) is the
 * largest (the one q is on, or nearest to; ties -> first in the order listed), the normal is the gradient of that s_k:
 *   BOX   s_i = |q_i| - h_i, i = x, y, z                       n = sign(q_i) e_i          (q_i = 0 counts as +)
 *   TUBE  s_z = |z| - hz; s_out = r - rmax; s_in = rmin - r; s_S; s_E     n = sign(z) e_z; (x, y, 0)/r; -(x, y, 0)/r;
 *                                                              (sS, -cS, 0); (-sE, cE, 0)
 *   ORB   n = q / |q|
 *   CONE  s_z, s_c = (r - u(z)) cs                             n = sign(z) e_z; cs (x/r, y/r, -m)
 * (r = 0 on a cylinder or |q| = 0 on an orb cannot be on the surface; the x axis is returned.) */
template <class R> void solid_normal(const SolidR<R>& s, const R q[3], R n[3]) {
    n[0] = n[1] = n[2] = 0;
    if (s.type == ORACLE_BOX) {
        const R h[3] = {s.a, s.b, s.c};
        int k = 0; R best = r_abs(q[0]) - h[0];
        for (int i = 1; i < 3; ++i) { R si = r_abs(q[i]) - h[i]; if (si > best) { best = si; k = i; } }
        n[k] = q[k] < 0 ? (R)-1 : (R)1;
        return;
    }
    if (s.type == ORACLE_ORB) {
        R rp = r_sqrt((q[0] * q[0] + q[1] * q[1]) + q[2] * q[2]);
        if (!(rp > 0)) { n[0] = 1; return; }
        n[0] = q[0] / rp; n[1] = q[1] / rp; n[2] = q[2] / rp;
        return;
    }
    if (s.type == ORACLE_CONE) {                  /* surfaces: z planes, cone; grad s_c = cs (x/r, y/r, -m) */
        R rc = r_sqrt(q[0] * q[0] + q[1] * q[1]);
        R sz = r_abs(q[2]) - s.c, sc = (rc - (s.a + s.b * q[2])) * s.cS;
        if (!(sc > sz)) { n[2] = q[2] < 0 ? (R)-1 : (R)1; return; }
        if (!(rc > 0)) { n[0] = 1; return; }
        n[0] = (q[0] / rc) * s.cS; n[1] = (q[1] / rc) * s.cS; n[2] = -s.b * s.cS;
        return;
    }
    R r = r_sqrt(q[0] * q[0] + q[1] * q[1]);
    int k = 0; R best = r_abs(q[2]) - s.c;
    { R so = r - s.b; if (so > best) { best = so; k = 1; } }
    if (s.a > 0) { R si = s.a - r; if (si > best) { best = si; k = 2; } }
    if (s.sector) {
        R sS = s.sS * q[0] - s.cS * q[1]; if (sS > best) { best = sS; k = 3; }
        R sE = s.cE * q[1] - s.sE * q[0]; if (sE > best) { best = sE; k = 4; }
    }
    if (k == 0) n[2] = q[2] < 0 ? (R)-1 : (R)1;
    else if (k == 1 || k == 2) {
        if (!(r > 0)) { n[0] = 1; return; }
        R sg = k == 1 ? (R)1 : (R)-1;
        n[0] = sg * (q[0] / r); n[1] = sg * (q[1] / r);
    } else if (k == 3) { n[0] = s.sS; n[1] = -s.cS; }
    else { n[0] = -s.sE; n[1] = s.cE; }
}

/* the "fork" on solid type */
/* Isotropic safety (S:8(f) NEXT-4, D:reading 17): every s of S:C2 is the signed distance of p to ONE bounding surface's
 * half-space / cylinder / sphere / cone (negative inside), and the solid is the intersection of those sets.  So for a
 * point inside, min_i(-s_i) = -D is the distance to the nearest bounding surface (no boundary is nearer: a lower bound
 * of the exit distance in EVERY direction; exact for box, tube and orb, a lower bound for the cone, whose (r - u) cs is
 * the distance to the generator LINE); for a point outside, dist(p, intersection) >= max_i dist(p, set_i) = D. */
template <class R> R solid_outsideness(const SolidR<R>& s, const R p[3]) {
    return s.type == ORACLE_BOX ? box_outsideness(s, p) : (s.type == ORACLE_TUBE ? tube_outsideness(s, p) : (s.type == ORACLE_ORB ? orb_outsideness(s, p) : cone_outsideness(s, p)));
}
template <class R> R solid_safety_out(const SolidR<R>& s, const R p[3]) { return r_max(-solid_outsideness(s, p), (R)0); }
template <class R> R solid_safety_in(const SolidR<R>& s, const R p[3]) { return r_max(solid_outsideness(s, p), (R)0); }

template <class R> int solid_inside(const SolidR<R>& s, const R p[3], R delta) {
    return s.type == ORACLE_BOX ? box_inside(s, p, delta) : (s.type == ORACLE_TUBE ? tube_inside(s, p, delta) : (s.type == ORACLE_ORB ? orb_inside(s, p, delta) : cone_inside(s, p, delta)));
}
template <class R> R solid_dist_in(const SolidR<R>& s, const R p[3], const R v[3], R delta) {
    return s.type == ORACLE_BOX ? box_dist_in(s, p, v, delta) : (s.type == ORACLE_TUBE ? tube_dist_in(s, p, v, delta) : (s.type == ORACLE_ORB ? orb_dist_in(s, p, v, delta) : cone_dist_in(s, p, v, delta)));
}
template <class R> R solid_dist_out(const SolidR<R>& s, const R p[3], const R v[3], R delta) {
    return s.type == ORACLE_BOX ? box_dist_out(s, p, v, delta) : (s.type == ORACLE_TUBE ? tube_dist_out(s, p, v, delta) : (s.type == ORACLE_ORB ? orb_dist_out(s, p, v, delta) : cone_dist_out(s, p, v, delta)));
}

/* ---- navigator (S:C3, S:C4) ------------------------------------------------------------ */
template <class R> struct Navigator {
    const Geo& g; bool use_grid; R tol, delta;
    const std::vector<XformR<R>>& X; const std::vector<SolidR<R>>& S;
    Navigator(const Geo& geo, bool grid)
        : g(geo), use_grid(grid), tol(Sel<R>::tol(geo)), delta(Sel<R>::tol(geo) / 2), X(Sel<R>::x(geo)), S(Sel<R>::s(geo)) {}

    /* S:C0 affine transform with the explicit fma placement */
    void local_point(int node, const R x[3], R p[3]) const {
        const XformR<R>& t = X[node];
        R d[3] = {x[0] - t.T[0], x[1] - t.T[1], x[2] - t.T[2]};
        for (int k = 0; k < 3; ++k) p[k] = r_fma(t.M[3 * k + 2], d[2], r_fma(t.M[3 * k + 1], d[1], t.M[3 * k] * d[0]));
    }
    void local_dir(int node, const R w[3], R v[3]) const {
        const XformR<R>& t = X[node];
        for (int k = 0; k < 3; ++k) v[k] = r_fma(t.M[3 * k + 2], w[2], r_fma(t.M[3 * k + 1], w[1], t.M[3 * k] * w[0]));
    }
    /* S:C3 occupies */
    bool occupies(int node, const R x[3], const R* w) const {
        R p[3]; local_point(node, x, p);
        const SolidR<R>& s = S[g.solid[node]];
        int c = solid_inside(s, p, delta);
        if (c == IN) return true;
        if (c == OUT) return false;
        if (!w) return true;
        R v[3]; local_dir(node, w, v);
        return solid_dist_out(s, p, v, delta) > 0;
    }
    /* descend from an occupied node through first-occupying daughters in index order (S:C3) */
    int descend(int cur, const R x[3], const R* w) const {
        for (;;) {
            int found = -1;
            int gi = use_grid ? g.grid_of[cur] : -1;
            if (gi >= 0) {
                /* accelerator: candidates of the grid cell holding the local point; padded lists are a
                 * superset of every daughter that could occupy, kept in index order */
                const Grid& G = g.grids[gi];
                R p[3]; local_point(cur, x, p);
                int c[3];
                note_ops<R>(3, 3);                       /* (p - gmin) * inv_w per axis, in plain double below */
                for (int k = 0; k < 3; ++k) {
                    double f = std::floor(((double)p[k] - G.gmin[k]) * G.inv_w[k]);
                    c[k] = (int)std::min(std::max(f, 0.0), (double)(G.n[k] - 1));
                }
                int cell = c[0] + G.n[0] * (c[1] + G.n[1] * c[2]);
                for (int i = G.start[cell]; i < G.start[cell + 1]; ++i)
                    if (occupies(G.cand[i], x, w)) { found = G.cand[i]; break; }
            } else {
                for (int d : g.daughters[cur]) if (occupies(d, x, w)) { found = d; break; }
            }
            if (found < 0) return cur;
            cur = found;
        }
    }
    /* Isotropic safety of point x in volume vol (S:8(f) NEXT-4, D:reading 17): plain linear scan -- the smaller of
     * SafetyToOut of vol's own solid and SafetyToIn of every daughter of vol, in index order.  No boundary of vol or of
     * one of its daughters is nearer than this in any direction.  vol = -1 -> 0. */
    R safety(int vol, const R x[3]) const {
        if (vol < 0) return 0;
        R p[3]; local_point(vol, x, p);
        R best = solid_safety_out(S[g.solid[vol]], p);
        for (int d : g.daughters[vol]) {
            R q[3]; local_point(d, x, q);
            best = r_min(best, solid_safety_in(S[g.solid[d]], q));
        }
        return best;
    }
    int locate(const R x[3], const R* w) const {
        if (!occupies(0, x, w)) return -1;
        return descend(0, x, w);
    }
    /* S:C4 relocate: climb while not occupied, then descend */
    int relocate(int X0, const R x[3], const R* w) const {
        int cur = X0;
        while (cur != -1 && !occupies(cur, x, w)) cur = g.parent[cur];
        if (cur == -1) return -1;
        return descend(cur, x, w);
    }
    /* S:C4 ComputeStep, plain definition: linear scan over all daughters */
    void compute_step(int vol, const R x[3], const R w[3], R max_step, R& step, int& next) const {
        if (vol < 0) { step = r_inf<R>(); next = -1; return; }
        R p[3], v[3];
        local_point(vol, x, p); local_dir(vol, w, v);
        R best = solid_dist_out(S[g.solid[vol]], p, v, delta);
        for (int d : g.daughters[vol]) {
            local_point(d, x, p); local_dir(d, w, v);
            R t = solid_dist_in(S[g.solid[d]], p, v, delta);
            if (t < best) best = t;
        }
        if (best > max_step) { step = r_inf<R>(); next = vol; return; }
        step = best;
        R xn[3] = {r_fma(best, w[0], x[0]), r_fma(best, w[1], x[1]), r_fma(best, w[2], x[2])};
        next = relocate(vol, xn, w);
    }
    /* ComputeStep that also answers "what is the normal of the boundary surface at that point?": the outward
     * normal, in the global frame, of the solid whose surface ends the step -- the current volume's own solid (exit), or
     * the daughter entered (strict <: ties favour the mother, then the lowest daughter index, S:C4).  No boundary within
     * max_step -> normal (0,0,0).  Local -> global: n_g[k] = fma(M[2][k], n.z, fma(M[1][k], n.y, M[0][k] n.x)) (M = X.M). */
    void compute_step_normal(int vol, const R x[3], const R w[3], R max_step, R& step, int& next, R ng[3]) const {
        ng[0] = ng[1] = ng[2] = 0;
        if (vol < 0) { step = r_inf<R>(); next = -1; return; }
        R p[3], v[3];
        local_point(vol, x, p); local_dir(vol, w, v);
        R best = solid_dist_out(S[g.solid[vol]], p, v, delta);
        int hit = vol;
        for (int d : g.daughters[vol]) {
            local_point(d, x, p); local_dir(d, w, v);
            R t = solid_dist_in(S[g.solid[d]], p, v, delta);
            if (t < best) { best = t; hit = d; }
        }
        if (best > max_step) { step = r_inf<R>(); next = vol; return; }
        step = best;
        R xn[3] = {r_fma(best, w[0], x[0]), r_fma(best, w[1], x[1]), r_fma(best, w[2], x[2])};
        R q[3], nl[3];
        local_point(hit, xn, q);
        solid_normal(S[g.solid[hit]], q, nl);
        const XformR<R>& t = X[hit];
        for (int k = 0; k < 3; ++k) ng[k] = r_fma(t.M[6 + k], nl[2], r_fma(t.M[3 + k], nl[1], t.M[k] * nl[0]));
        next = relocate(vol, xn, w);
    }
};

/* ---- physics (S:C6) -------------------------------------------------------------------- */
/* Klein-Nishina total cross-section per electron, cm^2 */
template <class W> W sigma_kn_over_2pire2(W k) {          /* sigma_KN / (2 pi r_e^2), S:C6 closed form */
    W l = r_log<W>(W(1.0) + W(2.0) * k);
    W t1 = (W(1.0) + k) / (k * k) * (W(2.0) * (W(1.0) + k) / (W(1.0) + W(2.0) * k) - l / k);
    W t2 = l / (W(2.0) * k);
    W t3 = (W(1.0) + W(3.0) * k) / ((W(1.0) + W(2.0) * k) * (W(1.0) + W(2.0) * k));
    return t1 + t2 - t3;
}
double sigma_kn(double k) { return 2.0 * kPi * kRe * kRe * sigma_kn_over_2pire2<double>(k); }
double pair_cap(double Z) { return (28.0 / 9.0) * std::log(183.0 * std::pow(Z, -1.0 / 3.0)) - 2.0 / 27.0; }
double sigma_pair(double k, double Z) {
    if (!(k > 2.0)) return 0.0;
    double P = std::min((28.0 / 9.0) * std::log(2.0 * k) - 218.0 / 27.0, pair_cap(Z));
    return kAlpha * kRe * kRe * Z * Z * std::max(P, 0.0);
}
double sigma_pe(double E, double Z, double s0_barn) {
    return s0_barn * kBarn * std::pow(Z / 82.0, 5.0) * std::pow(0.1 / E, 3.5);
}

/* D:"mu factorisation": energy factors are evaluated in fp64 from E and rounded once to Real;
 * material factors are evaluated in fp64 at create time and rounded once to Real; the products and
 * the sum are in Real.  In fp64 mode this is the closed form of S:C6 evaluated in a fixed order. */
template <class R> struct EnergyFactors { R gPE, gKN, L2k; bool above_pair; };
template <class R> EnergyFactors<R> energy_factors(R E) {
    typedef typename Wide<R>::type W;
    W e = W((double)E), k = e / W(kMeC2);
    EnergyFactors<R> f;
    /* (0.1 / E)^3.5 as x x x sqrt(x), x = 0.1 / E (D:reading 1): products, one division and one square root are correctly
     * rounded by every IEEE-754 implementation, a library pow is not -- host and device libm differ in the last bit */
    { const W xq = W(0.1) / e; f.gPE = (R)(double)(((xq * xq) * xq) * r_sqrt<W>(xq)); }
    const W two_pi_re2(2.0 * kPi * kRe * kRe);
    f.gKN = (R)(double)((two_pi_re2 * sigma_kn_over_2pire2<W>(k)) / two_pi_re2);      /* sigma_KN(k) / (2 pi r_e^2), as D:reading 1 writes it */
    f.L2k = (R)(double)r_log<W>(W(2.0) * k);
    f.above_pair = k > W(2.0);
    return f;
}
template <class R> void mu_partials(const MaterialR<R>& m, const EnergyFactors<R>& f, R mu[3]) {
    mu[0] = m.aPE * f.gPE;
    mu[1] = m.aC * f.gKN;
    R P = r_min((R)(28.0 / 9.0) * f.L2k - (R)(218.0 / 27.0), m.capZ);
    mu[2] = (f.above_pair && P > 0) ? m.aP * P : (R)0;
}

/* D:reading 19, tabulated photoelectric coefficient.  Grid E_k = E_min 10^(k / P), E_min = 0.01 MeV, k = 0 .. 5 P (1 GeV).
 * Table (fp64, at create time): T_k = n sigma_PE(E_k) / 10 with sigma_PE = sigma_PE0 (Z/82)^5 (0.1/E)^3.5, divided by the K jump
 * ratio 5 below E_K = 13.6e-6 MeV (Z - 1)^2 when the edge model is on; rounded once to Real.
 * Look-up: u = clamp((ln E - ln E_min) P / ln 10, 0, 5 P (1 - 2^-24)) in fp64, rounded once to Real, evaluated when the energy
 * changes; per step i = floor(u), f = u - i, mu_PE = T_i + f (T_{i+1} - T_i) in Real, left to right. */
const double kPeEmin = 0.01, kPeDecades = 5.0, kKJump = 5.0;
double pe_sigma_tab(double E, double Z, double s0_barn, int k_edge) {
    double s = s0_barn * kBarn * std::pow(Z / 82.0, 5.0) * std::pow(0.1 / E, 3.5);
    if (k_edge) { double eK = 13.6e-6 * (Z - 1.0) * (Z - 1.0); if (E < eK) s = s / kKJump; }
    return s;
}
template <class R> R pe_table_coordinate(R E, int per_decade) {
    typedef typename Wide<R>::type W;
    W u = (r_log<W>(W((double)E)) - W(std::log(kPeEmin))) * W((double)per_decade / std::log(10.0));
    const W top(kPeDecades * per_decade * (1.0 - 0x1p-24));
    if (u < W(0.0)) u = W(0.0);
    if (u > top) u = top;
    return (R)(double)u;
}
template <class R> R pe_table_mu(const std::vector<double>& T, R u) {
    int i = (int)std::floor((double)u);
    R f = u - (R)(double)i;
    R t0 = (R)T[i], t1 = (R)T[i + 1];
    return t0 + f * (t1 - t0);
}
/* D:reading 18, Rayleigh: mu_R = aR gR, aR = n sigma_R0 (Z/13)^2 / 10 (fp64 at create time, rounded once), gR = 1 / (E E)
 * evaluated in Real (one product, one division) */
template <class R> R mu_rayleigh(const Geo& g, int material, R E) {
    if (!g.rayleigh) return (R)0;
    return (R)g.aR[material] * ((R)1 / (E * E));
}
/* the four partial coefficients of material `mat` for a photon of energy E (factors f, table coordinate u) */
template <class R> void mu_all(const Geo& g, int mat, R E, const EnergyFactors<R>& f, R u_pe, R mu4[4]) {
    R m3[3]; mu_partials(Sel<R>::m(g)[mat], f, m3);
    mu4[0] = g.pe_per_decade > 0 ? pe_table_mu<R>(g.pe_tab[mat], u_pe) : m3[0];
    mu4[1] = m3[1];
    mu4[2] = mu_rayleigh<R>(g, mat, E);
    mu4[3] = m3[2];
}

/* ---- RNG (S:C7) ------------------------------------------------------------------------ */
void philox4x32_10(uint32_t c[4], uint32_t k0, uint32_t k1) {
    for (int r = 0; r < 10; ++r) {
        if (r > 0) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
        uint64_t p0 = (uint64_t)0xD2511F53u * c[0];
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c[2];
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
    }
}
template <class R> R uniform_from_lane(uint64_t lane);
template <> double uniform_from_lane<double>(uint64_t lane) { return (double)((lane >> 11) + 1) * 0x1p-53; }
template <> float uniform_from_lane<float>(uint64_t lane) { return (float)((lane >> 40) + 1) * 0x1p-24f; }
template <> Counted uniform_from_lane<Counted>(uint64_t lane) { ++g_ops.mul; return Counted((double)((lane >> 11) + 1) * 0x1p-53); }

struct Stream {      /* draw j of photon id: lane (j mod 2) of block j/2; tag 0 = the primary, 1 / 2 = its annihilation photons */
    uint64_t seed, id; uint32_t j; uint32_t tag = 0;
    uint64_t lane() {
        uint32_t c[4] = {(uint32_t)id, (uint32_t)(id >> 32), j >> 1, tag};
        philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
        uint64_t l = (j & 1) ? ((uint64_t)c[2] | ((uint64_t)c[3] << 32)) : ((uint64_t)c[0] | ((uint64_t)c[1] << 32));
        ++j;
        return l;
    }
    template <class R> R u() { return uniform_from_lane<R>(lane()); }
};

/* ---- sampling (S:C7) ------------------------------------------------------------------- */
/* Klein-Nishina composition-rejection on eps = E'/E */
template <class R> int kn_sample(R E, Stream& rng, R& eps, R& cost, R& sint2) {
    R k = E / (R)kMeC2;
    R eps0 = (R)1 / ((R)1 + (R)2 * k);
    R a1 = -r_log(eps0);
    R eps0sq = eps0 * eps0;
    R a2 = ((R)1 - eps0sq) / (R)2;
    int trials = 0;
    for (;;) {
        ++trials;
        R u1 = rng.u<R>(), u2 = rng.u<R>(), u3 = rng.u<R>();
        R e, e2;
        if (u1 < a1 / (a1 + a2)) { e = r_exp(-a1 * u2); e2 = e * e; }
        else { e2 = eps0sq + ((R)1 - eps0sq) * u2; e = r_sqrt(e2); }
        R t = ((R)1 - e) / (k * e);
        R s2 = t * ((R)2 - t);
        if ((R)1 - e * s2 / ((R)1 + e2) >= u3) { eps = e; cost = (R)1 - t; sint2 = s2; return trials; }
    }
}
/* direction update */
template <class R> void rotate_dir(R w[3], R cost, R sint, R phi) {
    R cp = r_cos(phi), sp = r_sin(phi);
    R u = w[0], v = w[1], ww = w[2];
    R s2 = u * u + v * v;
    R n[3];
    if (s2 >= (R)1e-10) {
        R s = r_sqrt(s2);
        n[0] = u * cost + sint * (u * ww * cp - v * sp) / s;
        n[1] = v * cost + sint * (v * ww * cp + u * sp) / s;
        n[2] = ww * cost - s * sint * cp;
    } else {
        n[0] = sint * cp; n[1] = sint * sp; n[2] = (ww < 0 ? -cost : cost);
    }
    R nn = r_sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
    w[0] = n[0] / nn; w[1] = n[1] / nn; w[2] = n[2] / nn;
}

/* Rayleigh angle (D:reading 18): cos(theta) from p(c) ~ 1 + c^2 on [-1, 1] by rejection, two draws per trial:
 * c = 2 U1 - 1, accepted when 2 U2 <= 1 + c c.  Only + - * and a comparison: the same bits everywhere. */
template <class R> int rayleigh_sample(Stream& rng, R& cost) {
    int trials = 0;
    for (;;) {
        ++trials;
        R u1 = rng.u<R>(), u2 = rng.u<R>();
        R c = (R)2 * u1 - (R)1;
        if ((R)2 * u2 <= (R)1 + c * c) { cost = c; return trials; }
    }
}

/* ---- source (S:C8, D:"source frame") ---------------------------------------------------- */
template <class R> struct SourceR {
    int kind, energy_kind;
    R o[3], a[3], e1[3], e2[3];
    R sigma, cos_half, e0, ln_e0, ln_ratio;
};
template <class R> bool make_source(const oracle_source_t& s, SourceR<R>& o) {
    double n = std::sqrt(s.axis[0] * s.axis[0] + s.axis[1] * s.axis[1] + s.axis[2] * s.axis[2]);
    if (!(n > 0)) return false;
    double a[3] = {s.axis[0] / n, s.axis[1] / n, s.axis[2] / n};
    int m = 0;                                                       /* smallest |a_i|, ties x<y<z */
    if (std::fabs(a[1]) < std::fabs(a[m])) m = 1;
    if (std::fabs(a[2]) < std::fabs(a[m])) m = 2;
    double h[3] = {0, 0, 0}; h[m] = 1;
    double ha = a[m];
    double e1[3] = {h[0] - ha * a[0], h[1] - ha * a[1], h[2] - ha * a[2]};
    double n1 = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
    for (int i = 0; i < 3; ++i) e1[i] /= n1;
    double e2[3] = {a[1] * e1[2] - a[2] * e1[1], a[2] * e1[0] - a[0] * e1[2], a[0] * e1[1] - a[1] * e1[0]};
    o.kind = s.kind; o.energy_kind = s.energy_kind;
    for (int i = 0; i < 3; ++i) { o.o[i] = (R)s.origin[i]; o.a[i] = (R)a[i]; o.e1[i] = (R)e1[i]; o.e2[i] = (R)e2[i]; }
    o.sigma = (R)s.sigma; o.cos_half = (R)std::cos(s.half_angle);
    o.e0 = (R)s.e0;
    if (s.energy_kind == ORACLE_E_LOGUNIFORM) {
        if (!(s.e0 > 0) || !(s.e1 >= s.e0)) return false;
        o.ln_e0 = (R)std::log(s.e0); o.ln_ratio = (R)std::log(s.e1 / s.e0);
    } else { o.ln_e0 = 0; o.ln_ratio = 0; }
    return s.e0 > 0;
}
template <class R> void sample_source(const SourceR<R>& s, Stream& rng, R x[3], R w[3], R& E) {
    const R twopi = (R)6.283185307179586;
    for (int i = 0; i < 3; ++i) { x[i] = s.o[i]; w[i] = s.a[i]; }
    if (s.kind == ORACLE_SRC_GAUSS_PENCIL) {
        R u0 = rng.u<R>(), u1 = rng.u<R>();
        R r = s.sigma * r_sqrt((R)-2 * r_log(u0));
        R phi = twopi * u1;
        R gx = r * r_cos(phi), gy = r * r_sin(phi);
        for (int i = 0; i < 3; ++i) x[i] = s.o[i] + (gx * s.e1[i] + gy * s.e2[i]);
    } else if (s.kind == ORACLE_SRC_CONE || s.kind == ORACLE_SRC_ISOTROPIC) {
        R u0 = rng.u<R>(), u1 = rng.u<R>();
        R ct = (s.kind == ORACLE_SRC_CONE) ? (R)1 - u0 * ((R)1 - s.cos_half) : (R)1 - (R)2 * u0;
        R st = r_sqrt(r_max(((R)1 - ct) * ((R)1 + ct), (R)0));
        R phi = twopi * u1;
        R cx = st * r_cos(phi), cy = st * r_sin(phi);
        R n[3];
        for (int i = 0; i < 3; ++i) n[i] = (cx * s.e1[i] + cy * s.e2[i]) + ct * s.a[i];
        R nn = r_sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
        for (int i = 0; i < 3; ++i) w[i] = n[i] / nn;
    }
    if (s.energy_kind == ORACLE_E_LOGUNIFORM) E = r_exp(s.ln_e0 + rng.u<R>() * s.ln_ratio);
    else E = s.e0;
}

/* ---- transport loop (Algorithm 1 generalised, S:C9) ---------------------------- */
/* History hash (S:C9): FNV-1a, 64 bit -- offset basis 0xcbf29ce484222325, per byte h = (h xor byte) * 0x100000001b3 mod 2^64 --
 * over the bytes of the 32-bit words (vol_before, event) of every step, least significant byte first. */
const uint64_t kFnvOffset = 0xcbf29ce484222325ull, kFnvPrime = 0x100000001b3ull;
inline void fnv_byte(uint64_t& h, uint8_t b) { h ^= b; h *= kFnvPrime; }
inline void fnv_word(uint64_t& h, uint32_t w) {
    for (int i = 0; i < 4; ++i) fnv_byte(h, (uint8_t)((w >> (8 * i)) & 0xffu));
}
enum { EV_BOUNDARY = 0, EV_PE = 1, EV_COMPTON = 2, EV_PAIR = 3, EV_CUT = 4, EV_ESCAPE = 5, EV_STUCK = 6, EV_RAYLEIGH = 7 };

/* One history from (x, w, E) with stream rng: locate, first optical depth, then the loop of Algorithm 1.
 * Returns the history hash and the step count; E holds the energy at the end.  With g.secondaries (S:8(f) NEXT-3,
 * D:reading 16) a pair event deposits E - 2 me c^2 and the two annihilation photons are followed right after the parent. */
template <class R> struct History { uint64_t h; uint32_t ns; };

/* per-volume tally (S:8(a) A9): edep[vol] += deposit.  Optionally also the number of deposits and the sum of their squares
 * per volume, from which a test estimates the Monte Carlo error of a group of volumes (S:C10 "3 sigma_MC"). */
struct Tally {
    double* edep; double* edep_sq; uint32_t* n_dep;
    void add(int vol, double dep) const {
        edep[vol] += dep;
        if (edep_sq) edep_sq[vol] += dep * dep;
        if (n_dep) n_dep[vol] += 1;
    }
};

template <class R>
void pair_directions(uint64_t seed, uint64_t id, R w1[3], R w2[3], Stream& s1) {
    /* isotropic u from draws 0, 1 of stream (seed, id, tag 1): cos(theta) = 1 - 2 u0, phi = 2 pi u1; second photon exactly -u */
    const R twopi = (R)6.283185307179586;
    s1 = Stream{seed, id, 0, 1};
    R u0 = s1.u<R>(), u1 = s1.u<R>();
    R ct = (R)1 - (R)2 * u0;
    R st = r_sqrt(r_max(((R)1 - ct) * ((R)1 + ct), (R)0));
    R phi = twopi * u1;
    w1[0] = st * r_cos(phi); w1[1] = st * r_sin(phi); w1[2] = ct;
    for (int i = 0; i < 3; ++i) w2[i] = -w1[i];
}

template <class R>
History<R> track(const Geo& g, const Navigator<R>& nav, uint64_t seed, uint64_t id, Stream& rng, R x[3], R w[3], R& E,
                 const Tally& edep, oracle_stats_t& st) {
    const R twopi = (R)6.283185307179586;
    uint64_t h = kFnvOffset; uint32_t ns = 0;
    int vol = nav.locate(x, w);
    bool alive = true;
    if (vol < 0) { st.n_escaped++; st.e_escaped += (double)E; alive = false; }
    R Y = 0; EnergyFactors<R> ef{}; R u_pe = 0;
    const bool pe_tab = g.pe_per_decade > 0;
    if (alive) { Y = -r_log(rng.u<R>()); ef = energy_factors(E); if (pe_tab) u_pe = pe_table_coordinate<R>(E, g.pe_per_decade); }           /* Alg.1 steps 1-2 */
    int zero_steps = 0;
    bool annihilate = false;
    while (alive) {
        R mu4[4]; mu_all<R>(g, g.material[vol], E, ef, u_pe, mu4);             /* PE, Compton, Rayleigh, pair */
        R mu = ((mu4[0] + mu4[1]) + mu4[2]) + mu4[3];
        R s_int = mu > 0 ? Y / mu : r_inf<R>();                                 /* Eq.7 remaining part */
        R step; int next;
        nav.compute_step(vol, x, w, s_int, step, next);                         /* "next intersection" P:L67 */
        ++ns; st.n_steps++;
        int vol_before = vol, ev; R len;
        if (step == r_inf<R>()) {                                               /* S_j >= Y: interact here */
            len = s_int;
            for (int i = 0; i < 3; ++i) x[i] = r_fma(s_int, w[i], x[i]);
            R t = rng.u<R>() * mu;
            /* process choice (D:reading 2): cumulative thresholds; U = 1 falls to the last process with a non-zero coefficient */
            const bool last_is_pair = mu4[3] > 0, last_is_rayleigh = !last_is_pair && mu4[2] > 0;
            if (t < mu4[0]) {                                                   /* photoelectric */
                edep.add(vol, (double)E); st.e_deposited += (double)E; st.n_pe++; ev = EV_PE; alive = false;
            } else if (t < mu4[0] + mu4[1] || (!last_is_pair && !last_is_rayleigh)) {       /* Compton */
                R eps, cost, s2; kn_sample(E, rng, eps, cost, s2);
                R Ep = eps * E;
                R phi = twopi * rng.u<R>();
                rotate_dir(w, cost, r_sqrt(r_max(s2, (R)0)), phi);
                R dep = E - Ep;
                st.n_compton++; ev = EV_COMPTON;
                E = Ep;
                if (Ep < (R)g.e_cut) { dep = dep + Ep; st.n_cut++; ev = EV_CUT; alive = false; }
                edep.add(vol, (double)dep); st.e_deposited += (double)dep;
                if (alive) { ef = energy_factors(E); if (pe_tab) u_pe = pe_table_coordinate<R>(E, g.pe_per_decade); Y = -r_log(rng.u<R>()); }
            } else if (t < (mu4[0] + mu4[1]) + mu4[2] || last_is_rayleigh) {    /* Rayleigh: direction changes, energy does not */
                R cost; rayleigh_sample<R>(rng, cost);
                R sint = r_sqrt(r_max(((R)1 - cost) * ((R)1 + cost), (R)0));
                R phi = twopi * rng.u<R>();
                rotate_dir(w, cost, sint, phi);
                st.n_rayleigh++; ev = EV_RAYLEIGH;
                Y = -r_log(rng.u<R>());
            } else {                                                            /* pair */
                R dep = g.secondaries ? E - (R)(2.0 * kMeC2) : E;               /* local deposit: all of E, or the pair's kinetic energy */
                edep.add(vol, (double)dep); st.e_deposited += (double)dep; st.n_pair++; ev = EV_PAIR; alive = false;
                annihilate = g.secondaries != 0;
            }
        } else {                                                                /* boundary */
            len = step;
            for (int i = 0; i < 3; ++i) x[i] = r_fma(step, w[i], x[i]);
            Y = r_max(Y - step * mu, (R)0);                                     /* S_j update */
            vol = next;
            if (vol < 0) { st.n_escaped++; st.e_escaped += (double)E; ev = EV_ESCAPE; alive = false; }
            else ev = EV_BOUNDARY;
        }
        if (len <= nav.delta) ++zero_steps; else zero_steps = 0;
        if (alive && zero_steps >= g.stuck_limit) { st.n_stuck++; st.e_stuck += (double)E; ev = EV_STUCK; alive = false; }
        fnv_word(h, (uint32_t)vol_before); fnv_word(h, (uint32_t)ev);
    }
    if (annihilate) {
        /* positron at rest at the vertex x: two photons of me c^2, back to back; photon 1 carries on with stream tag 1
         * (after the two direction draws), photon 2 starts stream tag 2.  Their hashes and step counts are added to the
         * parent's (sums, so the order in which an implementation follows them does not matter). */
        R w1[3], w2[3]; Stream s1{seed, id, 0, 1}, s2{seed, id, 0, 2};
        pair_directions<R>(seed, id, w1, w2, s1);
        R xa[3] = {x[0], x[1], x[2]}, xb[3] = {x[0], x[1], x[2]};
        R Ea = (R)kMeC2, Eb = (R)kMeC2;
        History<R> a = track<R>(g, nav, seed, id, s1, xa, w1, Ea, edep, st);
        History<R> b = track<R>(g, nav, seed, id, s2, xb, w2, Eb, edep, st);
        h += a.h + b.h; ns += a.ns + b.ns;
    }
    return History<R>{h, ns};
}

template <class R>
void transport_photon(const Geo& g, const Navigator<R>& nav, const SourceR<R>& src, uint64_t seed, uint64_t id,
                      const Tally& edep, oracle_stats_t& st, uint64_t* hash_out, uint32_t* nsteps_out, double* efinal_out) {
    Stream rng{seed, id, 0, 0};
    R x[3], w[3], E;
    sample_source(src, rng, x, w, E);
    st.n_photons++; st.e_source += (double)E;
    History<R> hs = track<R>(g, nav, seed, id, rng, x, w, E, edep, st);
    if (hash_out) *hash_out = hs.h;
    if (nsteps_out) *nsteps_out = hs.ns;
    if (efinal_out) *efinal_out = (double)E;
}

/* ---- the paper's own benchmark: Algorithm 1 with attenuation only (Eq. 9) ----------
 * Input per particle: x0, w, Y (the paper generates these on the host, Algorithm 2 steps 2-3).
 * mu_j = rho(volume) * mu_mass [cm^2/g] / 10 in 1/mm, evaluated in fp64 per material and rounded once to Real.
 * Walk the boundaries ("Compute the next intersection ... using Geant4") carrying the remaining optical
 * depth Yrem = Y - S_{j-1}: the free path ends inside the current volume when Yrem / mu_j is not beyond the next
 * boundary, T = t_{j-1} + (Y - S_{j-1}) / mu_j; leaving the world gives T = +inf ("S_j may be infinite").
 * Tie s_int == boundary -> boundary, Yrem <- max(Yrem - step mu, 0), stuck guard: as S:C9 / D:readings.
 * t accumulates in Real: t <- t + step. */
template <class R>
void free_path(const Geo& g, const Navigator<R>& nav, const std::vector<R>& mu_of_mat, const R x0[3], const R w[3], R Y,
               R& T_out, uint32_t& nsteps_out) {
    R x[3] = {x0[0], x0[1], x0[2]};
    int vol = nav.locate(x, w);
    R t = 0, Yrem = Y; uint32_t ns = 0; int zero_steps = 0;
    T_out = r_inf<R>();
    while (vol >= 0) {
        R mu = mu_of_mat[g.material[vol]];
        R s_int = mu > 0 ? Yrem / mu : r_inf<R>();
        R step; int next;
        nav.compute_step(vol, x, w, s_int, step, next);
        ++ns;
        if (step == r_inf<R>()) { T_out = t + s_int; break; }          /* S_j >= Y inside this volume */
        for (int i = 0; i < 3; ++i) x[i] = r_fma(step, w[i], x[i]);
        t = t + step;
        Yrem = r_max(Yrem - step * mu, (R)0);
        vol = next;
        if (step <= nav.delta) ++zero_steps; else zero_steps = 0;
        if (vol >= 0 && zero_steps >= g.stuck_limit) break;           /* stuck: T stays +inf */
    }
    nsteps_out = ns;
}
template <class R> int run_free_path(const Geo& g, const void* pos, const void* dir, const void* Y, int64_t n, double mu_mass,
                                     void* T_out, uint32_t* nsteps_out, bool grid) {
    Navigator<R> nav(g, grid);
    std::vector<R> mu(g.mats.size());
    for (size_t m = 0; m < g.mats.size(); ++m) mu[m] = (R)(g.mats[m].rho * mu_mass / 10.0);
    const R* P = (const R*)pos; const R* D = (const R*)dir; const R* Yv = (const R*)Y; R* T = (R*)T_out;
    for (int64_t i = 0; i < n; ++i) {
        uint32_t ns;
        free_path(g, nav, mu, P + 3 * i, D + 3 * i, Yv[i], T[i], ns);
        if (nsteps_out) nsteps_out[i] = ns;
    }
    return ORACLE_OK;
}

/* ---- geometry construction -------------------------------------------------------------- */
void mat3_mul(const double* A, const double* B, double* C) {
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j)
        C[3 * i + j] = (A[3 * i] * B[j] + A[3 * i + 1] * B[3 + j]) + A[3 * i + 2] * B[6 + j];
}

/* tight AABB of a solid in its own frame */
void solid_aabb(const SolidD& s, double lo[3], double hi[3]) {
    if (s.type == ORACLE_BOX) { lo[0] = -s.a; hi[0] = s.a; lo[1] = -s.b; hi[1] = s.b; lo[2] = -s.c; hi[2] = s.c; return; }
    if (s.type == ORACLE_ORB) { for (int k = 0; k < 3; ++k) { lo[k] = -s.a; hi[k] = s.a; } return; }
    if (s.type == ORACLE_CONE) { lo[0] = lo[1] = -s.sphi; hi[0] = hi[1] = s.sphi; lo[2] = -s.c; hi[2] = s.c; return; }
    lo[2] = -s.c; hi[2] = s.c;
    if (!s.sector) { lo[0] = lo[1] = -s.b; hi[0] = hi[1] = s.b; return; }
    double xs[16], ys[16]; int n = 0;
    double ang[2] = {s.sphi, s.sphi + s.dphi}, rr[2] = {s.a, s.b};
    for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) { xs[n] = rr[j] * std::cos(ang[i]); ys[n] = rr[j] * std::sin(ang[i]); ++n; }
    for (int k = -8; k <= 8; ++k) {
        double th = k * (kPi / 2);
        if (th >= ang[0] && th <= ang[1]) { xs[n] = s.b * std::cos(th); ys[n] = s.b * std::sin(th); ++n; }
    }
    lo[0] = hi[0] = xs[0]; lo[1] = hi[1] = ys[0];
    for (int i = 1; i < n; ++i) { lo[0] = std::min(lo[0], xs[i]); hi[0] = std::max(hi[0], xs[i]); lo[1] = std::min(lo[1], ys[i]); hi[1] = std::max(hi[1], ys[i]); }
}

void build_grid(Geo& g, int mother) {
    const std::vector<int>& ds = g.daughters[mother];
    Grid G;
    double mlo[3], mhi[3];
    const SolidD& ms = g.solids[g.solid[mother]];
    if (ms.type == ORACLE_BOX) { mlo[0] = -ms.a; mhi[0] = ms.a; mlo[1] = -ms.b; mhi[1] = ms.b; mlo[2] = -ms.c; mhi[2] = ms.c; }
    else if (ms.type == ORACLE_ORB) { for (int k = 0; k < 3; ++k) { mlo[k] = -ms.a; mhi[k] = ms.a; } }
    else if (ms.type == ORACLE_CONE) { mlo[0] = mlo[1] = -ms.sphi; mhi[0] = mhi[1] = ms.sphi; mlo[2] = -ms.c; mhi[2] = ms.c; }
    else { mlo[0] = mlo[1] = -ms.b; mhi[0] = mhi[1] = ms.b; mlo[2] = -ms.c; mhi[2] = ms.c; }
    int nper = (int)std::ceil(std::cbrt((double)ds.size()));
    nper = std::max(1, std::min(nper, 64));
    double pad = 2.0 * std::max(g.tol32, g.tol64);
    for (int k = 0; k < 3; ++k) { G.n[k] = nper; G.gmin[k] = mlo[k]; G.inv_w[k] = nper / (mhi[k] - mlo[k]); }
    size_t ncell = (size_t)nper * nper * nper;
    std::vector<std::vector<int>> lists(ncell);
    for (int d : ds) {
        double lo[3], hi[3]; solid_aabb(g.solids[g.solid[d]], lo, hi);
        const double* Rm = &g.Rin[9 * d]; const double* T = &g.Tin[3 * d];
        double alo[3] = {1e300, 1e300, 1e300}, ahi[3] = {-1e300, -1e300, -1e300};
        for (int c = 0; c < 8; ++c) {
            double q[3] = {(c & 1) ? hi[0] : lo[0], (c & 2) ? hi[1] : lo[1], (c & 4) ? hi[2] : lo[2]};
            for (int k = 0; k < 3; ++k) {
                double y = Rm[3 * k] * q[0] + Rm[3 * k + 1] * q[1] + Rm[3 * k + 2] * q[2] + T[k];
                alo[k] = std::min(alo[k], y); ahi[k] = std::max(ahi[k], y);
            }
        }
        int c0[3], c1[3];
        for (int k = 0; k < 3; ++k) {
            c0[k] = (int)std::min(std::max(std::floor((alo[k] - pad - G.gmin[k]) * G.inv_w[k]), 0.0), (double)(nper - 1));
            c1[k] = (int)std::min(std::max(std::floor((ahi[k] + pad - G.gmin[k]) * G.inv_w[k]), 0.0), (double)(nper - 1));
        }
        for (int iz = c0[2]; iz <= c1[2]; ++iz) for (int iy = c0[1]; iy <= c1[1]; ++iy) for (int ix = c0[0]; ix <= c1[0]; ++ix)
            lists[ix + (size_t)nper * (iy + (size_t)nper * iz)].push_back(d);   /* ds ascending -> lists ascending */
    }
    G.start.resize(ncell + 1); G.start[0] = 0;
    for (size_t c = 0; c < ncell; ++c) G.start[c + 1] = G.start[c] + (int)lists[c].size();
    G.cand.reserve(G.start[ncell]);
    for (size_t c = 0; c < ncell; ++c) G.cand.insert(G.cand.end(), lists[c].begin(), lists[c].end());
    g.grid_of[mother] = (int)g.grids.size();
    g.grids.push_back(std::move(G));
}

template <class R> SolidR<R> round_solid(const SolidD& s) {
    SolidR<R> o; o.type = s.type; o.a = (R)s.a; o.b = (R)s.b; o.c = (R)s.c; o.sector = s.sector;
    o.cS = (R)s.cS; o.sS = (R)s.sS; o.cE = (R)s.cE; o.sE = (R)s.sE; return o;
}
template <class R> MaterialR<R> round_material(const MaterialD& m, double s0) {
    double n = m.rho * kNA / m.A;                 /* atoms / cm^3;  mu[1/mm] = n sigma / 10 (S:C6) */
    MaterialR<R> o;
    o.aPE = (R)(n * (s0 * kBarn * std::pow(m.Z / 82.0, 5.0)) / 10.0);
    o.aC = (R)(n * (m.Z * (2.0 * kPi * kRe * kRe)) / 10.0);
    o.aP = (R)(n * (kAlpha * kRe * kRe * m.Z * m.Z) / 10.0);
    o.capZ = (R)pair_cap(m.Z);
    return o;
}

template <class R> int run_locate(const Geo& g, const void* pos, const void* dir, int64_t n, int32_t* out, bool grid) {
    Navigator<R> nav(g, grid);
    const R* P = (const R*)pos; const R* D = (const R*)dir;
    for (int64_t i = 0; i < n; ++i) out[i] = nav.locate(P + 3 * i, D ? D + 3 * i : nullptr);
    return ORACLE_OK;
}
template <class R> int run_step(const Geo& g, const void* pos, const void* dir, const int32_t* vol, const void* maxs,
                                int64_t n, void* step_out, int32_t* next_out, bool grid) {
    Navigator<R> nav(g, grid);
    const R* P = (const R*)pos; const R* D = (const R*)dir; const R* Mx = (const R*)maxs; R* S = (R*)step_out;
    for (int64_t i = 0; i < n; ++i) {
        R st; int nx;
        if (vol[i] >= (int32_t)g.parent.size()) return ORACLE_INVALID_ARGUMENT;
        nav.compute_step(vol[i], P + 3 * i, D + 3 * i, Mx ? Mx[i] : r_inf<R>(), st, nx);
        S[i] = st; next_out[i] = nx;
    }
    return ORACLE_OK;
}
template <class R> int run_step_normal(const Geo& g, const void* pos, const void* dir, const int32_t* vol, const void* maxs,
                                       int64_t n, void* step_out, int32_t* next_out, void* normal_out, bool grid) {
    Navigator<R> nav(g, grid);
    const R* P = (const R*)pos; const R* D = (const R*)dir; const R* Mx = (const R*)maxs; R* S = (R*)step_out; R* N = (R*)normal_out;
    for (int64_t i = 0; i < n; ++i) {
        R st; int nx;
        if (vol[i] >= (int32_t)g.parent.size()) return ORACLE_INVALID_ARGUMENT;
        nav.compute_step_normal(vol[i], P + 3 * i, D + 3 * i, Mx ? Mx[i] : r_inf<R>(), st, nx, N + 3 * i);
        S[i] = st; next_out[i] = nx;
    }
    return ORACLE_OK;
}
template <class R> int run_transport(const Geo& g, const oracle_source_t* src, uint64_t seed, int64_t first, int64_t n,
                                     const Tally& edep, oracle_stats_t* st, uint64_t* hash, uint32_t* ns, double* ef, bool grid) {
    SourceR<R> s;
    if (!make_source(*src, s)) return ORACLE_INVALID_ARGUMENT;
    Navigator<R> nav(g, grid);
    oracle_stats_t local; std::memset(&local, 0, sizeof local);
    for (int64_t i = 0; i < n; ++i)
        transport_photon<R>(g, nav, s, seed, (uint64_t)(first + i), edep, local, hash ? hash + i : nullptr,
                            ns ? ns + i : nullptr, ef ? ef + i : nullptr);
    if (st) *st = local;
    return ORACLE_OK;
}

template <class R> int run_safety(const Geo& g, const void* pos, const int32_t* vol_in, int64_t n, void* out) {
    Navigator<R> nav(g, false);
    const R* P = (const R*)pos; R* O = (R*)out;
    for (int64_t i = 0; i < n; ++i) {
        if (vol_in[i] < -1 || vol_in[i] >= (int32_t)g.parent.size()) return ORACLE_INVALID_ARGUMENT;
        O[i] = nav.safety(vol_in[i], P + 3 * i);
    }
    return ORACLE_OK;
}

template <class R> int run_solid_eval(const SolidD& sd, double tol, int what, const void* pos, const void* dir, int64_t n, void* out) {
    SolidR<R> s = round_solid<R>(sd);
    R delta = (R)tol / 2;
    const R* P = (const R*)pos; const R* D = (const R*)dir; R* O = (R*)out;
    for (int64_t i = 0; i < n; ++i) {
        if (what == 0) O[i] = (R)solid_inside(s, P + 3 * i, delta);
        else if (what == 1) O[i] = solid_dist_in(s, P + 3 * i, D + 3 * i, delta);
        else if (what == 3) solid_normal(s, P + 3 * i, O + 3 * i);            /* out: n x 3 */
        else if (what == 4) O[i] = solid_safety_in(s, P + 3 * i);
        else if (what == 5) O[i] = solid_safety_out(s, P + 3 * i);
        else O[i] = solid_dist_out(s, P + 3 * i, D + 3 * i, delta);
    }
    return ORACLE_OK;
}

int make_solid(int type, const double* p, SolidD& s) {
    s.type = type; s.sector = false; s.cS = s.sS = s.cE = s.sE = 0; s.sphi = s.dphi = 0;
    if (type == ORACLE_BOX) {
        s.a = p[0]; s.b = p[1]; s.c = p[2];
        if (!(s.a > 0 && s.b > 0 && s.c > 0)) return ORACLE_INVALID_ARGUMENT;
        return ORACLE_OK;
    }
    if (type == ORACLE_ORB) {
        s.a = p[0]; s.b = s.c = 0;
        if (!(s.a > 0)) return ORACLE_INVALID_ARGUMENT;
        return ORACLE_OK;
    }
    if (type == ORACLE_CONE) {                    /* params r1, r2, hz -> a = r0, b = slope, c = hz, cS = 1/sqrt(1 + slope^2) */
        double r1 = p[0], r2 = p[1], hz = p[2];
        if (!(r1 >= 0 && r2 >= 0 && r1 + r2 > 0 && hz > 0)) return ORACLE_INVALID_ARGUMENT;
        s.a = (r1 + r2) / 2; s.b = (r2 - r1) / (2 * hz); s.c = hz;
        s.cS = 1 / std::sqrt(1 + s.b * s.b);
        s.sphi = r1 > r2 ? r1 : r2;               /* largest radius, for bounding boxes only */
        return ORACLE_OK;
    }
    if (type != ORACLE_TUBE) return ORACLE_UNSUPPORTED_SOLID;
    s.a = p[0]; s.b = p[1]; s.c = p[2]; s.sphi = p[3]; s.dphi = p[4];
    if (!(s.a >= 0 && s.b > s.a && s.c > 0)) return ORACLE_INVALID_ARGUMENT;
    if (s.dphi >= 2 * kPi) return ORACLE_OK;
    if (!(s.dphi > 0) || s.dphi > kPi) return ORACLE_UNSUPPORTED_SOLID;      /* convex sectors only (S:C2) */
    s.sector = true;
    s.cS = std::cos(s.sphi); s.sS = std::sin(s.sphi);
    s.cE = std::cos(s.sphi + s.dphi); s.sE = std::sin(s.sphi + s.dphi);
    return ORACLE_OK;
}

}  // namespace

/* ======================================================================================== */
extern "C" {

int oracle_geometry_create(const double* materials, int32_t n_mats, const int32_t* solid_type, const double* solid_params,
                           int32_t n_solids, const int32_t* placements, int32_t n_places, const double* transforms,
                           int32_t n_transforms, const oracle_opts_t* opts, void** out) {
    if (!materials || !solid_type || !solid_params || !placements || !transforms || !out) return ORACLE_INVALID_ARGUMENT;
    if (n_mats <= 0 || n_solids <= 0 || n_places <= 0 || n_transforms <= 0) return ORACLE_INVALID_ARGUMENT;
    Geo* g = new Geo();
    for (int i = 0; i < n_mats; ++i) {
        MaterialD m{materials[3 * i], materials[3 * i + 1], materials[3 * i + 2]};
        if (!(m.Z > 0 && m.A > 0 && m.rho >= 0)) { delete g; return ORACLE_INVALID_ARGUMENT; }
        g->mats.push_back(m);
    }
    for (int i = 0; i < n_solids; ++i) {
        SolidD s; int rc = make_solid(solid_type[i], solid_params + 5 * i, s);
        if (rc != ORACLE_OK) { delete g; return rc; }
        g->solids.push_back(s);
    }
    g->parent.resize(n_places); g->solid.resize(n_places); g->material.resize(n_places); g->xform_in.resize(n_places);
    g->daughters.resize(n_places); g->Rin.resize(9 * (size_t)n_places); g->Tin.resize(3 * (size_t)n_places);
    g->x64.resize(n_places); g->x32.resize(n_places);
    std::vector<double> Rg(9 * (size_t)n_places), Tg(3 * (size_t)n_places);
    for (int i = 0; i < n_places; ++i) {
        int p = placements[4 * i], s = placements[4 * i + 1], m = placements[4 * i + 2], t = placements[4 * i + 3];
        if (s < 0 || s >= n_solids || m < 0 || m >= n_mats || t < 0 || t >= n_transforms) { delete g; return ORACLE_INVALID_ARGUMENT; }
        if ((i == 0 && p != -1) || (i > 0 && (p < 0 || p >= i))) { delete g; return ORACLE_BAD_TREE; }
        g->parent[i] = p; g->solid[i] = s; g->material[i] = m; g->xform_in[i] = t;
        const double* Rl = transforms + 12 * (size_t)t; const double* Tl = Rl + 9;
        for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) {          /* orthonormality */
            double dot = Rl[3 * a] * Rl[3 * b] + Rl[3 * a + 1] * Rl[3 * b + 1] + Rl[3 * a + 2] * Rl[3 * b + 2];
            if (std::fabs(dot - (a == b ? 1.0 : 0.0)) > 1e-9) { delete g; return ORACLE_BAD_TREE; }
        }
        std::memcpy(&g->Rin[9 * (size_t)i], Rl, 9 * sizeof(double)); std::memcpy(&g->Tin[3 * (size_t)i], Tl, 3 * sizeof(double));
        /* S:C0 composition root-down in fp64: Rg = Rg_parent R, Tg = Rg_parent T + Tg_parent */
        double* R = &Rg[9 * (size_t)i]; double* T = &Tg[3 * (size_t)i];
        if (p < 0) { std::memcpy(R, Rl, 9 * sizeof(double)); std::memcpy(T, Tl, 3 * sizeof(double)); }
        else {
            const double* Rp = &Rg[9 * (size_t)p]; const double* Tp = &Tg[3 * (size_t)p];
            mat3_mul(Rp, Rl, R);
            for (int a = 0; a < 3; ++a) T[a] = ((Rp[3 * a] * Tl[0] + Rp[3 * a + 1] * Tl[1]) + Rp[3 * a + 2] * Tl[2]) + Tp[a];
            g->daughters[p].push_back(i);
        }
        for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) {          /* M = Rg^T */
            g->x64[i].M[3 * a + b] = R[3 * b + a]; g->x32[i].M[3 * a + b] = (float)R[3 * b + a];
        }
        for (int a = 0; a < 3; ++a) { g->x64[i].T[a] = T[a]; g->x32[i].T[a] = (float)T[a]; }
    }
    const SolidD& ws = g->solids[g->solid[0]];
    double ext = ws.type == ORACLE_BOX ? std::max(ws.a, std::max(ws.b, ws.c)) : (ws.type == ORACLE_ORB ? ws.a : (ws.type == ORACLE_CONE ? std::max(ws.sphi, ws.c) : std::max(ws.b, ws.c)));
    g->tol64 = (opts && opts->tol64 > 0) ? opts->tol64 : 1e-9;
    g->tol32 = (opts && opts->tol32 > 0) ? opts->tol32 : (double)(float)(ext * 0x1p-18);
    g->sigma_pe0 = (opts && opts->sigma_pe0 > 0) ? opts->sigma_pe0 : 1750.0;
    g->e_cut = (opts && opts->e_cut > 0) ? opts->e_cut : 0.010;
    g->grid_min = (opts && opts->grid_min_daughters > 0) ? opts->grid_min_daughters : 8;
    g->stuck_limit = (opts && opts->stuck_limit > 0) ? opts->stuck_limit : 8;
    g->secondaries = (opts && opts->secondaries > 0) ? 1 : 0;
    g->rayleigh = (opts && opts->rayleigh > 0) ? 1 : 0;
    g->sigma_r0 = (opts && opts->sigma_r0 > 0) ? opts->sigma_r0 : 7.886e-3;
    g->pe_per_decade = (opts && opts->pe_table_per_decade > 0) ? opts->pe_table_per_decade : 0;
    g->pe_k_edge = (opts && opts->pe_k_edge > 0) ? 1 : 0;
    if (g->pe_per_decade > 4096) { delete g; return ORACLE_INVALID_ARGUMENT; }
    for (const MaterialD& m : g->mats) {
        double n = m.rho * kNA / m.A;
        g->aR.push_back(n * (g->sigma_r0 * kBarn * (m.Z / 13.0) * (m.Z / 13.0)) / 10.0);
        std::vector<double> T;
        if (g->pe_per_decade > 0) {
            int np = (int)(kPeDecades * g->pe_per_decade) + 1;
            for (int k = 0; k < np; ++k) {
                double Ek = kPeEmin * std::pow(10.0, (double)k / g->pe_per_decade);
                T.push_back(n * pe_sigma_tab(Ek, m.Z, g->sigma_pe0, g->pe_k_edge) / 10.0);
            }
        }
        g->pe_tab.push_back(T);
    }
    for (const SolidD& s : g->solids) { g->s64.push_back(round_solid<double>(s)); g->s32.push_back(round_solid<float>(s)); }
    for (const MaterialD& m : g->mats) { g->m64.push_back(round_material<double>(m, g->sigma_pe0)); g->m32.push_back(round_material<float>(m, g->sigma_pe0)); }
    /* operation counter: the fp64 tables again, element by element, in the counting type */
    g->xc.resize(n_places);
    for (int i = 0; i < n_places; ++i) {
        for (int k = 0; k < 9; ++k) g->xc[i].M[k] = Counted(g->x64[i].M[k]);
        for (int k = 0; k < 3; ++k) g->xc[i].T[k] = Counted(g->x64[i].T[k]);
    }
    for (const SolidR<double>& s : g->s64) {
        SolidR<Counted> c; c.type = s.type; c.a = s.a; c.b = s.b; c.c = s.c; c.sector = s.sector; c.cS = s.cS; c.sS = s.sS; c.cE = s.cE; c.sE = s.sE;
        g->sc.push_back(c);
    }
    for (const MaterialR<double>& m : g->m64) { MaterialR<Counted> c; c.aPE = m.aPE; c.aC = m.aC; c.aP = m.aP; c.capZ = m.capZ; g->mc.push_back(c); }
    g->grid_of.assign(n_places, -1);
    for (int i = 0; i < n_places; ++i) if ((int)g->daughters[i].size() >= g->grid_min) build_grid(*g, i);
    *out = g;
    return ORACLE_OK;
}

int oracle_geometry_destroy(void* geo) { delete (Geo*)geo; return ORACLE_OK; }
double oracle_geometry_tolerance(const void* geo, int precision) {
    const Geo* g = (const Geo*)geo; return precision == 32 ? g->tol32 : g->tol64;
}

int oracle_nav_locate(const void* geo, int precision, const void* pos, const void* dir, int64_t n, int32_t* vol_out, int use_grid) {
    if (!geo || (n > 0 && (!pos || !vol_out)) || n < 0) return ORACLE_INVALID_ARGUMENT;
    const Geo& g = *(const Geo*)geo;
    if (precision == 64) return run_locate<double>(g, pos, dir, n, vol_out, use_grid != 0);
    if (precision == 32) return run_locate<float>(g, pos, dir, n, vol_out, use_grid != 0);
    return ORACLE_INVALID_ARGUMENT;
}

/* Pin for locate (S:C3 "plain definition"): every node, hierarchical per-level transforms in fp64,
 * surface counts as inside; answer = deepest node containing the point with all ancestors containing it. */
int oracle_nav_locate_bruteforce(const void* geo, const double* pos, int64_t n, int32_t* vol_out) {
    if (!geo || !pos || !vol_out) return ORACLE_INVALID_ARGUMENT;
    const Geo& g = *(const Geo*)geo;
    size_t V = g.parent.size();
    std::vector<double> pl(3 * V); std::vector<char> in(V); std::vector<int> depth(V);
    double delta = g.tol64 / 2;
    for (int64_t q = 0; q < n; ++q) {
        int best = -1, bestd = -1;
        for (size_t i = 0; i < V; ++i) {
            const double* Rl = &g.Rin[9 * i]; const double* Tl = &g.Tin[3 * i];
            double x[3];
            int p = g.parent[i];
            if (p < 0) { x[0] = pos[3 * q]; x[1] = pos[3 * q + 1]; x[2] = pos[3 * q + 2]; depth[i] = 0; }
            else { x[0] = pl[3 * p]; x[1] = pl[3 * p + 1]; x[2] = pl[3 * p + 2]; depth[i] = depth[p] + 1; }
            double d[3] = {x[0] - Tl[0], x[1] - Tl[1], x[2] - Tl[2]};
            for (int k = 0; k < 3; ++k) pl[3 * i + k] = Rl[k] * d[0] + Rl[3 + k] * d[1] + Rl[6 + k] * d[2];   /* R^T d */
            bool anc = p < 0 ? true : (bool)in[p];
            in[i] = anc && solid_inside(g.s64[g.solid[i]], &pl[3 * i], delta) != OUT;
            if (in[i] && depth[i] > bestd) { best = (int)i; bestd = depth[i]; }
        }
        vol_out[q] = best;
    }
    return ORACLE_OK;
}

int oracle_nav_compute_step(const void* geo, int precision, const void* pos, const void* dir, const int32_t* vol_in,
                            const void* max_step, int64_t n, void* step_out, int32_t* next_vol_out, int use_grid) {
    if (!geo || n < 0 || (n > 0 && (!pos || !dir || !vol_in || !step_out || !next_vol_out))) return ORACLE_INVALID_ARGUMENT;
    const Geo& g = *(const Geo*)geo;
    if (precision == 64) return run_step<double>(g, pos, dir, vol_in, max_step, n, step_out, next_vol_out, use_grid != 0);
    if (precision == 32) return run_step<float>(g, pos, dir, vol_in, max_step, n, step_out, next_vol_out, use_grid != 0);
    return ORACLE_INVALID_ARGUMENT;
}

int oracle_nav_compute_safety(const void* geo, int precision, const void* pos, const int32_t* vol_in, int64_t n, void* safety_out) {
    if (!geo || n < 0 || (n > 0 && (!pos || !vol_in || !safety_out))) return ORACLE_INVALID_ARGUMENT;
    const Geo& g = *(const Geo*)geo;
    if (precision == 64) return run_safety<double>(g, pos, vol_in, n, safety_out);
    if (precision == 32) return run_safety<float>(g, pos, vol_in, n, safety_out);
    return ORACLE_INVALID_ARGUMENT;
}

int oracle_nav_compute_step_normal(const void* geo, int precision, const void* pos, const void* dir, const int32_t* vol_in,
                                   const void* max_step, int64_t n, void* step_out, int32_t* next_vol_out, void* normal_out, int use_grid) {
    if (!geo || n < 0 || (n > 0 && (!pos || !dir || !vol_in || !step_out || !next_vol_out || !normal_out))) return ORACLE_INVALID_ARGUMENT;
    const Geo& g = *(const Geo*)geo;
    if (precision == 64) return run_step_normal<double>(g, pos, dir, vol_in, max_step, n, step_out, next_vol_out, normal_out, use_grid != 0);
    if (precision == 32) return run_step_normal<float>(g, pos, dir, vol_in, max_step, n, step_out, next_vol_out, normal_out, use_grid != 0);
    return ORACLE_INVALID_ARGUMENT;
}

int oracle_transport_run(const void* geo, int precision, const oracle_source_t* src, uint64_t seed, int64_t first_id,
                         int64_t n_photons, double* edep_out, oracle_stats_t* stats_out, uint64_t* hash_out,
                         uint32_t* nsteps_out, double* efinal_out, int use_grid) {
    return oracle_transport_run_tally(geo, precision, src, seed, first_id, n_photons, edep_out, nullptr, nullptr, stats_out, hash_out, nsteps_out,
                                      efinal_out, use_grid);
}

int oracle_transport_run_tally(const void* geo, int precision, const oracle_source_t* src, uint64_t seed, int64_t first_id,
                               int64_t n_photons, double* edep_out, double* edep_sq_out, uint32_t* n_dep_out, oracle_stats_t* stats_out,
                               uint64_t* hash_out, uint32_t* nsteps_out, double* efinal_out, int use_grid) {
    if (!geo || !src || !edep_out || n_photons < 0 || first_id < 0) return ORACLE_INVALID_ARGUMENT;
    const Geo& g = *(const Geo*)geo;
    const Tally tally{edep_out, edep_sq_out, n_dep_out};
    if (precision == 64) return run_transport<double>(g, src, seed, first_id, n_photons, tally, stats_out, hash_out, nsteps_out, efinal_out, use_grid != 0);
    if (precision == 32) return run_transport<float>(g, src, seed, first_id, n_photons, tally, stats_out, hash_out, nsteps_out, efinal_out, use_grid != 0);
    return ORACLE_INVALID_ARGUMENT;
}

/* ---- operation counts (S:8(d)): the same templates run in the counting type ------------------------------- */
static void ops_out(uint64_t c[8]) {
    c[0] = g_ops.add; c[1] = g_ops.mul; c[2] = g_ops.div; c[3] = g_ops.sqrt; c[4] = g_ops.cmp; c[5] = g_ops.fma; c[6] = g_ops.trans;
    c[7] = g_ops.add + g_ops.mul + g_ops.div + g_ops.sqrt + g_ops.cmp + 2 * g_ops.fma + g_ops.trans;      /* flops: fma = 2, the rest 1 */
}
int oracle_transport_count_ops(const void* geo, const oracle_source_t* src, uint64_t seed, int64_t first_id, int64_t n_photons,
                               uint64_t counts_out[8], oracle_stats_t* stats_out) {
    if (!geo || !src || !counts_out || n_photons < 0 || first_id < 0) return ORACLE_INVALID_ARGUMENT;
    const Geo& g = *(const Geo*)geo;
    std::vector<double> edep(g.parent.size(), 0.0);
    const Tally tally{edep.data(), nullptr, nullptr};
    g_ops = OpCounts{0, 0, 0, 0, 0, 0, 0};
    int rc = run_transport<Counted>(g, src, seed, first_id, n_photons, tally, stats_out, nullptr, nullptr, nullptr, true);
    ops_out(counts_out);
    return rc;
}
int oracle_nav_count_ops(const void* geo, const double* pos, const double* dir, int64_t n, uint64_t counts_out[8]) {
    if (!geo || !counts_out || n < 0 || (n > 0 && (!pos || !dir))) return ORACLE_INVALID_ARGUMENT;
    const Geo& g = *(const Geo*)geo;
    Navigator<Counted> nav(g, true);
    g_ops = OpCounts{0, 0, 0, 0, 0, 0, 0};
    for (int64_t i = 0; i < n; ++i) {                       /* one config-5 query: locate, then ComputeStep */
        Counted x[3] = {pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]}, w[3] = {dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]};
        int vol = nav.locate(x, w);
        Counted step; int next;
        nav.compute_step(vol, x, w, r_inf<Counted>(), step, next);
    }
    ops_out(counts_out);
    return ORACLE_OK;
}

/* ---- test hooks for the history hash and the set-up arithmetic ------------------------------------------------ */
uint64_t oracle_fnv1a_bytes(const uint8_t* bytes, int64_t n) {
    uint64_t h = kFnvOffset;
    for (int64_t i = 0; i < n; ++i) fnv_byte(h, bytes[i]);
    return h;
}
uint64_t oracle_history_hash(const uint32_t* words, int64_t n_words) {
    uint64_t h = kFnvOffset;
    for (int64_t i = 0; i < n_words; ++i) fnv_word(h, words[i]);
    return h;
}
int oracle_source_frame(const oracle_source_t* src, int precision, double frame_out[9]) {
    if (!src || !frame_out) return ORACLE_INVALID_ARGUMENT;
    if (precision == 64) { SourceR<double> s; if (!make_source(*src, s)) return ORACLE_INVALID_ARGUMENT; for (int i = 0; i < 3; ++i) { frame_out[i] = s.a[i]; frame_out[3 + i] = s.e1[i]; frame_out[6 + i] = s.e2[i]; } }
    else if (precision == 32) { SourceR<float> s; if (!make_source(*src, s)) return ORACLE_INVALID_ARGUMENT; for (int i = 0; i < 3; ++i) { frame_out[i] = s.a[i]; frame_out[3 + i] = s.e1[i]; frame_out[6 + i] = s.e2[i]; } }
    else return ORACLE_INVALID_ARGUMENT;
    return ORACLE_OK;
}
int oracle_composed_transforms(const void* geo, int precision, double* M_out, double* T_out) {
    if (!geo || !M_out || !T_out) return ORACLE_INVALID_ARGUMENT;
    const Geo& g = *(const Geo*)geo;
    for (size_t i = 0; i < g.parent.size(); ++i) {
        for (int k = 0; k < 9; ++k) M_out[9 * i + k] = precision == 32 ? (double)g.x32[i].M[k] : g.x64[i].M[k];
        for (int k = 0; k < 3; ++k) T_out[3 * i + k] = precision == 32 ? (double)g.x32[i].T[k] : g.x64[i].T[k];
    }
    return ORACLE_OK;
}

int oracle_free_path_run(const void* geo, int precision, const void* pos, const void* dir, const void* Y, int64_t n,
                         double mu_mass_cm2_g, void* T_out, uint32_t* nsteps_out, int use_grid) {
    if (!geo || n < 0 || !(mu_mass_cm2_g >= 0) || (n > 0 && (!pos || !dir || !Y || !T_out))) return ORACLE_INVALID_ARGUMENT;
    const Geo& g = *(const Geo*)geo;
    if (precision == 64) return run_free_path<double>(g, pos, dir, Y, n, mu_mass_cm2_g, T_out, nsteps_out, use_grid != 0);
    if (precision == 32) return run_free_path<float>(g, pos, dir, Y, n, mu_mass_cm2_g, T_out, nsteps_out, use_grid != 0);
    return ORACLE_INVALID_ARGUMENT;
}

int oracle_solid_eval(int32_t type, const double* params5, double tol, int precision, int what, const void* pos,
                      const void* dir, int64_t n, void* out) {
    SolidD s; int rc = make_solid(type, params5, s);
    if (rc != ORACLE_OK) return rc;
    if (precision == 64) return run_solid_eval<double>(s, tol, what, pos, dir, n, out);
    if (precision == 32) return run_solid_eval<float>(s, tol, what, pos, dir, n, out);
    return ORACLE_INVALID_ARGUMENT;
}

double oracle_sigma_kn(double k) { return sigma_kn(k); }
double oracle_sigma_pair(double k, double Z) { return sigma_pair(k, Z); }
double oracle_sigma_pe(double E, double Z, double s0) { return sigma_pe(E, Z, s0); }

int oracle_mu(const void* geo, int precision, int32_t material, double E, double* mu3) {
    const Geo& g = *(const Geo*)geo;
    if (material < 0 || material >= (int)g.mats.size()) return ORACLE_INVALID_ARGUMENT;
    if (precision == 64) { double m[4]; mu_all<double>(g, material, E, energy_factors<double>(E), g.pe_per_decade > 0 ? pe_table_coordinate<double>(E, g.pe_per_decade) : 0.0, m); mu3[0] = m[0]; mu3[1] = m[1]; mu3[2] = m[3]; }
    else { float e = (float)E, m[4]; mu_all<float>(g, material, e, energy_factors<float>(e), g.pe_per_decade > 0 ? pe_table_coordinate<float>(e, g.pe_per_decade) : 0.0f, m); mu3[0] = m[0]; mu3[1] = m[1]; mu3[2] = m[3]; }
    return ORACLE_OK;
}
double oracle_mu_rayleigh(const void* geo, int precision, int32_t material, double E) {
    const Geo& g = *(const Geo*)geo;
    if (material < 0 || material >= (int)g.mats.size()) return -1.0;
    return precision == 64 ? mu_rayleigh<double>(g, material, E) : (double)mu_rayleigh<float>(g, material, (float)E);
}
int oracle_rayleigh_sample(int precision, uint64_t seed, int64_t first_id, int64_t n, double* cost_out, int32_t* ntrials_out) {
    for (int64_t i = 0; i < n; ++i) {
        Stream s{seed, (uint64_t)(first_id + i), 0};
        if (precision == 64) { double c; int t = rayleigh_sample<double>(s, c); cost_out[i] = c; if (ntrials_out) ntrials_out[i] = t; }
        else { float c; int t = rayleigh_sample<float>(s, c); cost_out[i] = c; if (ntrials_out) ntrials_out[i] = t; }
    }
    return ORACLE_OK;
}

void oracle_philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t* out4) {
    uint32_t c[4] = {c0, c1, c2, c3}; philox4x32_10(c, k0, k1); std::memcpy(out4, c, sizeof c);
}
double oracle_uniform_from_lane(uint64_t lane, int precision) {
    return precision == 32 ? (double)uniform_from_lane<float>(lane) : uniform_from_lane<double>(lane);
}
double oracle_draw(uint64_t seed, uint64_t id, uint32_t j, int precision) {
    Stream s{seed, id, j};
    return precision == 32 ? (double)s.u<float>() : s.u<double>();
}

int oracle_pair_directions(int precision, uint64_t seed, int64_t first_id, int64_t n, double* w1_out, double* w2_out) {
    for (int64_t i = 0; i < n; ++i) {
        Stream s1{seed, 0, 0, 0};
        if (precision == 64) {
            double a[3], b[3]; pair_directions<double>(seed, (uint64_t)(first_id + i), a, b, s1);
            for (int k = 0; k < 3; ++k) { w1_out[3 * i + k] = a[k]; w2_out[3 * i + k] = b[k]; }
        } else {
            float a[3], b[3]; pair_directions<float>(seed, (uint64_t)(first_id + i), a, b, s1);
            for (int k = 0; k < 3; ++k) { w1_out[3 * i + k] = a[k]; w2_out[3 * i + k] = b[k]; }
        }
    }
    return ORACLE_OK;
}

int oracle_kn_sample(int precision, double E, uint64_t seed, int64_t first_id, int64_t n, double* eps_out, double* cost_out, int32_t* ntrials_out) {
    for (int64_t i = 0; i < n; ++i) {
        Stream s{seed, (uint64_t)(first_id + i), 0};
        if (precision == 64) { double e, c, s2; int t = kn_sample<double>(E, s, e, c, s2); eps_out[i] = e; cost_out[i] = c; if (ntrials_out) ntrials_out[i] = t; }
        else { float e, c, s2; int t = kn_sample<float>((float)E, s, e, c, s2); eps_out[i] = e; cost_out[i] = c; if (ntrials_out) ntrials_out[i] = t; }
    }
    return ORACLE_OK;
}

int oracle_rotate(int precision, const double* w, const double* cost, const double* phi, int64_t n, double* w_out) {
    for (int64_t i = 0; i < n; ++i) {
        if (precision == 64) {
            double v[3] = {w[3 * i], w[3 * i + 1], w[3 * i + 2]};
            double st = std::sqrt(std::max(0.0, 1.0 - cost[i] * cost[i]));
            rotate_dir<double>(v, cost[i], st, phi[i]);
            for (int k = 0; k < 3; ++k) w_out[3 * i + k] = v[k];
        } else {
            float v[3] = {(float)w[3 * i], (float)w[3 * i + 1], (float)w[3 * i + 2]};
            float c = (float)cost[i]; float st = std::sqrt(std::max(0.0f, 1.0f - c * c));
            rotate_dir<float>(v, c, st, (float)phi[i]);
            for (int k = 0; k < 3; ++k) w_out[3 * i + k] = v[k];
        }
    }
    return ORACLE_OK;
}

/* S:C0 the canonical move x' = fma(t, w, x) */
int oracle_move(int precision, const void* pos, const void* dir, const void* step, int64_t n, void* pos_out) {
    if (precision == 64) {
        const double* P = (const double*)pos; const double* D = (const double*)dir; const double* S = (const double*)step; double* O = (double*)pos_out;
        for (int64_t i = 0; i < 3 * n; ++i) O[i] = std::fma(S[i / 3], D[i], P[i]);
    } else if (precision == 32) {
        const float* P = (const float*)pos; const float* D = (const float*)dir; const float* S = (const float*)step; float* O = (float*)pos_out;
        for (int64_t i = 0; i < 3 * n; ++i) O[i] = std::fma(S[i / 3], D[i], P[i]);
    } else return ORACLE_INVALID_ARGUMENT;
    return ORACLE_OK;
}

int oracle_source_sample(int precision, const oracle_source_t* src, uint64_t seed, int64_t first_id, int64_t n,
                         double* pos_out, double* dir_out, double* e_out, int32_t* ndraws_out) {
    if (!src) return ORACLE_INVALID_ARGUMENT;
    if (precision == 64) {
        SourceR<double> s; if (!make_source(*src, s)) return ORACLE_INVALID_ARGUMENT;
        for (int64_t i = 0; i < n; ++i) {
            Stream r{seed, (uint64_t)(first_id + i), 0}; double x[3], w[3], E; sample_source(s, r, x, w, E);
            for (int k = 0; k < 3; ++k) { pos_out[3 * i + k] = x[k]; dir_out[3 * i + k] = w[k]; }
            e_out[i] = E; if (ndraws_out) ndraws_out[i] = (int32_t)r.j;
        }
    } else {
        SourceR<float> s; if (!make_source(*src, s)) return ORACLE_INVALID_ARGUMENT;
        for (int64_t i = 0; i < n; ++i) {
            Stream r{seed, (uint64_t)(first_id + i), 0}; float x[3], w[3], E; sample_source(s, r, x, w, E);
            for (int k = 0; k < 3; ++k) { pos_out[3 * i + k] = x[k]; dir_out[3 * i + k] = w[k]; }
            e_out[i] = E; if (ndraws_out) ndraws_out[i] = (int32_t)r.j;
        }
    }
    return ORACLE_OK;
}

}  // extern "C"
