// physics.cuh -- device physics: Philox4x32-10 streams, attenuation coefficients, Klein-Nishina sampling,
// direction update, photon sources.  SURVEY.md 8(c) C6-C8 (the paper itself only has mu = rho * mu_Al,E,
// PAPER.md Eq. 9, and Exp(1) lifetimes from a uniform in (0,1], Algorithm 1 steps 1-2 L57-59).
#pragma once
#include "nav.cuh"

namespace gn {

// ---- counter-based RNG (C7): key = seed, counter = (photon id lo, hi, block, tag); draw j = 64-bit lane j&1 of block j>>1;
// tag 0 = the primary photon, 1 / 2 = the annihilation photons of its pair event
// One copy of the ten rounds, out of line: draws happen only at interactions (rare next to navigation steps).
// the ten rounds of one block: counter (id0, id1, blk, tag) under key (k0, k1) -> two 64-bit lanes
__device__ __forceinline__ void philox_block(uint32_t k0, uint32_t k1, uint32_t id0, uint32_t id1, uint32_t blk, uint32_t tag, uint64_t& l0, uint64_t& l1) {
    uint32_t c0 = id0, c1 = id1, c2 = blk, c3 = tag, a = k0, b = k1;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        uint32_t n0 = hi1 ^ c1 ^ a, n2 = hi0 ^ c3 ^ b;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        a += 0x9E3779B9u; b += 0xBB67AE85u;
    }
    l0 = (uint64_t)c0 | ((uint64_t)c1 << 32);
    l1 = (uint64_t)c2 | ((uint64_t)c3 << 32);
}
// draw j = lane (j & 1) of block j >> 1; the second lane of a block is kept for the next draw
struct PhiloxStream {
    uint32_t k0, k1, id0, id1, j, tag;
    uint64_t spare; bool have_spare;
    __device__ __forceinline__ void init(uint64_t seed, uint64_t id, uint32_t draws_done, uint32_t stream_tag = 0) {
        k0 = (uint32_t)seed; k1 = (uint32_t)(seed >> 32); id0 = (uint32_t)id; id1 = (uint32_t)(id >> 32); j = draws_done; tag = stream_tag;
        spare = 0; have_spare = false;
    }
    __device__ __forceinline__ uint64_t next() {
        uint64_t out;
        if ((j & 1u) && have_spare) { out = spare; have_spare = false; }
        else {
            uint64_t l0, l1; philox_block(k0, k1, id0, id1, j >> 1, tag, l0, l1);
            if (j & 1u) out = l1; else { out = l0; spare = l1; have_spare = true; }
        }
        ++j;
        return out;
    }
};
// uniforms in (0, 1] as Algorithm 1 step 1 requires
__device__ __forceinline__ float to_uniform(uint64_t lane, float) { return (float)((uint32_t)(lane >> 40) + 1u) * 5.9604644775390625e-08f; }
__device__ __forceinline__ double to_uniform(uint64_t lane, double) { return (double)((lane >> 11) + 1ull) * 1.1102230246251565e-16; }
template <class R> __device__ __forceinline__ R draw(PhiloxStream& s) { return to_uniform(s.next(), R()); }

// ---- transcendental wrappers (physics only; navigation never uses them) ------------------------------
__device__ __forceinline__ float rlog(float a) { return logf(a); }
__device__ __forceinline__ double rlog(double a) { return log(a); }
__device__ __forceinline__ float rexp(float a) { return expf(a); }
__device__ __forceinline__ double rexp(double a) { return exp(a); }
__device__ __forceinline__ void rsincos(float a, float* s, float* c) { *s = sinf(a); *c = cosf(a); }
__device__ __forceinline__ void rsincos(double a, double* s, double* c) { *s = sin(a); *c = cos(a); }

// ---- attenuation (C6) ---------------------------------------------------
// Energy-dependent factors are evaluated in fp64 from E and rounded once to Real; they change only when
// the energy changes, so the photon carries them.  Material factors are Real constants (MatRec).
#define GN_ME_C2 0.51099895
#define GN_PI 3.14159265358979323846
template <class R> struct EnergyFactors { R gPE, gKN, L2k; int above_pair; };

// photoelectric table coordinate (reading 19): u = clamp((ln E - ln 0.01) P / ln 10, 0, 5 P (1 - 2^-24)), fp64, rounded once
template <class R> __device__ __forceinline__ R pe_coordinate(R E, int per_decade) {
    double u = (log((double)E) - log(0.01)) * ((double)per_decade / log(10.0));
    const double top = 5.0 * per_decade * (1.0 - 0x1p-24);
    if (u < 0.0) u = 0.0;
    if (u > top) u = top;
    return (R)u;
}
// gPE is the closed-form factor (0.1 / E)^3.5, or -- pe_per_decade > 0 -- the table coordinate of E
template <class R> __device__ EnergyFactors<R> energy_factors(R E, int pe_per_decade) {
    // Klein-Nishina total cross-section per electron in units of 2 pi r_e^2 (C6):
    //   (1+k)/k^2 [2(1+k)/(1+2k) - ln(1+2k)/k] + ln(1+2k)/(2k) - (1+3k)/(1+2k)^2,  k = E / me c^2
    // DESIGN.md reading 1 writes g_KN as sigma_KN / (2 pi r_e^2): the prefactor is multiplied in and divided out again
    const double k = (double)E / GN_ME_C2;
    const double one_k = 1.0 + k, one_2k = 1.0 + 2.0 * k, lg = log(one_2k);
    const double bracket = 2.0 * one_k / one_2k - lg / k;
    const double first = one_k / (k * k) * bracket, second = lg / (2.0 * k), third = (1.0 + 3.0 * k) / (one_2k * one_2k);
    const double two_pi_re2 = 2.0 * GN_PI * 2.8179403262e-13 * 2.8179403262e-13;
    EnergyFactors<R> f;
    f.gKN = (R)((two_pi_re2 * (first + second - third)) / two_pi_re2);
    if (pe_per_decade > 0) f.gPE = pe_coordinate<R>(E, pe_per_decade);
    else { const double xq = __ddiv_rn(0.1, (double)E); f.gPE = (R)__dmul_rn(__dmul_rn(__dmul_rn(xq, xq), xq), __dsqrt_rn(xq)); }      // (0.1 / E)^3.5 = x x x sqrt(x): IEEE operations only (reading 1)
    f.L2k = (R)log(2.0 * k);
    f.above_pair = k > 2.0;
    return f;
}
// The four partial attenuation coefficients of a photon (energy E, factors gPE / gKN / L2k) in material `mat` (C6; readings
// 1, 18, 19).  With the options off the Rayleigh term is an exact zero and the sum is (mu_PE + mu_C) + mu_pair as before.
template <class R> struct MuParts { R pe, c, r, p, tot; };
template <class R> __device__ __forceinline__ MuParts<R> photon_mu(const GeoView<R>& g, const MatRec<R>& m, int mat, R E, R gPE, R gKN, R L2k, int above) {
    MuParts<R> o;
    if (g.pe_per_decade > 0) {                                   // table: T_i + f (T_{i+1} - T_i), i = floor(u), f = u - i
        const int i = (int)rfloor(gPE);
        const R f = gPE - (R)i;
        const R* T = g.pe_tab + (size_t)mat * g.pe_points + i;
        const R t0 = __ldg(T), t1 = __ldg(T + 1);
        o.pe = t0 + f * (t1 - t0);
    } else o.pe = m.aPE * gPE;
    o.c = m.aC * gKN;
    const R P = rmin((R)(28.0 / 9.0) * L2k - (R)(218.0 / 27.0), m.capZ);
    o.p = (above && P > 0) ? m.aP * P : (R)0;
    o.r = g.rayleigh ? __ldg(&g.mat_r[mat]) * rdiv((R)1, E * E) : (R)0;
    o.tot = ((o.pe + o.c) + o.r) + o.p;
    return o;
}

// ---- Klein-Nishina composition-rejection (C7) ------------------------------------------------------------
template <class R> __device__ void kn_sample(R E, PhiloxStream& rng, R& eps, R& cost, R& sint2) {
    R k = E / (R)GN_ME_C2;
    R eps0 = (R)1 / ((R)1 + (R)2 * k);
    R a1 = -rlog(eps0);
    R eps0sq = eps0 * eps0;
    R a2 = ((R)1 - eps0sq) / (R)2;
    R thr = a1 / (a1 + a2);
    for (;;) {
        R u1 = draw<R>(rng), u2 = draw<R>(rng), u3 = draw<R>(rng);
        R e, e2;
        if (u1 < thr) { e = rexp(-a1 * u2); e2 = e * e; }
        else { e2 = eps0sq + ((R)1 - eps0sq) * u2; e = rsqrt_(e2); }
        R t = ((R)1 - e) / (k * e);
        R s2 = t * ((R)2 - t);
        if ((R)1 - e * s2 / ((R)1 + e2) >= u3) { eps = e; cost = (R)1 - t; sint2 = s2; return; }
    }
}

// Rayleigh angle (reading 18): cos(theta) from p(c) ~ 1 + c^2 by rejection, two draws per trial: c = 2 U1 - 1, accepted when
// 2 U2 <= 1 + c c
template <class R> __device__ R rayleigh_sample(PhiloxStream& rng) {
    for (;;) {
        const R u1 = draw<R>(rng), u2 = draw<R>(rng);
        const R c = (R)2 * u1 - (R)1;
        if ((R)2 * u2 <= (R)1 + c * c) return c;
    }
}

template <class R> __device__ void rotate_direction(V3<R>& w, R cost, R sint, R phi) {
    R sp, cp; rsincos(phi, &sp, &cp);
    R u = w.x, v = w.y, ww = w.z;
    R s2 = u * u + v * v;
    R nx, ny, nz;
    if (s2 >= (R)1e-10) {
        R s = rsqrt_(s2);
        nx = u * cost + sint * (u * ww * cp - v * sp) / s;
        ny = v * cost + sint * (v * ww * cp + u * sp) / s;
        nz = ww * cost - s * sint * cp;
    } else {
        nx = sint * cp; ny = sint * sp; nz = (ww < 0 ? -cost : cost);
    }
    R nn = rsqrt_(nx * nx + ny * ny + nz * nz);
    w.x = nx / nn; w.y = ny / nn; w.z = nz / nn;
}

// ---- sources (C8) --------------------------------------------------------------------------------------
template <class R> struct SourceDev {
    int kind, energy_kind;
    R o[3], a[3], e1[3], e2[3];
    R sigma, cos_half, e0, ln_e0, ln_ratio;
};

template <class R> __device__ void sample_source(const SourceDev<R>& s, PhiloxStream& rng, V3<R>& x, V3<R>& w, R& E) {
    const R twopi = (R)6.283185307179586;
    x.x = s.o[0]; x.y = s.o[1]; x.z = s.o[2];
    w.x = s.a[0]; w.y = s.a[1]; w.z = s.a[2];
    if (s.kind == 1) {            // GAUSS_PENCIL: Box-Muller in the plane normal to the axis
        R u0 = draw<R>(rng), u1 = draw<R>(rng);
        R r = s.sigma * rsqrt_((R)-2 * rlog(u0));
        R sp, cp; rsincos(twopi * u1, &sp, &cp);
        R gx = r * cp, gy = r * sp;
        x.x = s.o[0] + (gx * s.e1[0] + gy * s.e2[0]);
        x.y = s.o[1] + (gx * s.e1[1] + gy * s.e2[1]);
        x.z = s.o[2] + (gx * s.e1[2] + gy * s.e2[2]);
    } else if (s.kind == 2 || s.kind == 3) {   // CONE / ISOTROPIC: uniform in solid angle
        R u0 = draw<R>(rng), u1 = draw<R>(rng);
        R ct = (s.kind == 2) ? (R)1 - u0 * ((R)1 - s.cos_half) : (R)1 - (R)2 * u0;
        R st = rsqrt_(rmax(((R)1 - ct) * ((R)1 + ct), (R)0));
        R sp, cp; rsincos(twopi * u1, &sp, &cp);
        R cx = st * cp, cy = st * sp;
        R nx = (cx * s.e1[0] + cy * s.e2[0]) + ct * s.a[0];
        R ny = (cx * s.e1[1] + cy * s.e2[1]) + ct * s.a[1];
        R nz = (cx * s.e1[2] + cy * s.e2[2]) + ct * s.a[2];
        R nn = rsqrt_(nx * nx + ny * ny + nz * nz);
        w.x = nx / nn; w.y = ny / nn; w.z = nz / nn;
    }
    E = (s.energy_kind == 1) ? rexp(s.ln_e0 + draw<R>(rng) * s.ln_ratio) : s.e0;
}

}  // namespace gn
