// kernels.cu -- navigation kernels, the wavefront transport kernels and the C entry points that launch them.
//
// transport_run design (B200-first; the paper's one-thread-runs-Algorithm-1-to-completion kernel, PAPER.md
// L143, and its CUDPP compaction experiment, L195, are the prior art):
//   * photon state lives in two queues in HBM, one 16-byte-aligned record per photon (64 B in fp32, 112 B in
//     fp64: position, direction, E, remaining optical depth Y, the three energy factors of mu, volume, photon
//     index, Philox draw counter, step counters), moved with 16-byte vector loads / stores;
//   * one wavefront pass = one launch of transport_pass: every thread loads one live photon, advances it by up
//     to K steps (Algorithm 1 loop body: mu, s_int, ComputeStep, move / interact) keeping the navigation cursor
//     (node record + frame of the current volume) in registers, and survivors are compacted into the other queue
//     with a ballot + block-aggregated atomic cursor; pass 0 generates the photons from the source instead of
//     loading them and uses a short K so that photons that miss everything leave the warps early;
//   * energy deposits are reduced across the warp per distinct volume (shuffle tree) before the fp64 atomic;
//   * rare physics (Klein-Nishina sampling, energy factors in fp64) is kept out of line so that the hot
//     navigation loop stays small in registers and instruction cache;
//   * solids and material factors are staged in shared memory; transforms and voxel cells stay in L2.
#include <cstdio>
#include <cstring>
#include <string>
#include "geometry.h"
#include "nav.cuh"
#include "physics.cuh"

namespace gn {

// -------------------------------------------------------------------------------------------------------
// navigation kernels: pure maps over queries
// -------------------------------------------------------------------------------------------------------
constexpr int NAV_THREADS = 256;
constexpr int MAX_SMEM_SOLIDS = 64;
constexpr int MAX_SMEM_MATS = 32;

template <class R> __device__ __forceinline__ const SolidRec<R>* stage_solids(const GeoView<R>& g, SolidRec<R>* sh) {
    if (g.n_solids > MAX_SMEM_SOLIDS) return g.solids;
    for (int i = threadIdx.x; i < g.n_solids; i += blockDim.x) sh[i] = g.solids[i];
    return sh;
}

template <class R, bool HAS_DIR>
__global__ void __launch_bounds__(NAV_THREADS) locate_kernel(GeoView<R> g, const R* __restrict__ pos, const R* __restrict__ dir,
                                                             int64_t n, int32_t* __restrict__ vol_out) {
    __shared__ SolidRec<R> sh_solids[MAX_SMEM_SOLIDS];
    const SolidRec<R>* solids = stage_solids(g, sh_solids);
    __syncthreads();
    Navigator<R, HAS_DIR> nav(g, solids);
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        V3<R> x{pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
        V3<R> w{0, 0, 0};
        if (HAS_DIR) { w.x = dir[3 * i]; w.y = dir[3 * i + 1]; w.z = dir[3 * i + 2]; }
        Cursor<R> c;
        vol_out[i] = nav.locate(x, w, c);
    }
}

template <class R>
__global__ void __launch_bounds__(NAV_THREADS) step_kernel(GeoView<R> g, const R* __restrict__ pos, const R* __restrict__ dir,
                                                           const int32_t* __restrict__ vol_in, const R* __restrict__ max_step,
                                                           int64_t n, R* __restrict__ step_out, int32_t* __restrict__ next_out) {
    __shared__ SolidRec<R> sh_solids[MAX_SMEM_SOLIDS];
    const SolidRec<R>* solids = stage_solids(g, sh_solids);
    __syncthreads();
    Navigator<R, true> nav(g, solids);
    for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        V3<R> x{pos[3 * i], pos[3 * i + 1], pos[3 * i + 2]};
        V3<R> w{dir[3 * i], dir[3 * i + 1], dir[3 * i + 2]};
        int vol = vol_in[i];
        R step = rinf<R>(); int next = -1;
        if (vol >= 0 && vol < g.n_nodes) {
            Cursor<R> c; nav.load_cursor(vol, c);
            V3<R> xn;
            nav.compute_step(c, x, w, max_step ? max_step[i] : rinf<R>(), step, xn);
            next = c.vol;
        }
        step_out[i] = step; next_out[i] = next;
    }
}

// -------------------------------------------------------------------------------------------------------
// transport
// -------------------------------------------------------------------------------------------------------
constexpr int TR_THREADS = 128;
enum : int { EV_BOUNDARY = 0, EV_PE = 1, EV_COMPTON = 2, EV_PAIR = 3, EV_CUT = 4, EV_ESCAPE = 5, EV_STUCK = 6 };

struct DevStats {
    unsigned long long n_steps, n_compton, n_pe, n_pair, n_cut, n_escaped, n_stuck, n_photons;
    double e_escaped, e_stuck, e_source, e_deposited;
};

// one photon in the queue; sizeof = 64 (float) / 112 (double), moved as 16-byte words
template <class R> struct alignas(16) PhotonRec {
    R x, y, z, wx, wy, wz, E, Y, gPE, gKN, L2k;
    int32_t vol; uint32_t idx, ctr, misc;        // misc = zero_steps | nsteps << 8
    uint32_t pad[sizeof(R) == 4 ? 1 : 2];
};
static_assert(sizeof(PhotonRec<float>) == 64 && sizeof(PhotonRec<double>) == 112, "photon record layout");

template <class R> __device__ __forceinline__ void load_rec(const PhotonRec<R>* q, unsigned i, PhotonRec<R>& r) {
    const uint4* s = reinterpret_cast<const uint4*>(q + i);
    uint4* d = reinterpret_cast<uint4*>(&r);
#pragma unroll
    for (int k = 0; k < (int)(sizeof(PhotonRec<R>) / 16); ++k) d[k] = __ldcs(s + k);      // streamed: read once
}
template <class R> __device__ __forceinline__ void store_rec(PhotonRec<R>* q, unsigned i, const PhotonRec<R>& r) {
    uint4* d = reinterpret_cast<uint4*>(q + i);
    const uint4* s = reinterpret_cast<const uint4*>(&r);
#pragma unroll
    for (int k = 0; k < (int)(sizeof(PhotonRec<R>) / 16); ++k) __stcs(d + k, s[k]);
}

struct PerPhotonOut { uint64_t* hash; uint32_t* nsteps; double* efinal; };

__device__ __forceinline__ void fnv_word(uint64_t& h, uint32_t w) {
#pragma unroll
    for (int i = 0; i < 4; ++i) { h ^= (w >> (8 * i)) & 0xffu; h *= 0x100000001b3ull; }
}

// warp-aggregated tally: one fp64 atomic per distinct volume per warp
__device__ __noinline__ void warp_tally(double* __restrict__ edep, int vol, double dep, bool has) {
    unsigned pending = __ballot_sync(0xffffffffu, has);
    const int lane = threadIdx.x & 31;
    while (pending) {
        int leader = __ffs(pending) - 1;
        int v = __shfl_sync(0xffffffffu, vol, leader);
        bool same = has && vol == v;
        unsigned grp = __ballot_sync(0xffffffffu, same);
        if (grp == (1u << leader)) {
            if (lane == leader) atomicAdd(&edep[v], dep);
        } else {
            double s = same ? dep : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == leader) atomicAdd(&edep[v], s);
        }
        pending &= ~grp;
    }
}

template <class T> __device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Compton scattering of one photon (C6/C7), out of line: rare (well under 1 % of steps)
template <class R>
__device__ __noinline__ void compton(R& E, V3<R>& w, PhiloxStream& rng, R& dep) {
    R eps, cost, s2;
    kn_sample(E, rng, eps, cost, s2);
    R Ep = eps * E;
    R phi = (R)6.283185307179586 * draw<R>(rng);
    rotate_direction(w, cost, rsqrt_(rmax(s2, (R)0)), phi);
    dep = E - Ep;
    E = Ep;
}
template <class R> __device__ __noinline__ void energy_factors_ool(R E, EnergyFactors<R>& ef) { ef = energy_factors(E); }

template <class R, bool FROM_SOURCE, bool TRACK>
__global__ void __launch_bounds__(TR_THREADS)
transport_pass(GeoView<R> g, SourceDev<R> src, uint64_t seed, uint64_t first_id, uint32_t n_in, const PhotonRec<R>* __restrict__ qin,
               PhotonRec<R>* __restrict__ qout, uint32_t* __restrict__ out_count, double* __restrict__ edep, DevStats* __restrict__ stats,
               PerPhotonOut pp, int K) {
    __shared__ SolidRec<R> sh_solids[MAX_SMEM_SOLIDS];
    __shared__ MatRec<R> sh_mats[MAX_SMEM_MATS];
    __shared__ unsigned sh_warp_count[TR_THREADS / 32];
    __shared__ unsigned sh_base;
    __shared__ unsigned long long sh_cnt[8];
    __shared__ double sh_en[4];
    const SolidRec<R>* solids = stage_solids(g, sh_solids);
    const MatRec<R>* mats = g.mats;
    if (g.n_mats <= MAX_SMEM_MATS) { for (int i = threadIdx.x; i < g.n_mats; i += blockDim.x) sh_mats[i] = g.mats[i]; mats = sh_mats; }
    if (threadIdx.x < 8) sh_cnt[threadIdx.x] = 0;
    if (threadIdx.x < 4) sh_en[threadIdx.x] = 0.0;
    __syncthreads();
    Navigator<R, true> nav(g, solids);
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    bool alive = i < n_in;
    V3<R> x{0, 0, 0}, w{0, 0, 1}; R E = 1, Y = 0; uint32_t idx = 0, misc = 0; uint64_t h = 0xcbf29ce484222325ull;
    EnergyFactors<R> ef{}; ef.above_pair = 0;
    Cursor<R> cur; cur.vol = -1; cur.nd = make_int4(-1, 0, 0, 0);
    PhiloxStream rng; rng.init(seed, 0, 0);
    unsigned c_steps = 0, c_compton = 0, c_pe = 0, c_pair = 0, c_cut = 0, c_esc = 0, c_stuck = 0, c_phot = 0;
    double e_esc = 0, e_stuck = 0, e_src = 0, e_dep = 0;

    if (alive) {
        if (FROM_SOURCE) {
            idx = i;
            rng.init(seed, first_id + i, 0);
            sample_source(src, rng, x, w, E);
            c_phot = 1; e_src = (double)E;
            if (nav.locate(x, w, cur) < 0) {
                c_esc = 1; e_esc = (double)E; alive = false;
                if (TRACK) { pp.hash[idx] = h; if (pp.nsteps) pp.nsteps[idx] = 0; if (pp.efinal) pp.efinal[idx] = (double)E; }
            } else {
                Y = -rlog(draw<R>(rng));                       // Algorithm 1 steps 1-2
                energy_factors_ool(E, ef);
            }
        } else {
            PhotonRec<R> r; load_rec(qin, i, r);
            x.x = r.x; x.y = r.y; x.z = r.z; w.x = r.wx; w.y = r.wy; w.z = r.wz; E = r.E; Y = r.Y;
            ef.gPE = r.gPE; ef.gKN = r.gKN; ef.L2k = r.L2k; ef.above_pair = ((double)E / GN_ME_C2) > 2.0;
            idx = r.idx; misc = r.misc;
            rng.init(seed, first_id + idx, r.ctr);
            nav.load_cursor(r.vol, cur);
            if (TRACK) h = pp.hash[idx];
        }
    }

    for (int k = 0; k < K; ++k) {
        if (!__any_sync(0xffffffffu, alive)) break;
        bool has_dep = false; double dep_d = 0.0; int dep_vol = 0;
        if (alive) {
            R muPE, muC, muP; mu_partials(mats[cur.nd.z], ef, muPE, muC, muP);
            R mu = (muPE + muC) + muP;
            R s_int = mu > 0 ? Y / mu : rinf<R>();                         // remaining part of Eq. 7
            const int vol_before = cur.vol;
            R step; V3<R> xn;
            nav.compute_step(cur, x, w, s_int, step, xn);                  // "next intersection"
            ++c_steps; misc += 0x100u;
            int ev; R len;
            if (step == rinf<R>()) {                                       // S_j >= Y: the photon interacts in vol
                len = s_int;
                x = advance(x, w, s_int);
                R t = draw<R>(rng) * mu;
                has_dep = true; dep_vol = vol_before;
                if (t < muPE) {
                    dep_d = (double)E; ++c_pe; ev = EV_PE; alive = false;
                } else if (t < muPE + muC || !(muP > 0)) {
                    R dep; compton(E, w, rng, dep);
                    ++c_compton; ev = EV_COMPTON;
                    if (E < g.e_cut) { dep = dep + E; ++c_cut; ev = EV_CUT; alive = false; }
                    dep_d = (double)dep;
                    if (alive) { energy_factors_ool(E, ef); Y = -rlog(draw<R>(rng)); }
                } else {
                    dep_d = (double)E; ++c_pair; ev = EV_PAIR; alive = false;
                }
                e_dep += dep_d;
            } else {                                                       // boundary: S_j update
                len = step;
                x = xn;
                Y = rmax(Y - step * mu, (R)0);
                if (cur.vol < 0) { ++c_esc; e_esc += (double)E; ev = EV_ESCAPE; alive = false; } else ev = EV_BOUNDARY;
            }
            uint32_t zs = misc & 0xffu;
            zs = (len <= g.delta) ? zs + 1 : 0;
            if (alive && zs >= (uint32_t)g.stuck_limit) { ++c_stuck; e_stuck += (double)E; ev = EV_STUCK; alive = false; }
            misc = (misc & ~0xffu) | (zs & 0xffu);
            if (TRACK) {
                fnv_word(h, (uint32_t)vol_before); fnv_word(h, (uint32_t)ev);
                if (!alive) { pp.hash[idx] = h; if (pp.nsteps) pp.nsteps[idx] = misc >> 8; if (pp.efinal) pp.efinal[idx] = (double)E; }
            }
        }
        if (__any_sync(0xffffffffu, has_dep)) warp_tally(edep, dep_vol, dep_d, has_dep);
    }

    // ---- compaction of survivors into the other queue ------------------------------------
    unsigned bal = __ballot_sync(0xffffffffu, alive);
    if (lane == 0) sh_warp_count[warp] = __popc(bal);
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned tot = 0;
        for (int q = 0; q < TR_THREADS / 32; ++q) { unsigned c = sh_warp_count[q]; sh_warp_count[q] = tot; tot += c; }
        sh_base = tot ? atomicAdd(out_count, tot) : 0u;
    }
    __syncthreads();
    if (alive) {
        unsigned o = sh_base + sh_warp_count[warp] + __popc(bal & ((1u << lane) - 1u));
        PhotonRec<R> r;
        r.x = x.x; r.y = x.y; r.z = x.z; r.wx = w.x; r.wy = w.y; r.wz = w.z; r.E = E; r.Y = Y;
        r.gPE = ef.gPE; r.gKN = ef.gKN; r.L2k = ef.L2k; r.vol = cur.vol; r.idx = idx; r.ctr = rng.j; r.misc = misc;
#pragma unroll
        for (int q = 0; q < (int)(sizeof(r.pad) / 4); ++q) r.pad[q] = 0;
        store_rec(qout, o, r);
        if (TRACK) pp.hash[idx] = h;
    }
    // ---- statistics: warp tree, shared atomics, one global atomic per counter per block -----------------------
    unsigned long long cs[8] = {c_steps, c_compton, c_pe, c_pair, c_cut, c_esc, c_stuck, c_phot};
    double es[4] = {e_esc, e_stuck, e_src, e_dep};
#pragma unroll
    for (int q = 0; q < 8; ++q) { unsigned long long v = warp_sum(cs[q]); if (lane == 0 && v) atomicAdd(&sh_cnt[q], v); }
#pragma unroll
    for (int q = 0; q < 4; ++q) { double v = warp_sum(es[q]); if (lane == 0 && v != 0.0) atomicAdd(&sh_en[q], v); }
    __syncthreads();
    if (threadIdx.x < 8 && sh_cnt[threadIdx.x]) atomicAdd(&(&stats->n_steps)[threadIdx.x], sh_cnt[threadIdx.x]);
    if (threadIdx.x >= 8 && threadIdx.x < 12 && sh_en[threadIdx.x - 8] != 0.0) atomicAdd(&(&stats->e_escaped)[threadIdx.x - 8], sh_en[threadIdx.x - 8]);
}

// -------------------------------------------------------------------------------------------------------
// host side
// -------------------------------------------------------------------------------------------------------
static int cuda_fail(cudaError_t e, const char* where) {
    return fail(GN_CUDA_ERROR, std::string(where) + ": " + cudaGetErrorString(e));
}
#define GN_CUDA(call, where) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return cuda_fail(e__, where); } while (0)

static int nav_grid(int64_t n) {
    int64_t blocks = (n + NAV_THREADS - 1) / NAV_THREADS;
    const int64_t cap = 148 * 64;                 // grid-stride beyond this; multiple of the SM count
    return (int)std::max<int64_t>(1, std::min(blocks, cap));
}

template <class R> const GeoView<R>& view(const gn_geometry* g);
template <> const GeoView<float>& view<float>(const gn_geometry* g) { return g->v32; }
template <> const GeoView<double>& view<double>(const gn_geometry* g) { return g->v64; }

template <class R> int locate_impl(const gn_geometry* geo, const void* pos, const void* dir, int64_t n, int32_t* out, cudaStream_t s) {
    if (n == 0) return GN_OK;
    if (dir) locate_kernel<R, true><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, n, out);
    else locate_kernel<R, false><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, nullptr, n, out);
    GN_CUDA(cudaGetLastError(), "gn_nav_locate launch");
    return GN_OK;
}
template <class R> int step_impl(const gn_geometry* geo, const void* pos, const void* dir, const int32_t* vol, const void* ms,
                                 int64_t n, void* step, int32_t* next, cudaStream_t s) {
    if (n == 0) return GN_OK;
    step_kernel<R><<<nav_grid(n), NAV_THREADS, 0, s>>>(view<R>(geo), (const R*)pos, (const R*)dir, vol, (const R*)ms, n, (R*)step, next);
    GN_CUDA(cudaGetLastError(), "gn_nav_compute_step launch");
    return GN_OK;
}

template <class R> bool make_source(const gn_source& s, SourceDev<R>& o) {
    // a = axis / |axis|; h = unit vector of the smallest |a_i| (ties x < y < z);
    // e1 = normalise(h - (h.a) a); e2 = a x e1 -- fp64 on the host, rounded once to Real.
    double n = std::sqrt(s.axis[0] * s.axis[0] + s.axis[1] * s.axis[1] + s.axis[2] * s.axis[2]);
    if (!(n > 0) || !(s.e0 > 0)) return false;
    double a[3] = {s.axis[0] / n, s.axis[1] / n, s.axis[2] / n};
    int m = 0;
    if (std::fabs(a[1]) < std::fabs(a[m])) m = 1;
    if (std::fabs(a[2]) < std::fabs(a[m])) m = 2;
    double hv[3] = {0, 0, 0}; hv[m] = 1;
    double ha = a[m];
    double e1[3] = {hv[0] - ha * a[0], hv[1] - ha * a[1], hv[2] - ha * a[2]};
    double n1 = std::sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
    for (int i = 0; i < 3; ++i) e1[i] /= n1;
    double e2[3] = {a[1] * e1[2] - a[2] * e1[1], a[2] * e1[0] - a[0] * e1[2], a[0] * e1[1] - a[1] * e1[0]};
    o.kind = s.kind; o.energy_kind = s.energy_kind;
    for (int i = 0; i < 3; ++i) { o.o[i] = (R)s.origin[i]; o.a[i] = (R)a[i]; o.e1[i] = (R)e1[i]; o.e2[i] = (R)e2[i]; }
    o.sigma = (R)s.sigma; o.cos_half = (R)std::cos(s.half_angle); o.e0 = (R)s.e0; o.ln_e0 = 0; o.ln_ratio = 0;
    if (s.energy_kind == GN_E_LOGUNIFORM) {
        if (!(s.e1 >= s.e0)) return false;
        o.ln_e0 = (R)std::log(s.e0); o.ln_ratio = (R)std::log(s.e1 / s.e0);
    } else if (s.energy_kind != GN_E_MONO) return false;
    return s.kind >= GN_SRC_PENCIL && s.kind <= GN_SRC_ISOTROPIC;
}

constexpr int64_t TR_BATCH = 1ll << 24;     // photons per batch (bounds scratch at 2 x 16.8 M x 64 B = 2.1 GB in fp32)

template <class R>
int transport_impl(const gn_geometry* geo, const gn_source* h_src, uint64_t seed, int64_t first_id, int64_t n_photons,
                   double* d_edep, gn_run_stats* h_stats, uint64_t* d_hash, uint32_t* d_nsteps, double* d_efinal, cudaStream_t s) {
    SourceDev<R> src;
    if (!make_source(*h_src, src)) return fail(GN_INVALID_ARGUMENT, "gn_transport_run: bad source (axis, energies or kind)");
    const bool track = d_hash || d_nsteps || d_efinal;
    const int K = geo->opts.steps_per_pass;
    const int K0 = std::min(K, geo->opts.first_pass_steps > 0 ? geo->opts.first_pass_steps : 4);      // first pass: short, sheds photons that miss
    const size_t cap = (size_t)std::min<int64_t>(std::max<int64_t>(n_photons, 1), TR_BATCH);
    const size_t qb = cap * sizeof(PhotonRec<R>);
    const size_t hb = (track && !d_hash) ? cap * 8 : 0;       // the hash array doubles as per-photon state between passes
    char* scratch = nullptr;
    GN_CUDA(cudaMemsetAsync(d_edep, 0, sizeof(double) * (size_t)geo->n_places, s), "gn_transport_run memset edep");
    cudaError_t e = cudaMallocAsync((void**)&scratch, 2 * qb + hb + 512, s);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(GN_OUT_OF_MEMORY, std::string("gn_transport_run scratch: ") + cudaGetErrorString(e)); }
    PhotonRec<R>* qa = (PhotonRec<R>*)scratch; PhotonRec<R>* qb_ = (PhotonRec<R>*)(scratch + qb);
    uint64_t* tmp_hash = hb ? (uint64_t*)(scratch + 2 * qb) : nullptr;
    DevStats* d_stats = (DevStats*)(scratch + 2 * qb + hb);
    uint32_t* d_count = (uint32_t*)(scratch + 2 * qb + hb + 256);
    uint32_t* h_count = nullptr;
    int rc = GN_OK;
    uint64_t passes = 0, launches = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    double kernel_ms = 0.0;
    auto cleanup = [&]() { if (h_count) cudaFreeHost(h_count); if (ev0) cudaEventDestroy(ev0); if (ev1) cudaEventDestroy(ev1); cudaFreeAsync(scratch, s); };
    if (cudaMallocHost((void**)&h_count, 64) != cudaSuccess) { cudaGetLastError(); cleanup(); return fail(GN_OUT_OF_MEMORY, "gn_transport_run: pinned alloc"); }
    if (cudaEventCreate(&ev0) != cudaSuccess || cudaEventCreate(&ev1) != cudaSuccess) { cudaGetLastError(); cleanup(); return fail(GN_CUDA_ERROR, "gn_transport_run: event create"); }
    cudaMemsetAsync(d_stats, 0, 512, s);
    const GeoView<R>& g = view<R>(geo);
    for (int64_t done = 0; done < n_photons && rc == GN_OK; done += (int64_t)cap) {
        uint32_t n_in = (uint32_t)std::min<int64_t>((int64_t)cap, n_photons - done);
        PerPhotonOut pp{d_hash ? d_hash + done : tmp_hash, d_nsteps ? d_nsteps + done : nullptr, d_efinal ? d_efinal + done : nullptr};
        PhotonRec<R>* in = qb_; PhotonRec<R>* out = qa;
        bool first = true;
        while (n_in > 0) {
            cudaMemsetAsync(d_count, 0, 4, s);
            unsigned blocks = (n_in + TR_THREADS - 1) / TR_THREADS;
            cudaEventRecord(ev0, s);
            if (first) {
                if (track) transport_pass<R, true, true><<<blocks, TR_THREADS, 0, s>>>(g, src, seed, (uint64_t)(first_id + done), n_in, in, out, d_count, d_edep, d_stats, pp, K0);
                else transport_pass<R, true, false><<<blocks, TR_THREADS, 0, s>>>(g, src, seed, (uint64_t)(first_id + done), n_in, in, out, d_count, d_edep, d_stats, pp, K0);
            } else {
                if (track) transport_pass<R, false, true><<<blocks, TR_THREADS, 0, s>>>(g, src, seed, (uint64_t)(first_id + done), n_in, in, out, d_count, d_edep, d_stats, pp, K);
                else transport_pass<R, false, false><<<blocks, TR_THREADS, 0, s>>>(g, src, seed, (uint64_t)(first_id + done), n_in, in, out, d_count, d_edep, d_stats, pp, K);
            }
            ++passes; ++launches;
            e = cudaGetLastError();
            cudaEventRecord(ev1, s);
            if (e == cudaSuccess) e = cudaMemcpyAsync(h_count, d_count, 4, cudaMemcpyDeviceToHost, s);
            if (e == cudaSuccess) e = cudaStreamSynchronize(s);
            if (e != cudaSuccess) { rc = cuda_fail(e, "gn_transport_run pass"); break; }
            { float ms = 0.f; if (cudaEventElapsedTime(&ms, ev0, ev1) == cudaSuccess) kernel_ms += ms; }
            n_in = *h_count;
            first = false;
            PhotonRec<R>* t = in; in = out; out = t;
        }
    }
    if (rc == GN_OK) {
        DevStats hs;
        e = cudaMemcpyAsync(&hs, d_stats, sizeof hs, cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) rc = cuda_fail(e, "gn_transport_run stats");
        else if (h_stats) {
            h_stats->n_steps = hs.n_steps; h_stats->n_compton = hs.n_compton; h_stats->n_pe = hs.n_pe; h_stats->n_pair = hs.n_pair;
            h_stats->n_cut = hs.n_cut; h_stats->n_escaped = hs.n_escaped; h_stats->n_stuck = hs.n_stuck; h_stats->n_photons = hs.n_photons;
            h_stats->e_escaped = hs.e_escaped; h_stats->e_stuck = hs.e_stuck; h_stats->e_source = hs.e_source; h_stats->e_deposited = hs.e_deposited;
            h_stats->n_passes = passes; h_stats->n_kernel_launches = launches; h_stats->kernel_ms = kernel_ms;
        }
    }
    cleanup();
    return rc;
}

}  // namespace gn

using namespace gn;

extern "C" int gn_nav_locate(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir, int64_t n,
                             int32_t* d_vol_out, void* cuda_stream) {
    if (!geo || n < 0 || (n > 0 && (!d_pos || !d_vol_out))) return fail(GN_INVALID_ARGUMENT, "gn_nav_locate: bad argument");
    if (precision == 32) return locate_impl<float>(geo, d_pos, d_dir, n, d_vol_out, (cudaStream_t)cuda_stream);
    if (precision == 64) return locate_impl<double>(geo, d_pos, d_dir, n, d_vol_out, (cudaStream_t)cuda_stream);
    return fail(GN_INVALID_ARGUMENT, "gn_nav_locate: precision must be 32 or 64");
}

extern "C" int gn_nav_compute_step(const gn_geometry* geo, int precision, const void* d_pos, const void* d_dir,
                                   const int32_t* d_vol_in, const void* d_max_step, int64_t n, void* d_step_out,
                                   int32_t* d_next_vol_out, void* cuda_stream) {
    if (!geo || n < 0 || (n > 0 && (!d_pos || !d_dir || !d_vol_in || !d_step_out || !d_next_vol_out)))
        return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_step: bad argument");
    if (precision == 32) return step_impl<float>(geo, d_pos, d_dir, d_vol_in, d_max_step, n, d_step_out, d_next_vol_out, (cudaStream_t)cuda_stream);
    if (precision == 64) return step_impl<double>(geo, d_pos, d_dir, d_vol_in, d_max_step, n, d_step_out, d_next_vol_out, (cudaStream_t)cuda_stream);
    return fail(GN_INVALID_ARGUMENT, "gn_nav_compute_step: precision must be 32 or 64");
}

extern "C" int gn_transport_run(const gn_geometry* geo, int precision, const gn_source* h_src, uint64_t seed, int64_t first_photon_id,
                                int64_t n_photons, double* d_edep_out, gn_run_stats* h_stats_out, uint64_t* d_hash_out,
                                uint32_t* d_nsteps_out, double* d_efinal_out, void* cuda_stream) {
    if (!geo || !h_src || !d_edep_out || n_photons < 0 || first_photon_id < 0) return fail(GN_INVALID_ARGUMENT, "gn_transport_run: bad argument");
    if (h_stats_out) std::memset(h_stats_out, 0, sizeof *h_stats_out);
    if (precision == 32) return transport_impl<float>(geo, h_src, seed, first_photon_id, n_photons, d_edep_out, h_stats_out, d_hash_out, d_nsteps_out, d_efinal_out, (cudaStream_t)cuda_stream);
    if (precision == 64) return transport_impl<double>(geo, h_src, seed, first_photon_id, n_photons, d_edep_out, h_stats_out, d_hash_out, d_nsteps_out, d_efinal_out, (cudaStream_t)cuda_stream);
    return fail(GN_INVALID_ARGUMENT, "gn_transport_run: precision must be 32 or 64");
}

extern "C" int gn_nav_query_host(const gn_geometry* geo, int precision, const void* h_pos, const void* h_dir, int64_t n,
                                 int32_t* h_vol_out, void* h_step_out, int32_t* h_next_vol_out) {
    if (!geo || n < 0 || (precision != 32 && precision != 64) || (n > 0 && (!h_pos || !h_dir || !h_vol_out || !h_step_out || !h_next_vol_out)))
        return fail(GN_INVALID_ARGUMENT, "gn_nav_query_host: bad argument");
    if (n == 0) return GN_OK;
    const size_t rs = precision == 32 ? 4 : 8;
    char* d = nullptr;
    const size_t b_pos = 3 * rs * (size_t)n, b_i = 4 * (size_t)n, b_r = rs * (size_t)n;
    cudaError_t e = cudaMalloc((void**)&d, 2 * b_pos + 2 * b_i + b_r);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(GN_OUT_OF_MEMORY, "gn_nav_query_host: cudaMalloc"); }
    char *dp = d, *dd = d + b_pos, *dstep = d + 2 * b_pos, *dvol = dstep + b_r, *dnext = dvol + b_i;
    int rc = GN_OK;
    e = cudaMemcpy(dp, h_pos, b_pos, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(dd, h_dir, b_pos, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        rc = gn_nav_locate(geo, precision, dp, dd, n, (int32_t*)dvol, nullptr);
        if (rc == GN_OK) rc = gn_nav_compute_step(geo, precision, dp, dd, (const int32_t*)dvol, nullptr, n, dstep, (int32_t*)dnext, nullptr);
    }
    if (rc == GN_OK && e == cudaSuccess) e = cudaMemcpy(h_vol_out, dvol, b_i, cudaMemcpyDeviceToHost);
    if (rc == GN_OK && e == cudaSuccess) e = cudaMemcpy(h_step_out, dstep, b_r, cudaMemcpyDeviceToHost);
    if (rc == GN_OK && e == cudaSuccess) e = cudaMemcpy(h_next_vol_out, dnext, b_i, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (rc != GN_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(e, "gn_nav_query_host");
    return GN_OK;
}

extern "C" int gn_transport_run_host(const gn_geometry* geo, int precision, const gn_source* h_src, uint64_t seed,
                                     int64_t first_photon_id, int64_t n_photons, double* h_edep_out, gn_run_stats* h_stats_out) {
    if (!geo || !h_edep_out) return fail(GN_INVALID_ARGUMENT, "gn_transport_run_host: bad argument");
    double* d = nullptr;
    const size_t bytes = sizeof(double) * (size_t)geo->n_places;
    if (cudaMalloc((void**)&d, bytes) != cudaSuccess) { cudaGetLastError(); return fail(GN_OUT_OF_MEMORY, "gn_transport_run_host: cudaMalloc"); }
    int rc = gn_transport_run(geo, precision, h_src, seed, first_photon_id, n_photons, d, h_stats_out, nullptr, nullptr, nullptr, nullptr);
    cudaError_t e = cudaSuccess;
    if (rc == GN_OK) e = cudaMemcpy(h_edep_out, d, bytes, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (rc != GN_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(e, "gn_transport_run_host");
    return GN_OK;
}
